"""GPU parity of image cleaning + moments (DESIGN.md
readings R31-R35) against oracle/rta_oracle_image.cpp, through the C ABI:
rta_image_moments on device charge / time arrays, and rta_extract_image (the
extraction and the cleaning in one kernel) against oracle.extract followed by
oracle.image_moments. n_pix, mask and q_max bit-exact; the fp32 parameters
within the tolerances of tests/_image.py::assert_image_parity."""
import json
import os

import numpy as np
import pytest

import dl0gen
import oracle
from tests._image import F32, assert_image_parity, blob_images

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden", "image7.json")


def dev(a, dtype=None):
    import torch
    a = np.ascontiguousarray(a, dtype)
    if a.dtype == np.uint16:
        a = a.view(np.int16)
    return torch.from_numpy(a).cuda()


def image_outputs(E, P, mask=True):
    import torch
    return (torch.full((E,), -7, dtype=torch.int32, device="cuda"),
            torch.full((E, 8), -7.0, dtype=torch.float32, device="cuda"),
            torch.full((E, P), 9, dtype=torch.uint8, device="cuda") if mask else None)


def host(outs):
    import torch
    torch.cuda.synchronize()
    return tuple(None if o is None else o.cpu().numpy() for o in outs)


def gpu_moments(q, t, x, y, nbr, tp, tb, mask=True):
    import paper_1307_6489_b200 as rta
    E, P = q.shape
    outs = image_outputs(E, P, mask)
    rta.rta_image_moments(dev(q, F32), dev(t, F32), E, P, dev(x, F32), dev(y, F32),
                          dev(nbr, np.int32), tp, tb, *outs)
    return host(outs)


def gpu_extract_image(wf, ped, gain, W, x, y, nbr, tp, tb, mask=True, generic=False, d_wf=None):
    import paper_1307_6489_b200 as rta
    E, P, S = wf.shape
    outs = image_outputs(E, P, mask)
    rta.rta_extract_image(dev(wf) if d_wf is None else d_wf, E, P, S, dev(ped, np.int32),
                          dev(gain, F32), W, dev(x, F32), dev(y, F32), dev(nbr, np.int32),
                          tp, tb, *outs, generic=generic)
    return host(outs)


def oracle_extract_image(wf, ped, gain, W, x, y, nbr, tp, tb):
    E, P, _ = wf.shape
    _, _, q, t = oracle.extract(wf, ped, gain, W)
    return oracle.image_moments(q.reshape(E, P), t.reshape(E, P), x, y, nbr, tp, tb)


# ---------------------------------------------------------------- rta_image_moments
def test_hand_worked_camera_on_the_device():
    g = json.load(open(GOLD))
    q = np.array([[float(v) for v in ev["charge"]] for ev in g["events"]], F32)
    t = np.array([ev["time"] for ev in g["events"]], F32)
    x, y, nbr = np.array(g["pix_x"], F32), np.array(g["pix_y"], F32), np.array(g["neighbors"], np.int32)
    got = gpu_moments(q, t, x, y, nbr, g["thr_picture"], g["thr_boundary"])
    for i, ev in enumerate(g["events"]):
        assert got[2][i].tolist() == ev["mask"], ev["name"]
        assert got[0][i] == ev["n_pix"]
    assert_image_parity(got, oracle.image_moments(q, t, x, y, nbr, g["thr_picture"], g["thr_boundary"]),
                        x, y, "image7")


@pytest.mark.parametrize("P,E,seed", [(1855, 70, 0), (1764, 33, 1), (2048, 40, 3), (37, 300, 2),
                                      (7, 50, 4), (1, 5, 5), (255, 64, 6), (257, 64, 7),
                                      (5000, 12, 8), (11328, 6, 9)])
def test_blob_images(P, E, seed):
    q, t, x, y, nbr = blob_images(E, P, seed)
    got = gpu_moments(q, t, x, y, nbr, 8.0, 4.0)
    want = oracle.image_moments(q, t, x, y, nbr, 8.0, 4.0)
    n_axis = assert_image_parity(got, want, x, y, "blobs P=%d" % P)
    if P >= 37:
        assert want[0].max() > 5 and n_axis > 0
    # without the mask output: same parameters, bit for bit
    got2 = gpu_moments(q, t, x, y, nbr, 8.0, 4.0, mask=False)
    assert np.array_equal(got2[0], got[0]) and np.array_equal(got2[1].view(np.int32), got[1].view(np.int32))


def test_symmetric_table_shortcut_equals_the_definition():
    """On a symmetric neighbour table (every hex camera) the cleaning does both
    steps in one pass over the core pixels; rta_debug_general_cleaning forces the
    two steps as written. Same mask, same parameters, bit for bit — on blobs, on
    dense images (every pixel core / every pixel above the boundary) and through
    both fused kernels."""
    import paper_1307_6489_b200 as rta
    for P, seed in ((1855, 31), (469, 32), (37, 33)):
        q, t, x, y, nbr = blob_images(40, P, seed)
        q[5, :] = 20.0                      # every pixel core
        q[6, :] = 5.0                       # every pixel above the boundary threshold only
        q[7, ::3] = 50.0                    # a third of the camera core
        want = oracle.image_moments(q, t, x, y, nbr, 8.0, 4.0)
        fast = gpu_moments(q, t, x, y, nbr, 8.0, 4.0)
        rta.rta_debug_general_cleaning(True)
        try:
            slow = gpu_moments(q, t, x, y, nbr, 8.0, 4.0)
        finally:
            rta.rta_debug_general_cleaning(False)
        assert_image_parity(fast, want, x, y, "symmetric P=%d" % P)
        for a, b in zip(fast, slow):
            assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch("C3", 40)
    for generic in (False, True):
        fast = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb, generic=generic)
        rta.rta_debug_general_cleaning(True)
        try:
            slow = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb, generic=generic)
        finally:
            rta.rta_debug_general_cleaning(False)
        for a, b in zip(fast, slow):
            assert np.array_equal(a.view(np.uint8), b.view(np.uint8))


def test_thresholds_and_special_values():
    q, t, x, y, nbr = blob_images(24, 469, 11)
    q[3, :] = np.nan                       # NaN never passes a threshold
    q[4, 10:40] = np.nan
    q[5, :] = -3.0                         # everything passes negative thresholds, size < 0 -> zeros
    q[6, :] = 20.0                         # every pixel is core
    q[7, :] = 0.0
    q[8, 100] = np.inf                     # an isolated infinite pixel is dropped
    for tp, tb in ((8.0, 4.0), (4.0, 8.0), (-5.0, -5.0), (1e9, 1.0), (8.0, -1e9),
                   (float("nan"), 1.0), (8.0, float("nan")), (8.0, 8.0)):
        got = gpu_moments(q, t, x, y, nbr, tp, tb)
        want = oracle.image_moments(q, t, x, y, nbr, tp, tb)
        assert_image_parity(got, want, x, y, "thr %r %r" % (tp, tb))
    assert want[0][6] == 469


def test_neighbour_table_is_used_as_given():
    """Out-of-range entries mean 'none'; self references, duplicates and a
    one-directional table follow the definition, not a symmetrised version."""
    rng = np.random.default_rng(5)
    P = 300
    q, t, x, y, _ = blob_images(40, P, 12)
    nbr = rng.integers(-50, P + 50, (P, 6)).astype(np.int32)
    nbr[::7, 0] = np.arange(P)[::7]        # self neighbours
    nbr[5] = [2**31 - 1, -2**31, P, -1, 6, 6]
    got = gpu_moments(q, t, x, y, nbr, 3.0, 1.0)
    want = oracle.image_moments(q, t, x, y, nbr, 3.0, 1.0)
    assert want[0].max() > 3
    assert_image_parity(got, want, x, y, "random table")


def test_unaligned_rows_and_outputs():
    """P % 4 != 0 makes most event rows 4-byte aligned only; odd output addresses."""
    import torch
    import paper_1307_6489_b200 as rta
    q, t, x, y, nbr = blob_images(9, 1855, 13)
    E, P = q.shape
    dq = torch.empty(E * P + 1, dtype=torch.float32, device="cuda")[1:]
    dt = torch.empty(E * P + 3, dtype=torch.float32, device="cuda")[3:]
    dq.copy_(torch.from_numpy(q).reshape(-1))
    dt.copy_(torch.from_numpy(t).reshape(-1))
    n = torch.empty(E + 1, dtype=torch.int32, device="cuda")[1:]
    par = torch.empty(E * 8 + 1, dtype=torch.float32, device="cuda")[1:]
    m = torch.empty(E * P + 1, dtype=torch.uint8, device="cuda")[1:]
    rta.rta_image_moments(dq, dt, E, P, dev(x), dev(y), dev(nbr), 8.0, 4.0, n, par, m)
    got = host((n, par.reshape(E, 8), m.reshape(E, P)))
    assert_image_parity(got, oracle.image_moments(q, t, x, y, nbr, 8.0, 4.0), x, y, "unaligned")


def test_image_moments_errors():
    import torch
    import paper_1307_6489_b200 as rta
    q, t, x, y, nbr = blob_images(2, 37, 1)
    a = dict(charge=dev(q), time=dev(t), x=dev(x), y=dev(y), nbr=dev(nbr))
    n, par, m = image_outputs(2, 37)

    def call(**kw):
        args = dict(charge=a["charge"], time=a["time"], E=2, P=37, x=a["x"], y=a["y"], nbr=a["nbr"],
                    n=n, par=par, m=m)
        args.update(kw)
        rta.rta_image_moments(args["charge"], args["time"], args["E"], args["P"], args["x"], args["y"],
                              args["nbr"], 8.0, 4.0, args["n"], args["par"], args["m"])
    for kw, status in ((dict(charge=None), rta.RTA_ERR_NULL), (dict(x=None), rta.RTA_ERR_NULL),
                       (dict(nbr=None), rta.RTA_ERR_NULL), (dict(n=None), rta.RTA_ERR_NULL),
                       (dict(par=None), rta.RTA_ERR_NULL), (dict(E=-1), rta.RTA_ERR_SHAPE),
                       (dict(P=0), rta.RTA_ERR_SHAPE),
                       (dict(P=rta.rta_image_max_pixels() + 1), rta.RTA_ERR_UNSUPPORTED),
                       (dict(charge=a["charge"].data_ptr() + 2), rta.RTA_ERR_ALIGN)):
        with pytest.raises(rta.RtaError) as ei:
            call(**kw)
        assert ei.value.status == status, kw
    torch.cuda.synchronize()
    assert (n.cpu() == -7).all() and (par.cpu() == -7).all()    # nothing was enqueued
    call(E=0, charge=None, x=None, n=None, par=None)             # empty input: ok, nothing touched
    call(m=None)
    torch.cuda.synchronize()
    assert (m.cpu() == 9).all()


def test_largest_camera():
    import paper_1307_6489_b200 as rta
    P = rta.rta_image_max_pixels()
    q, t, x, y, nbr = blob_images(3, P, 21)
    assert_image_parity(gpu_moments(q, t, x, y, nbr, 8.0, 4.0),
                        oracle.image_moments(q, t, x, y, nbr, 8.0, 4.0), x, y, "P max")


# ---------------------------------------------------------------- rta_extract_image
def config_batch(name, n_events, first=0):
    cfg = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(cfg)
    wf = dl0gen.events_cpu(cfg, first, n_events, threads=8)
    x, y, nbr = dl0gen.hex_camera(cfg.n_pixels)
    tp, tb = dl0gen.IMAGE_THRESHOLDS[name]
    return cfg, wf, ped, gain, x, y, nbr, tp, tb


@pytest.mark.parametrize("name,n_events", [("C1", 64), ("C2", 150), ("C3", 201), ("C4", 37)])
def test_fused_on_the_config_shapes(name, n_events):
    import paper_1307_6489_b200 as rta
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch(name, n_events)
    assert rta.rta_image_kernel_name(cfg.n_pixels, cfg.n_samples, cfg.W).startswith("image_tile")
    want = oracle_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    assert (want[0] > 0).sum() > n_events // 2
    got = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    assert_image_parity(got, want, x, y, name + " staged")
    gen = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb, generic=True)
    assert_image_parity(gen, want, x, y, name + " generic")
    # the two device paths run the same cleaning code on the same charges: bit-identical
    for a, b in zip(got, gen):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
    rta.rta_debug_static_schedule(True)
    try:
        st = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    finally:
        rta.rta_debug_static_schedule(False)
    for a, b in zip(got, st):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4"])
def test_fused_equals_extract_then_moments(name):
    """rta_extract_image == rta_extract followed by rta_image_moments, bit for bit."""
    import paper_1307_6489_b200 as rta
    from tests._gpu import alloc_outputs
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch(name, 48, first=100)
    E, P, S = wf.shape
    d_wf, d_ped, d_gain = dev(wf), dev(ped, np.int32), dev(gain, F32)
    outs = alloc_outputs(E * P)
    rta.rta_extract(d_wf, E, P, S, d_ped, d_gain, cfg.W, *outs)
    two = image_outputs(E, P)
    rta.rta_image_moments(outs[2], outs[3], E, P, dev(x), dev(y), dev(nbr), tp, tb, *two)
    one = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    for a, b in zip(one, host(two)):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))


@pytest.mark.parametrize("S,W,P,E", [
    (40, 7, 1, 50), (40, 7, 255, 40), (40, 7, 256, 40), (40, 7, 257, 40), (40, 7, 512, 20),
    (40, 7, 3000, 9),                       # staged, tiles per event 1 .. 12
    (40, 7, 12288, 3),                      # the largest camera (generic: the buffers fill the SM)
    (30, 7, 333, 31), (30, 7, 2, 100),      # 60-byte traces: events 4-byte aligned only
    (25, 4, 1764, 21), (25, 4, 510, 33), (25, 4, 2, 64),   # two traces per thread, 8-byte phases
    (25, 4, 1765, 11),                      # odd camera -> generic
    (128, 8, 2048, 9), (128, 8, 63, 40), (128, 8, 65, 40),
    (33, 5, 400, 20), (16, 16, 100, 20), (7, 1, 1855, 10),  # no specialisation -> generic
])
def test_fused_shapes_and_event_phases(S, W, P, E):
    rng = np.random.default_rng(S * 1000 + P)
    x, y, nbr = dl0gen.hex_camera(P)
    ped = rng.integers(380, 421, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(F32)
    wf = (400 + rng.normal(0, 4, (E, P, S))).round().clip(0, 4095).astype(np.uint16)
    # pulses on clusters of neighbouring pixels so that the cleaning keeps something
    for e in range(E):
        p = int(rng.integers(0, P))
        for n in [p] + [int(v) for v in nbr[p] if v >= 0]:
            wf[e, n, S // 2: S // 2 + max(1, W // 2)] += np.uint16(rng.integers(20, 200))
    want = oracle_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0)
    if P > 1:
        assert (want[0] > 0).any()
    got = gpu_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0)
    assert_image_parity(got, want, x, y, "S=%d P=%d" % (S, P))


@pytest.mark.parametrize("S,W,P,E", [(60, 7, 1855, 12), (96, 8, 300, 25), (33, 5, 400, 20), (50, 8, 37, 60)])
def test_fused_unspecialised_shapes_run_extract_then_moments(S, W, P, E):
    """Shapes without a fused specialisation: rta_extract's runtime-shape kernel
    into a stream-ordered scratch buffer, then the moments kernel (two launches);
    bit-identical to the generic fused kernel, repeatable (the scratch pool is reused)."""
    import paper_1307_6489_b200 as rta
    assert rta.rta_image_kernel_name(P, S, W) == "staged<any>+image_moments"
    rng = np.random.default_rng(S + P)
    x, y, nbr = dl0gen.hex_camera(P)
    ped = rng.integers(380, 421, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(F32)
    wf = (400 + rng.normal(0, 4, (E, P, S))).round().clip(0, 4095).astype(np.uint16)
    for e in range(E):
        p = int(rng.integers(0, P))
        for n in [p] + [int(v) for v in nbr[p] if v >= 0]:
            wf[e, n, S // 2: S // 2 + W // 2] += np.uint16(rng.integers(20, 200))
    want = oracle_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0)
    assert (want[0] > 0).any()
    before = rta.rta_launch_count()
    got = gpu_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0)
    assert rta.rta_launch_count() - before == 2
    assert_image_parity(got, want, x, y, "S=%d P=%d" % (S, P))
    gen = gpu_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0, generic=True)
    again = gpu_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0)
    for a, b, c in zip(got, gen, again):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
        assert np.array_equal(a.view(np.uint8), c.view(np.uint8))
    rta.rta_shutdown()                          # drops the scratch pool; the next call rebuilds it
    after = gpu_extract_image(wf, ped, gain, W, x, y, nbr, 60.0, 30.0)
    for a, b in zip(got, after):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))


@pytest.mark.parametrize("name,n_events", [("C2", 1300), ("C3", 1500), ("C4", 700)])
def test_fused_dense_images_and_buffer_reuse(name, n_events):
    """Pedestals 25 counts too low make almost every pixel pass the picture threshold:
    the cleaning warps become the bound, so the extraction groups wait for free event
    buffers (several events per CTA: every buffer is reused) — the hand-off under the
    opposite load of the sparse configs. Sampled events against the oracle, all events
    against the generic fused kernel."""
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch(name, n_events)
    ped = (ped - 25).astype(np.int32)
    got = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    assert got[0].mean() > 0.5 * cfg.n_pixels
    gen = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb, generic=True)
    for a, b in zip(got, gen):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
    pick = np.r_[0:6, n_events // 2: n_events // 2 + 6, n_events - 6: n_events]
    want = oracle_extract_image(wf[pick], ped, gain, cfg.W, x, y, nbr, tp, tb)
    assert_image_parity(tuple(g[pick] for g in got), want, x, y, name + " dense")


def test_fused_unaligned_waveforms_take_the_generic_kernel():
    import torch
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch("C2", 20)
    want = oracle_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    for off in (1, 3, 4):   # halfwords
        buf = torch.empty(wf.size + 8, dtype=torch.int16, device="cuda")
        d_wf = buf[off: off + wf.size]
        d_wf.copy_(torch.from_numpy(wf.view(np.int16)).reshape(-1))
        got = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb, d_wf=d_wf)
        assert_image_parity(got, want, x, y, "offset %d" % off)


def test_fused_last_event_tail_is_not_overread():
    """C1: 111 300 bytes per event, so the last tile of the last event ends 12
    bytes past a 16-byte boundary; the buffer ends exactly there, followed by a
    guard the kernel must not need (values differ, results must not)."""
    import torch
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch("C1", 5)
    want = oracle_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    n = wf.size
    for guard in (0, -1):
        buf = torch.full((n + 64,), guard, dtype=torch.int16, device="cuda")
        buf[:n].copy_(torch.from_numpy(wf.view(np.int16)).reshape(-1))
        got = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb, d_wf=buf[:n])
        assert_image_parity(got, want, x, y, "tail")


def test_fused_full_uint16_range_and_extreme_calibration():
    rng = np.random.default_rng(77)
    E, P, S, W = 12, 700, 40, 7
    x, y, nbr = dl0gen.hex_camera(P)
    wf = rng.integers(0, 65536, (E, P, S)).astype(np.uint16)
    ped = rng.integers(-2**20, 2**20, P).astype(np.int32)
    gain = rng.uniform(-2, 2, P).astype(F32)
    gain[::50] = np.nan
    gain[1::50] = np.inf
    want = oracle_extract_image(wf, ped, gain, W, x, y, nbr, 1e5, 1e4)
    got = gpu_extract_image(wf, ped, gain, W, x, y, nbr, 1e5, 1e4)
    # (+inf charges make size infinite and the ratios NaN on both sides: assert_image_parity)
    assert_image_parity(got, want, x, y, "extreme")


def test_fused_errors():
    import paper_1307_6489_b200 as rta
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch("C1", 2)
    E, P, S = wf.shape
    d = dict(wf=dev(wf), ped=dev(ped, np.int32), gain=dev(gain, F32), x=dev(x), y=dev(y), nbr=dev(nbr))
    n, par, m = image_outputs(E, P)

    def call(**kw):
        a = dict(d, E=E, P=P, S=S, W=cfg.W, n=n, par=par, m=m)
        a.update(kw)
        rta.rta_extract_image(a["wf"], a["E"], a["P"], a["S"], a["ped"], a["gain"], a["W"], a["x"],
                              a["y"], a["nbr"], tp, tb, a["n"], a["par"], a["m"])
    for kw, status in ((dict(wf=None), rta.RTA_ERR_NULL), (dict(ped=None), rta.RTA_ERR_NULL),
                       (dict(nbr=None), rta.RTA_ERR_NULL), (dict(par=None), rta.RTA_ERR_NULL),
                       (dict(W=0), rta.RTA_ERR_SHAPE), (dict(W=S + 1), rta.RTA_ERR_SHAPE),
                       (dict(E=-2), rta.RTA_ERR_SHAPE), (dict(S=40000, W=1), rta.RTA_ERR_UNSUPPORTED),
                       (dict(P=rta.rta_image_max_pixels() + 1), rta.RTA_ERR_UNSUPPORTED),
                       (dict(wf=d["wf"].data_ptr() + 1), rta.RTA_ERR_ALIGN)):
        with pytest.raises(rta.RtaError) as ei:
            call(**kw)
        assert ei.value.status == status, kw
    call(E=0, wf=None)


# ------------------------------------------------------------ host-fed variants
def test_stream_and_host_variants_match_the_device_call():
    import torch
    import paper_1307_6489_b200 as rta
    cfg, wf, ped, gain, x, y, nbr, tp, tb = config_batch("C2", 100)
    E, P, S = wf.shape
    ref = gpu_extract_image(wf, ped, gain, cfg.W, x, y, nbr, tp, tb)
    ev_bytes = P * S * 2
    pinned = torch.from_numpy(wf.view(np.int16)).pin_memory()
    for src in (pinned, wf):                                    # pinned and pageable sources
        for chunk in (0, 7 * ev_bytes + 5, ev_bytes, 64 * ev_bytes):
            for want_mask in (True, False):
                outs = image_outputs(E, P, want_mask)
                rta.rta_extract_image_stream(src, E, P, S, dev(ped, np.int32), dev(gain, F32), cfg.W,
                                             dev(x), dev(y), dev(nbr), tp, tb, *outs, chunk_bytes=chunk)
                got = host(outs)
                for a, b in zip(got, ref):
                    if a is not None:
                        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
    for chunk in (0, 9 * ev_bytes):
        for want_mask in (True, False):
            n = np.full(E, -7, np.int32)
            par = np.full((E, 8), -7, F32)
            m = np.full((E, P), 9, np.uint8) if want_mask else None
            rta.rta_extract_image_host(wf, E, P, S, ped, gain, cfg.W, x, y, nbr, tp, tb, n, par, m,
                                       chunk_bytes=chunk)
            assert np.array_equal(n, ref[0]) and np.array_equal(par.view(np.int32), ref[1].view(np.int32))
            if want_mask:
                assert np.array_equal(m, ref[2])
    rta.rta_shutdown()


# ------------------------------------------------------ bench-sized, every event
@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_fused_and_two_call_route_at_full_size_every_event(name):
    """BASELINE.json configs at full size, generated on the device, in the launch
    configurations bench.py times: one rta_extract_image (no mask), and rta_extract
    followed by rta_image_moments (with the mask). EVERY event of both is compared
    with the oracle (extraction + cleaning + moments) run on the same bytes, copied
    back in ~1 GB slabs, on all host cores."""
    import torch
    import paper_1307_6489_b200 as rta
    from tests._full import alloc_filled_outputs, slabs, split_events
    cfg = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(cfg)
    x, y, nbr = dl0gen.hex_camera(cfg.n_pixels)
    tp, tb = dl0gen.IMAGE_THRESHOLDS[name]
    E, P, S = cfg.n_events, cfg.n_pixels, cfg.n_samples
    d_wf = torch.empty((E, P, S), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(cfg, d_wf.data_ptr(), 0, E, torch.cuda.current_stream().cuda_stream)
    cam = (dev(x), dev(y), dev(nbr), tp, tb)
    d_ped, d_gain = dev(ped, np.int32), dev(gain, F32)
    fused = image_outputs(E, P, mask=False)
    before = rta.rta_launch_count()
    rta.rta_extract_image(d_wf, E, P, S, d_ped, d_gain, cfg.W, *cam, *fused)
    assert rta.rta_launch_count() == before + 1
    per_trace = alloc_filled_outputs(E * P)
    two = image_outputs(E, P, mask=True)
    rta.rta_extract(d_wf, E, P, S, d_ped, d_gain, cfg.W, *per_trace)
    rta.rta_image_moments(per_trace[2], per_trace[3], E, P, *cam, *two)
    fn, fpar, _ = host(fused)
    tn, tpar, tmask = host(two)
    del per_trace, two, fused
    assert ((fpar == 0).all(1) == (fn == 0)).all()            # positive thresholds: empty <=> zero
    done = 0
    for e0, k in slabs(E, P * S * 2):
        wf = d_wf[e0:e0 + k].cpu().numpy().view(np.uint16)
        want = split_events(k, lambda a, b: oracle_extract_image(wf[a:b], ped, gain, cfg.W, x, y,
                                                                 nbr, tp, tb))
        what = "%s events %d..%d" % (name, e0, e0 + k)
        assert_image_parity((fn[e0:e0 + k], fpar[e0:e0 + k], None), want, x, y, what + " fused")
        assert_image_parity((tn[e0:e0 + k], tpar[e0:e0 + k], tmask[e0:e0 + k]), want, x, y,
                            what + " extract + moments")
        done += k
    assert done == E
