"""GPU parity of mixed-camera (ragged) batches: the
plan + rta_extract_ragged against oracle/rta_oracle_ragged.cpp, element by
element. Integers bit-exact, floats bit-identical (same construction as the
uniform path). Entries no block writes must stay untouched."""
import json
import os

import numpy as np
import pytest

import oracle
from tests._gpu import assert_parity, bit_identical
from tests._ragged import make_batch

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden", "ragged.json")
FILL = (-7, -7, -7.0, -7.0)


def run_gpu(b, wf=None, wf_shift=0, streams=1, static=False, serial=False, jit=True, jit_at_launch=None):
    """wf_shift: place the waveform buffer that many samples into a 256-byte-aligned
    allocation (so block alignments change without touching the tables)."""
    import torch
    import paper_1307_6489_b200 as rta
    wf = b.wf if wf is None else wf
    buf = torch.zeros(wf.size + wf_shift + 8, dtype=torch.int16, device="cuda")
    buf[wf_shift:wf_shift + wf.size] = torch.from_numpy(wf.view(np.int16)).cuda()
    d_wf = buf[wf_shift:]
    d_ped = torch.from_numpy(b.pedestal).cuda()
    d_gain = torch.from_numpy(b.gain).cuda()
    n = b.n_out + 3
    outs = [torch.full((n,), f, dtype=dt, device="cuda")
            for f, dt in zip(FILL, (torch.int32, torch.int32, torch.float32, torch.float32))]
    # the hooks live in librta_testing.so; while one is on the binding routes every
    # call there, so the plan is made and destroyed under the same switches
    # jit: are the run-time specialisations (NVRTC) on when the plan is made (the plan cuts the
    # tiles of an unspecialised shape for the kernel it expects); jit_at_launch: and at the launch
    rta.rta_debug_static_schedule(static)
    rta.rta_debug_serial_ragged(serial)
    rta.rta_debug_jit(jit)
    plan = rta.rta_ragged_plan_create(*b.tables())
    try:
        rta.rta_debug_jit(jit if jit_at_launch is None else jit_at_launch)
        before = rta.rta_launch_count()
        rta.rta_extract_ragged(plan, d_wf, d_ped, d_gain, *outs)
        torch.cuda.synchronize()
        assert rta.rta_launch_count() - before == rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_LAUNCHES)
        assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_TRACES) == sum(
            b.tel_n_pixels[k] for k in b.blk_tel)
    finally:
        rta.rta_ragged_plan_destroy(plan)
        rta.rta_debug_static_schedule(False)
        rta.rta_debug_serial_ragged(False)
        rta.rta_debug_jit(True)
    return tuple(o.cpu().numpy() for o in outs)


def check(b, **kw):
    want = oracle.extract_ragged(b.wf, *b.tables(), b.pedestal, b.gain, b.n_out + 3, fill=FILL)
    got = run_gpu(b, **kw)
    written = want[1] != FILL[1]                            # a real out_start is never negative
    assert_parity(tuple(g[written] for g in got), tuple(w[written] for w in want))
    assert bit_identical(got, want)                         # including the untouched entries
    return want


def test_hand_assembled_fixture_on_gpu():
    import torch
    import paper_1307_6489_b200 as rta
    g = json.load(open(GOLD))
    d_wf = torch.from_numpy(np.array(g["wf"], np.uint16).view(np.int16)).cuda()
    outs = [torch.full((g["n_out"],), f, dtype=dt, device="cuda")
            for f, dt in zip(FILL, (torch.int32, torch.int32, torch.float32, torch.float32))]
    plan = rta.rta_ragged_plan_create(g["tel_n_pixels"], g["tel_n_samples"], g["tel_W"], g["tel_calib_offset"],
                                      g["blk_tel"], g["blk_wf_offset"], g["blk_out_offset"])
    rta.rta_extract_ragged(plan, d_wf, torch.tensor(g["pedestal"], dtype=torch.int32).cuda(),
                           torch.tensor(g["gain"], dtype=torch.float32).cuda(), *outs)
    torch.cuda.synchronize()
    rta.rta_ragged_plan_destroy(plan)
    s, t, q, tm = (o.cpu().numpy() for o in outs)
    n = len(g["out_sum"])
    assert s[:n].tolist() == g["out_sum"] and t[:n].tolist() == g["out_start"]
    assert q[:n].tolist() == g["out_charge"]
    assert tm[:n].tolist() == [float(np.float32(np.float64(a) / np.float64(b)))
                               for a, b in zip(g["time_num"], g["time_den"])]
    assert s[n] == FILL[0] and tm[n] == FILL[3]


SPECIAL = [((300, 30, 7), 1), ((523, 40, 7), 2), ((1031, 25, 4), 1), ((67, 128, 8), 2)]
MIXED = SPECIAL + [((5, 9, 3), 1), ((40, 31, 5), 1), ((3, 200, 3), 1), ((700, 7, 7), 1)]


@pytest.mark.parametrize("seed", [0, 1])
@pytest.mark.parametrize("gap,align", [(0, 1), (0, 8), (5, 1), (6, 2), (9, 8)])
def test_random_mixed_batches(seed, gap, align):
    """Specialised and generic shapes in one batch, blocks larger and smaller
    than a tile, odd pixel counts, every source alignment (2, 4, 8, 16 bytes)."""
    b = make_batch(MIXED, n_events=5, seed=seed, gap=gap, align=align, shuffle_out=bool(seed))
    check(b)


# shapes without a specialisation, one per case of the runtime-shape kernel
# (word stride odd / 2 mod 4 / 0 mod 4, padded layout, odd S, blocks of several tiles)
ANY_SHAPE = [((700, 60, 7), 2), ((300, 96, 8), 1), ((129, 64, 16), 1), ((77, 33, 5), 2),
             ((1031, 50, 8), 1), ((515, 40, 5), 1), ((9, 128, 10), 2), ((3, 576, 12), 1)]


@pytest.mark.parametrize("gap,align", [(0, 8), (5, 1), (6, 2), (9, 8)])
@pytest.mark.parametrize("wf_shift", [0, 1, 2])
def test_unspecialised_shapes_take_the_runtime_shape_kernel(gap, align, wf_shift):
    """extract_ragged_dyn_kernel (run-time specialisations off): every ingest path (TMA /
    16-byte cp.async into the padded layout, 4-byte cp.async, halfwords) for every
    bank-conflict class."""
    b = make_batch(ANY_SHAPE, n_events=4, seed=3 + gap, gap=gap, align=align)
    check(b, wf_shift=wf_shift, jit=False)
    check(b, wf_shift=wf_shift, static=True, jit=False)


@pytest.mark.parametrize("gap,align", [(0, 8), (5, 1), (6, 2), (9, 8)])
@pytest.mark.parametrize("wf_shift", [0, 1, 2])
def test_unspecialised_shapes_take_the_run_time_specialisation(gap, align, wf_shift):
    """The tile-table kernel compiled for the shape at first use (units up to 320 bytes; the
    576-sample camera of the batch keeps the runtime-shape kernel): the same batches, both
    tile schedules; and a plan cut for the specialisation's tiles that is launched after the
    compiler has gone away (the runtime-shape kernel with as many threads as a tile has units),
    and the other way round."""
    b = make_batch(ANY_SHAPE, n_events=4, seed=3 + gap, gap=gap, align=align)
    check(b, wf_shift=wf_shift)
    check(b, wf_shift=wf_shift, static=True)
    check(b, wf_shift=wf_shift, jit=True, jit_at_launch=False)
    check(b, wf_shift=wf_shift, jit=False, jit_at_launch=True)


@pytest.mark.parametrize("wf_shift", [0, 1, 2, 3, 4, 6])
def test_every_alignment_of_the_waveform_buffer(wf_shift):
    """The same tables over a buffer that starts 0..12 bytes off a 16-byte boundary:
    the TMA, 4-byte cp.async and halfword ingest paths must agree."""
    b = make_batch(SPECIAL, n_events=4, seed=7, align=8, trigger=1.0)
    check(b, wf_shift=wf_shift)


def test_static_and_dynamic_tile_schedules_agree():
    b = make_batch(SPECIAL, n_events=6, seed=9, gap=3)
    check(b, static=True)
    check(b, static=False)


def test_side_streams_and_serial_launches_agree():
    """One launch per camera shape: forked onto library-owned side streams
    (default) or one after the other on the caller's stream; also on a
    non-default caller stream followed by dependent work on that stream."""
    import torch
    b = make_batch(SPECIAL, n_events=6, seed=21, gap=3)
    assert len({(b.tel_n_samples[k], b.tel_W[k]) for k in b.blk_tel}) > 1
    check(b, serial=True)
    check(b, serial=False)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        for _ in range(3):
            check(b)


def test_config_cameras_full_blocks():
    """Whole C1/C2/C3/C4 cameras (1855, 1855, 1764, 2048 pixels) as blocks: several
    full tiles plus a partial one per block."""
    b = make_batch([("C1", 1), ("C2", 2), ("C3", 2), ("C4", 1)], n_events=4, seed=2, trigger=0.7, align=8)
    check(b)
    b = make_batch([("C2", 1), ("C3", 3)], n_events=5, seed=3, trigger=1.0, align=1)   # MST blocks 8-byte aligned only
    check(b)


def test_uniform_batch_through_the_ragged_path_equals_rta_extract():
    import torch
    import dl0gen
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS["C2"]
    E = 9
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 50, E, threads=4)
    want = oracle.extract(wf, ped, gain, c.W)
    P, S = c.n_pixels, c.n_samples
    plan = rta.rta_ragged_plan_create([P], [S], [c.W], [0], [0] * E, [e * P * S for e in range(E)],
                                      [e * P for e in range(E)])
    d_wf = torch.from_numpy(wf.view(np.int16)).cuda()
    outs = [torch.empty(E * P, dtype=dt, device="cuda")
            for dt in (torch.int32, torch.int32, torch.float32, torch.float32)]
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    torch.cuda.synchronize()
    for st in (s1, s2, s1):                                 # a plan is reusable, from any stream
        for o in outs:
            o.zero_()
        torch.cuda.synchronize()
        rta.rta_extract_ragged(plan, d_wf, d_ped, d_gain, *outs, stream=st)
        torch.cuda.synchronize()
        assert bit_identical(tuple(o.cpu().numpy() for o in outs), want)
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_LAUNCHES) == 1
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_WF_BYTES) == wf.nbytes
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_WF_END_BYTES) == wf.nbytes
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_OUT_END) == E * P
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_TILES) == E * -(-P // 256)
    rta.rta_ragged_plan_destroy(plan)


def test_bench_sized_mixed_array_every_block_against_oracle():
    """The mixed array bench.py times (1000 events x (4 LST-, 10 MST-, 6 SST-like
    telescopes), every event triggers all, blocks on 16-byte boundaries): generated
    on the GPU, one rta_extract_ragged into sentinel-filled outputs, then EVERY block
    against oracle.extract_ragged on the same bytes (copied back in slabs of whole
    events, all host cores). A few blocks are also regenerated on the host."""
    import torch
    import dl0gen
    import paper_1307_6489_b200 as rta
    from tests._full import alloc_filled_outputs, bits_equal, first_mismatch, slabs, split_events
    m = dl0gen.MixedArray(n_events=1000)
    ped, gain = m.calib()
    d_wf = torch.zeros(m.n_samples_total, dtype=torch.int16, device="cuda")
    m.fill_cuda(torch, d_wf)
    outs = alloc_filled_outputs(m.n_traces)
    plan = rta.rta_ragged_plan_create(*m.tables())
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_LAUNCHES) == 3
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_WF_BYTES) == m.wf_bytes
    rta.rta_extract_ragged(plan, d_wf, torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda(), *outs)
    torch.cuda.synchronize()
    rta.rta_ragged_plan_destroy(plan)
    n_slots, tpe, stride = len(m.slots), m.traces_per_event, m.event_stride

    def oracle_events(wf, a, b):                       # events [a, b) of the slab `wf`
        idx = range((b - a) * n_slots)
        tel = [i % n_slots for i in idx]
        wo = [(i // n_slots) * stride + m.slot_offset[i % n_slots] for i in idx]
        oo = [(i // n_slots) * tpe + m.slot_out[i % n_slots] for i in idx]
        return oracle.extract_ragged(wf[a * stride:b * stride], m.tel_n_pixels, m.tel_n_samples,
                                     m.tel_W, m.tel_calib_offset, tel, wo, oo, ped, gain,
                                     (b - a) * tpe)
    done = 0
    for e0, k in slabs(m.n_events, stride * 2):
        wf = d_wf[e0 * stride:(e0 + k) * stride].cpu().numpy().view(np.uint16)
        want = split_events(k, lambda a, b: oracle_events(wf, a, b))
        got = tuple(o[e0 * tpe:(e0 + k) * tpe].cpu().numpy() for o in outs)
        assert bits_equal(got, want), "events %d..%d: %s" % (e0, e0 + k, first_mismatch(got, want))
        done += k
    assert done == m.n_events
    rng = np.random.default_rng(8)
    for e, j in [(0, 0), (m.n_events - 1, n_slots - 1)] + [
            (int(rng.integers(0, m.n_events)), int(rng.integers(0, n_slots))) for _ in range(6)]:
        blk = m.block_cpu(e, j)
        P, S = m.tel_n_pixels[j], m.tel_n_samples[j]
        w0 = e * stride + m.slot_offset[j]
        assert (d_wf[w0:w0 + P * S].cpu().numpy().view(np.uint16) == blk.ravel()).all()
