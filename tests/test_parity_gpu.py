"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by
element on the same seeded inputs. Bar = BASELINE.json:north_star: out_sum and
out_start bit-exact, charge within relative 1e-6, peak time within absolute
1e-4 samples. (The kernels are designed to be bit-identical on the floats too;
`bit_identical` is asserted where the design guarantees it.)"""
import itertools
import json
import os

import numpy as np
import pytest

import dl0gen
import oracle
from tests._checks import check_invariants
from tests._full import alloc_filled_outputs, compare_every_event, slabs
from tests._gpu import alloc_outputs, assert_parity, bit_identical, run_gpu, to_dev_u16

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden", "hand_worked.json")
SHAPES = [(30, 7), (40, 7), (25, 4), (128, 8)]          # specialised tile kernels


def both(wf, ped, gain, W):
    want = oracle.extract(wf, ped, gain, W)
    for generic in (False, True):
        got = run_gpu(wf, ped, gain, W, generic=generic)
        assert_parity(got, want, "generic" if generic else "dispatch")
        assert bit_identical(got, want)
    return want


def test_hand_worked_fixtures_on_gpu():
    for c in json.load(open(GOLD))["cases"]:
        E, P, S = c["n_events"], c["n_pixels"], c["n_samples"]
        wf = np.array(c["wf"], np.uint16).reshape(E, P, S)
        got = run_gpu(wf, np.array(c["pedestal"], np.int32),
                      np.array(c["gain"], np.float32), c["W"])
        assert got[0].tolist() == c["out_sum"] and got[1].tolist() == c["out_start"]
        assert got[2].tolist() == [float(np.float32(v)) for v in c["out_charge"]]
        want_t = [float(np.float32(np.float64(n) / np.float64(d)))
                  for n, d in zip(c["time_num"], c["time_den"])]
        assert got[3].tolist() == want_t


@pytest.mark.parametrize("S,Ws,values,ped", [
    (4, [2], [9, 10, 11], 10), (5, [1, 2, 3, 4, 5], [0, 1, 2, 3], 1), (12, [3], [0, 1], 0)])
def test_exhaustive_tiny_traces(S, Ws, values, ped):
    """Pin P10 through the GPU: every trace over a small alphabet."""
    tr = np.array(list(itertools.product(values, repeat=S)), np.uint16)
    n = len(tr)
    P = 4 if n % 4 == 0 else 3
    wf = tr.reshape(n // P, P, S)
    pedv = np.full(P, ped, np.int32)
    gain = np.linspace(0.9, 1.1, P).astype(np.float32)
    for W in Ws:
        both(wf, pedv, gain, W)


@pytest.mark.parametrize("S,W", SHAPES)
def test_exhaustive_tie_patterns_in_specialised_shapes(S, W):
    """All 2^12 on/off patterns of a 12-sample region placed at the start, the
    middle and the end of the trace — every tie pattern the key must resolve."""
    pats = np.array(list(itertools.product([0, 1], repeat=12)), np.uint16)  # 4096
    for off in (0, (S - 12) // 2, S - 12):
        tr = np.full((4096, S), 100, np.uint16)
        tr[:, off:off + 12] += pats * 5
        wf = tr.reshape(64, 64, S)
        ped = np.full(64, 100, np.int32)
        ped[::3] = 101                                   # some negative samples
        both(wf, ped, np.linspace(0.9, 1.1, 64).astype(np.float32), W)


@pytest.mark.parametrize("S,W", SHAPES)
def test_closed_forms_in_specialised_shapes(S, W):
    P = 3
    ped = np.array([400, 0, 4095], np.int32)
    gain = np.array([1.0, 0.5, 1.0625], np.float32)
    # P1 constant traces: below, at and above pedestal
    for c in (0, 400, 4095, 65535):
        wf = np.full((5, P, S), c, np.uint16)
        s, t, q, tm = run_gpu(wf, ped, gain, W)
        assert (t == 0).all()
        assert (s.reshape(5, P) == W * (c - ped.astype(np.int64))).all()
        assert (tm == np.float32((W - 1) / 2)).all()
        assert (q.reshape(5, P) == (W * (c - ped.astype(np.float64)) * gain).astype(np.float32)).all()
    # P2 delta at every position, one event per position
    A = 57
    wf = np.broadcast_to(ped.astype(np.uint16)[None, :, None], (S, P, S)).copy()
    for k in range(S):
        wf[k, :, k] += A
    s, t, q, tm = run_gpu(wf, ped, gain, W)
    ks = np.repeat(np.arange(S), P)
    assert (s == A).all()
    assert (t == np.maximum(0, ks - W + 1)).all()
    assert (tm == ks.astype(np.float32)).all()
    assert (q == (A * np.tile(gain, S).astype(np.float64)).astype(np.float32)).all()
    both(wf, ped, gain, W)


@pytest.mark.parametrize("S,W", SHAPES + [(31, 5), (64, 16), (7, 7), (9, 1), (200, 3)])
@pytest.mark.parametrize("n_traces_shape", [(1, 1), (3, 5), (7, 37), (2, 129), (5, 257), (4, 1031)])
def test_random_full_uint16_range_and_ragged_sizes(S, W, n_traces_shape):
    """Any uint16 value (R13), sizes around the tile boundaries (128/256/512
    traces) and pedestals of both signs and beyond the samples (R2)."""
    E, P = n_traces_shape
    rng = np.random.default_rng(S * 7919 + W * 31 + E * P)
    wf = rng.integers(0, 65536, size=(E, P, S)).astype(np.uint16)
    wf[rng.random((E, P)) < 0.2] = 65535                  # key overflow guard: all-max traces
    ped = rng.integers(-70000, 70000, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    both(wf, ped, gain, W)


@pytest.mark.parametrize("S,W", SHAPES)
def test_extreme_pedestals_take_the_wide_path(S, W):
    """|pedestal| up to 2^30: int64 numerator and the double-precision branch."""
    rng = np.random.default_rng(S)
    E, P = 3, 300
    wf = rng.integers(0, 65536, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(-2 ** 30, 2 ** 30, P).astype(np.int32)
    ped[:50] = rng.integers(-2 ** 26, 2 ** 26, 50)
    gain = rng.uniform(-3, 3, P).astype(np.float32)
    gain[0], gain[1], gain[2] = np.float32("nan"), np.float32("inf"), np.float32(1e-42)
    want = oracle.extract(wf, ped, gain, W)
    got = run_gpu(wf, ped, gain, W)
    assert (got[0] == want[0]).all() and (got[1] == want[1]).all()
    assert bit_identical(got, want)


@pytest.mark.parametrize("S,W", SHAPES + [(33, 5)])
def test_pedestals_at_the_edges_of_the_sample_range(S, W):
    """finish_trace computes in 32 bits when 0 <= pedestal <= 65535 and in 64 bits
    otherwise: both sides of both edges, on full-range samples (largest sums and
    numerators the ABI guard allows) and on all-0 / all-65535 traces."""
    rng = np.random.default_rng(S + 1000)
    E = 4
    edge = np.array([0, 1, 65534, 65535, 65536, 65537, -1, -2, 32767, 32768, 40000, 2 ** 31 - 1,
                     -2 ** 31, 70000, -65535], np.int32)
    P = len(edge) * 8
    ped = np.tile(edge, 8)
    wf = rng.integers(0, 65536, size=(E, P, S)).astype(np.uint16)
    wf[0, :, :] = 65535
    wf[1, :, :] = 0
    wf[2, :, S // 2:] = 65535                             # late plateau: largest time numerators
    gain = rng.uniform(0.5, 2, P).astype(np.float32)
    want = oracle.extract(wf, ped, gain, W)
    for generic in (False, True):
        got = run_gpu(wf, ped, gain, W, generic=generic)
        assert (got[0] == want[0]).all() and (got[1] == want[1]).all()
        assert bit_identical(got, want)


def test_unaligned_input_agrees():
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS["C1"]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 0, 8)
    want = oracle.extract(wf, ped, gain, c.W)
    flat = torch.empty(wf.size + 8, dtype=torch.int16, device="cuda")
    flat[1:1 + wf.size] = torch.from_numpy(wf.reshape(-1).view(np.int16)).cuda()
    view = flat[1:1 + wf.size]                            # 2-byte aligned only
    assert view.data_ptr() % 16 != 0
    d_ped = torch.from_numpy(ped).cuda()
    d_gain = torch.from_numpy(gain).cuda()
    outs = alloc_outputs(8 * c.n_pixels)
    rta.rta_extract(view, 8, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs)
    torch.cuda.synchronize()
    assert bit_identical(tuple(o.cpu().numpy() for o in outs), want)


def test_odd_output_alignment_takes_scalar_stores():
    """S=25 pairs traces per thread and prefers 8-byte stores; outputs that are
    only 4-byte aligned must still be written correctly."""
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS["C3"]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 0, 3)
    n = 3 * c.n_pixels
    want = oracle.extract(wf, ped, gain, c.W)
    d_wf = to_dev_u16(wf)
    bufs = [torch.zeros(n + 1, dtype=dt, device="cuda")
            for dt in (torch.int32, torch.int32, torch.float32, torch.float32)]
    outs = [b[1:] for b in bufs]
    assert outs[0].data_ptr() % 8 == 4
    rta.rta_extract(d_wf, 3, c.n_pixels, c.n_samples, torch.from_numpy(ped).cuda(),
                    torch.from_numpy(gain).cuda(), c.W, *outs)
    torch.cuda.synchronize()
    assert bit_identical(tuple(o.cpu().numpy() for o in outs), want)
    assert all(float(b[0]) == 0 for b in bufs)            # nothing written before the view


def test_C1_full_parity():
    c = dl0gen.CONFIGS["C1"]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, threads=4)
    want = both(wf, ped, gain, c.W)
    check_invariants(wf, ped, gain, c.W, *want)


@pytest.mark.parametrize("name,n_ev", [("C2", 23), ("C3", 19), ("C4", 11)])
def test_config_models_small_batches(name, n_ev):
    """The C2-C4 signal models at sizes the oracle finishes at once: several
    tiles per CTA plus a ragged tail (n_traces is not a multiple of the tile)."""
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 100, n_ev, threads=4)
    both(wf, ped, gain, c.W)


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_full_size_configs_every_event_against_oracle(name):
    """BASELINE.json's full sizes, in the launch configuration bench.py times
    (one rta_extract over the whole device-resident batch): generate on the
    GPU, extract into sentinel-filled outputs, then compare EVERY event with the
    oracle run on the same bytes (copied back in ~1 GB slabs, all host cores):
    a tile dropped or duplicated anywhere in the launch fails here. A few event
    blocks are also regenerated on the host (device bytes == host generator's
    bytes) and put through the size-independent invariants (P8/P9)."""
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    d_wf = torch.empty((c.n_events, c.n_pixels, c.n_samples), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(c, d_wf.data_ptr(), 0, c.n_events, torch.cuda.current_stream().cuda_stream)
    d_ped = torch.from_numpy(ped).cuda()
    d_gain = torch.from_numpy(gain).cuda()
    outs = alloc_filled_outputs(c.n_traces)
    before = rta.rta_launch_count()
    rta.rta_extract(d_wf, c.n_events, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs)
    torch.cuda.synchronize()
    assert rta.rta_launch_count() == before + 1
    n = compare_every_event(
        c.n_events, c.n_pixels, slabs(c.n_events, c.n_pixels * c.n_samples * 2),
        lambda e0, k: d_wf[e0:e0 + k].cpu().numpy().view(np.uint16),
        lambda wf, a, b: oracle.extract(wf[a:b], ped, gain, c.W), outs)
    assert n == c.n_events
    rng = np.random.default_rng(5)
    for e0 in [0, c.n_events - 12] + sorted(rng.integers(12, c.n_events - 24, 2).tolist()):
        wf = dl0gen.events_cpu(c, e0, 12, threads=4)
        assert (d_wf[e0:e0 + 12].cpu().numpy().view(np.uint16) == wf).all()
        lo, hi = e0 * c.n_pixels, (e0 + 12) * c.n_pixels
        got = tuple(o[lo:hi].cpu().numpy() for o in outs)
        assert_parity(got, oracle.extract(wf, ped, gain, c.W), "%s events %d.." % (name, e0))
        check_invariants(wf, ped, gain, c.W, *got)


# ---- tile scheduler (dynamic by default) ---------------
@pytest.mark.parametrize("name,n_ev", [("C1", 64), ("C2", 301), ("C3", 257), ("C4", 97)])
def test_static_and_dynamic_tile_schedules_agree(name, n_ev):
    """The tile->CTA map must not change any result: run the staged kernel with
    the dynamic scheduler (default) and with the static round-robin."""
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 5, n_ev, threads=4)
    want = oracle.extract(wf, ped, gain, c.W)
    try:
        for static in (True, False, True, False):
            rta.rta_debug_static_schedule(static)
            got = run_gpu(wf, ped, gain, c.W)
            assert bit_identical(got, want), "static=%s" % static
    finally:
        rta.rta_debug_static_schedule(False)


def test_back_to_back_launches_reuse_the_scheduler_words():
    """The dynamic scheduler's counters are left zeroed by each launch: many
    launches in a row on one stream, alternating shapes and sizes."""
    import torch
    import paper_1307_6489_b200 as rta
    cases = []
    for name, n_ev in [("C2", 120), ("C4", 40), ("C3", 77), ("C2", 3), ("C1", 64), ("C2", 119)]:
        c = dl0gen.CONFIGS[name]
        ped, gain = dl0gen.calib(c)
        wf = dl0gen.events_cpu(c, 11, n_ev, threads=4)
        cases.append((c, n_ev, to_dev_u16(wf), torch.from_numpy(ped).cuda(),
                      torch.from_numpy(gain).cuda(), alloc_outputs(n_ev * c.n_pixels),
                      oracle.extract(wf, ped, gain, c.W)))
    for _ in range(3):
        for c, n_ev, d_wf, d_ped, d_gain, outs, want in cases:      # no sync in between
            rta.rta_extract(d_wf, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs)
    torch.cuda.synchronize()
    for c, n_ev, d_wf, d_ped, d_gain, outs, want in cases:
        assert bit_identical(tuple(o.cpu().numpy() for o in outs), want)


def test_concurrent_streams_have_their_own_scheduler_words():
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS["C2"]
    ped, gain = dl0gen.calib(c)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    streams = [torch.cuda.Stream() for _ in range(6)]
    jobs = []
    for i, st in enumerate(streams):
        n_ev = 150 + 17 * i
        wf = dl0gen.events_cpu(c, 1000 * i, n_ev, threads=4)
        jobs.append((st, n_ev, to_dev_u16(wf), alloc_outputs(n_ev * c.n_pixels),
                     oracle.extract(wf, ped, gain, c.W)))
    torch.cuda.synchronize()
    for _ in range(4):
        for st, n_ev, d_wf, outs, want in jobs:
            rta.rta_extract(d_wf, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs,
                            stream=st)
    torch.cuda.synchronize()
    for st, n_ev, d_wf, outs, want in jobs:
        assert bit_identical(tuple(o.cpu().numpy() for o in outs), want)


def test_cuda_graph_capture_and_replay():
    """rta_extract is capturable (a captured launch takes the static tile schedule)."""
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS["C2"]
    n_ev = 200
    ped, gain = dl0gen.calib(c)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    wfs = [dl0gen.events_cpu(c, 300 * i, n_ev, threads=4) for i in range(3)]
    d_wf = to_dev_u16(wfs[0])
    outs = alloc_outputs(n_ev * c.n_pixels)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):                         # warm-up on the capture stream
        rta.rta_extract(d_wf, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        rta.rta_extract(d_wf, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs)
    for wf in wfs[::-1]:
        d_wf.copy_(to_dev_u16(wf))
        for o in outs:
            o.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert bit_identical(tuple(o.cpu().numpy() for o in outs),
                             oracle.extract(wf, ped, gain, c.W))


@pytest.mark.parametrize("S,W,warm", [(52, 6, True), (54, 9, False), (2048, 12, False)])
def test_cuda_graph_capture_of_shapes_without_an_ahead_of_time_kernel(S, W, warm):
    """A shape whose specialisation is compiled at first use: captured after an eager call the
    graph holds the compiled kernel; captured as the very first call of the shape nothing is
    compiled inside the capture (the runtime-shape kernel is recorded instead). Long traces
    (the segment kernel) are capturable too. Replays on other data must match the oracle."""
    import torch
    import paper_1307_6489_b200 as rta
    rng = np.random.default_rng(S)
    E, P = 3, 1500 if S < 1000 else 40
    ped = rng.integers(0, 600, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    wfs = [rng.integers(0, 4096, size=(E, P, S)).astype(np.uint16) for _ in range(3)]
    d_wf = to_dev_u16(wfs[0])
    outs = alloc_outputs(E * P)
    side = torch.cuda.Stream()
    if warm:
        with torch.cuda.stream(side):
            rta.rta_extract(d_wf, E, P, S, d_ped, d_gain, W, *outs)
        torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        rta.rta_extract(d_wf, E, P, S, d_ped, d_gain, W, *outs)
    for wf in wfs[::-1]:
        d_wf.copy_(to_dev_u16(wf))
        for o in outs:
            o.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert bit_identical(tuple(o.cpu().numpy() for o in outs), oracle.extract(wf, ped, gain, W))
    # and eagerly afterwards (the shape that was first seen inside a capture compiles now)
    rta.rta_extract(d_wf, E, P, S, d_ped, d_gain, W, *outs)
    torch.cuda.synchronize()
    assert bit_identical(tuple(o.cpu().numpy() for o in outs), oracle.extract(wfs[0], ped, gain, W))


def test_graph_replays_run_next_to_eager_calls_and_to_each_other():
    """Two graphs captured on ONE stream, replayed on two other streams at the
    same time as eager calls on the capture stream, 50 rounds: a captured launch
    must not share tile-scheduler state with anything (it takes the static
    round-robin), or tiles are skipped and outputs stay unwritten. Batches are
    small enough for several grids to be resident together."""
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS["C2"]
    ped, gain = dl0gen.calib(c)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    A, B, C = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    jobs = []
    for i, n_ev in enumerate((37, 41, 29)):               # graph 1, graph 2, eager
        wf = dl0gen.events_cpu(c, 500 * i, n_ev, threads=4)
        jobs.append((n_ev, to_dev_u16(wf), alloc_outputs(n_ev * c.n_pixels),
                     oracle.extract(wf, ped, gain, c.W)))

    def call(j):
        n_ev, d_wf, outs, _ = jobs[j]
        rta.rta_extract(d_wf, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs)
    with torch.cuda.stream(A):                            # warm-up on the capture stream
        call(2)
    torch.cuda.synchronize()
    graphs = []
    for j in (0, 1):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=A):
            call(j)
        graphs.append(g)
    for rnd in range(50):
        for n_ev, d_wf, outs, want in jobs:
            for o in outs:
                o.fill_(-3)
        torch.cuda.synchronize()
        for _ in range(4):                                # several of each in flight
            with torch.cuda.stream(B):
                graphs[0].replay()
            with torch.cuda.stream(C):
                graphs[1].replay()
            with torch.cuda.stream(A):
                call(2)
        torch.cuda.synchronize()
        for j, (n_ev, d_wf, outs, want) in enumerate(jobs):
            assert bit_identical(tuple(o.cpu().numpy() for o in outs), want), (rnd, j)


@pytest.mark.parametrize("S,W,kernel", [(25, 4, "tile<S=25,W=4>"), (2, 1, "staged<jit>"), (2, 1, "staged<any>")])
def test_largest_trace_count(S, W, kernel):
    """n_events * n_pixels just below the ABI guard 2^31 (R14): the 32-bit trace
    indices, tile counts and the scheduler must hold up to the last trace. Sampled
    blocks of traces (first, middle, last tiles and the ragged tail) against the oracle."""
    import torch
    import paper_1307_6489_b200 as rta
    E, P = 1049088, 2047                       # 2 147 483 136 traces, 512 short of 2^31
    n = E * P
    need = n * (2 * S + 16) + (2 << 30)
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < need:
        pytest.skip("needs %.0f GB of device memory" % (need / 1e9))
    if kernel == "staged<any>":
        rta.rta_debug_jit(False)                # the runtime-shape kernel, as without libnvrtc
    try:
        assert rta.rta_kernel_name(S, W) == kernel
        _largest_trace_count(S, W, E, P, n)
    finally:
        rta.rta_debug_jit(True)


def _largest_trace_count(S, W, E, P, n):
    import torch
    import paper_1307_6489_b200 as rta
    wf = torch.empty(n * S, dtype=torch.int16, device="cuda")
    step = 1 << 28
    gen = torch.Generator(device="cuda").manual_seed(5)
    for a in range(0, n * S, step):
        b = min(a + step, n * S)
        wf[a:b] = torch.randint(0, 4096, (b - a,), generator=gen, device="cuda", dtype=torch.int16)
    rng = np.random.default_rng(9)
    ped = rng.integers(0, 600, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    outs = [torch.full((n,), f, dtype=dt, device="cuda") for f, dt in
            zip((-7, -7, -7.0, -7.0), (torch.int32, torch.int32, torch.float32, torch.float32))]
    rta.rta_extract(wf, E, P, S, torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda(), W, *outs)
    torch.cuda.synchronize()
    assert int((outs[1] < 0).sum()) == 0        # every trace was written (a start is never negative)
    blocks = [0, 1 << 20, n // 2 - 333, (1 << 31) - (1 << 16), n - 5000, n - 700]
    for g0 in blocks:
        m = min(3001, n - g0)
        sub = wf[g0 * S:(g0 + m) * S].cpu().numpy().view(np.uint16).reshape(1, m, S)
        pix = (g0 + np.arange(m)) % P
        want = oracle.extract(sub, ped[pix], gain[pix], W)
        got = tuple(o[g0:g0 + m].cpu().numpy() for o in outs)
        assert bit_identical(got, want), g0
    del wf, outs
    torch.cuda.empty_cache()
