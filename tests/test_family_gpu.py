"""GPU parity of the extractor family (rta_extract_fixed / _local_peak / _fir;
SURVEY.md §8(f) NEXT-1) against oracle/rta_oracle_windows.cpp, element by
element on the same seeded inputs. Same bar as the sliding extractor: integers
bit-exact, charge rel 1e-6, time abs 1e-4 — and, by construction, bit-identical
floats, which is asserted too. Both device paths (staged tile kernels and the
generic kernel) are run."""
import json
import os

import numpy as np
import pytest

import dl0gen
import oracle
from tests._full import alloc_filled_outputs, bits_equal, first_mismatch, slabs, split_events
from tests._gpu import alloc_outputs, assert_parity, bit_identical, to_dev_u16

pytestmark = pytest.mark.gpu
SHAPES = [(30, 7), (40, 7), (25, 4), (128, 8)]
GOLD = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_windows.json")


def run_family(kind, wf, ped, gain, generic=False, **kw):
    import torch
    import paper_1307_6489_b200 as rta
    E, P, S = wf.shape
    d_wf = to_dev_u16(wf)
    d_ped = torch.from_numpy(np.ascontiguousarray(ped, np.int32)).cuda()
    d_gain = torch.from_numpy(np.ascontiguousarray(gain, np.float32)).cuda()
    outs = alloc_outputs(E * P)
    rta.rta_debug_force_generic(generic)
    try:
        if kind == "fixed":
            d_ws = torch.from_numpy(np.ascontiguousarray(kw["window_start"], np.int32)).cuda()
            rta.rta_extract_fixed(d_wf, E, P, S, d_ped, d_gain, kw["W"], d_ws, *outs)
        elif kind == "local_peak":
            rta.rta_extract_local_peak(d_wf, E, P, S, d_ped, d_gain, kw["W"], kw["shift"], *outs)
        else:
            rta.rta_extract_fir(d_wf, E, P, S, d_ped, d_gain, kw["taps"], *outs)
        torch.cuda.synchronize()
    finally:
        rta.rta_debug_force_generic(False)
    return tuple(o.cpu().numpy() for o in outs)


def want_family(kind, wf, ped, gain, **kw):
    if kind == "fixed":
        return oracle.extract_fixed(wf, ped, gain, kw["W"], kw["window_start"])
    if kind == "local_peak":
        return oracle.extract_local_peak(wf, ped, gain, kw["W"], kw["shift"])
    return oracle.extract_fir(wf, ped, gain, kw["taps"])


def both(kind, wf, ped, gain, **kw):
    want = want_family(kind, wf, ped, gain, **kw)
    for generic in (False, True):
        got = run_family(kind, wf, ped, gain, generic=generic, **kw)
        assert_parity(got, want, "%s generic=%s" % (kind, generic))
        assert bit_identical(got, want), "%s generic=%s" % (kind, generic)
    return want


def test_hand_worked_window_fixtures_on_gpu():
    for c in json.load(open(GOLD))["cases"]:
        wf = np.array(c["wf"], np.uint16).reshape(1, 1, -1)
        kw = {k: c[k] for k in ("W", "shift", "taps") if k in c}
        if "window_start" in c:
            kw["window_start"] = [c["window_start"]]
        got = run_family(c["kind"], wf, [c["pedestal"]], [c["gain"]], **kw)
        assert (int(got[0][0]), int(got[1][0])) == (c["out_sum"], c["out_start"]), c["name"]
        assert got[2][0] == np.float32(c["out_charge"]), c["name"]
        assert got[3][0] == np.float32(np.float64(c["time_num"]) / np.float64(c["time_den"])), c["name"]


def _random_case(S, E, P, seed, full_range):
    rng = np.random.default_rng(seed)
    hi = 65536 if full_range else 4096
    wf = rng.integers(0, hi, size=(E, P, S)).astype(np.uint16)
    wf[rng.random((E, P)) < 0.15] = hi - 1                  # all-max traces: every window ties
    wf[rng.random((E, P)) < 0.15] //= np.uint16(2048 if not full_range else 16384)   # tie-heavy
    ped = (rng.integers(-70000, 70000, P) if full_range else rng.integers(0, 600, P)).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    return rng, wf, ped, gain


@pytest.mark.parametrize("S,W", SHAPES + [(31, 5), (64, 16), (7, 7), (9, 1), (200, 3)])
@pytest.mark.parametrize("E,P", [(1, 1), (3, 5), (2, 129), (5, 257), (4, 1031)])
@pytest.mark.parametrize("full_range", [False, True])
def test_fixed_window_random(S, W, E, P, full_range):
    rng, wf, ped, gain = _random_case(S, E, P, S * 7919 + W * 31 + E * P, full_range)
    start = rng.integers(-5, S + 5, P).astype(np.int32)
    start[:: 7] = rng.integers(-2 ** 31, 2 ** 31 - 1, len(start[:: 7]))   # far outside: clamped
    both("fixed", wf, ped, gain, W=W, window_start=start)


@pytest.mark.parametrize("S,W", SHAPES + [(31, 5), (64, 16), (7, 7), (9, 1), (200, 3)])
@pytest.mark.parametrize("E,P", [(1, 1), (3, 5), (2, 129), (5, 257), (4, 1031)])
@pytest.mark.parametrize("shift", [0, 3, -2, 1000, -2 ** 31, 2 ** 31 - 1])
def test_local_peak_random(S, W, E, P, shift):
    full = (E * P) % 2 == 0
    rng, wf, ped, gain = _random_case(S, E, P, S * 31 + W * 7 + E * P + 5, full)
    both("local_peak", wf, ped, gain, W=W, shift=shift)


@pytest.mark.parametrize("S,K", SHAPES + [(31, 5), (64, 16), (7, 7), (9, 1), (200, 3), (64, 32)])
@pytest.mark.parametrize("E,P", [(1, 1), (3, 5), (2, 129), (5, 257), (4, 1031)])
def test_fir_random(S, K, E, P):
    full = (E * P) % 2 == 0
    rng, wf, ped, gain = _random_case(S, E, P, S * 131 + K * 17 + E * P, full)
    lim = max(1, min(9, (2 ** 31 - 1) // (S * 65535 * K)))   # stay inside the int32 guard
    for taps in (rng.integers(-lim + 1 if lim > 1 else 0, lim + 1, K),
                 np.ones(K, np.int64), np.zeros(K, np.int64)):
        if S * 65535 * max(1, int(np.abs(taps).sum())) >= 2 ** 31:
            continue
        both("fir", wf, ped, gain, taps=taps.astype(np.int32))


@pytest.mark.parametrize("S,K", SHAPES)
@pytest.mark.parametrize("edge", [127, -128, 128, -129, 200])
def test_fir_tap_range_paths(S, K, edge):
    """Taps inside [-128, 127] take the packed IDP.2A path of the staged kernels,
    anything else the int32 multiply-add path; both must match the oracle at the
    boundary values (few non-zero taps keep S * sum|c| * 65535 < 2^31)."""
    full = edge > 0
    rng, wf, ped, gain = _random_case(S, 4, 300, S * 3 + K + abs(edge), full)
    taps = np.zeros(K, np.int32)
    taps[0] = edge
    taps[K - 1] = -3 if edge > 0 else 2
    if K > 2:
        taps[K // 2] = 1
    assert S * 65535 * int(np.abs(taps).sum()) < 2 ** 31
    both("fir", wf, ped, gain, taps=taps)


@pytest.mark.parametrize("S,W", SHAPES)
def test_fir_all_ones_equals_rta_extract_on_device(S, W):
    import torch
    import paper_1307_6489_b200 as rta
    rng, wf, ped, gain = _random_case(S, 6, 300, S + W, False)
    got = run_family("fir", wf, ped, gain, taps=[1] * W)
    E, P, _ = wf.shape
    outs = alloc_outputs(E * P)
    rta.rta_extract(to_dev_u16(wf), E, P, S, torch.from_numpy(ped).cuda(),
                    torch.from_numpy(gain).cuda(), W, *outs)
    torch.cuda.synchronize()
    assert bit_identical(got, tuple(o.cpu().numpy() for o in outs))


@pytest.mark.parametrize("S,W", SHAPES)
def test_family_extreme_pedestals(S, W):
    rng = np.random.default_rng(S)
    E, P = 3, 300
    wf = rng.integers(0, 65536, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(-2 ** 30, 2 ** 30, P).astype(np.int32)
    gain = rng.uniform(-3, 3, P).astype(np.float32)
    gain[0], gain[1] = np.float32("nan"), np.float32("inf")
    both("fixed", wf, ped, gain, W=W, window_start=rng.integers(0, S, P).astype(np.int32))
    both("local_peak", wf, ped, gain, W=W, shift=2)
    both("fir", wf, ped, gain, taps=rng.integers(-3, 4, W).astype(np.int32))


@pytest.mark.parametrize("name,n_ev", [("C1", 64), ("C2", 23), ("C3", 19), ("C4", 11)])
def test_family_on_config_models(name, n_ev):
    """The config signal models, several tiles per CTA plus a ragged tail."""
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 100 if name != "C1" else 0, n_ev, threads=4)
    rng = np.random.default_rng(n_ev)
    both("fixed", wf, ped, gain, W=c.W,
         window_start=rng.integers(0, c.n_samples - c.W + 1, c.n_pixels).astype(np.int32))
    both("local_peak", wf, ped, gain, W=c.W, shift=c.W // 2)
    taps = np.array([1, 2, 3, 4, 3, 2, 1, 1][:c.W], np.int32)          # triangular matched filter
    both("fir", wf, ped, gain, taps=taps)


@pytest.mark.parametrize("name", ["C2", "C4"])
def test_family_full_size_every_event(name):
    """BASELINE.json's full sizes in one launch per extractor into sentinel-filled
    outputs; EVERY event against the oracle on the same bytes (copied back in
    ~1 GB slabs, all host cores)."""
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    d_wf = torch.empty((c.n_events, c.n_pixels, c.n_samples), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(c, d_wf.data_ptr(), 0, c.n_events, torch.cuda.current_stream().cuda_stream)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    rng = np.random.default_rng(9)
    start = rng.integers(0, c.n_samples - c.W + 1, c.n_pixels).astype(np.int32)
    taps = np.array([1, 2, 3, 4, 3, 2, 1, 1][:c.W], np.int32)
    kinds = (("fixed", dict(W=c.W, window_start=start)),
             ("local_peak", dict(W=c.W, shift=2)), ("fir", dict(taps=taps)))
    results = {}
    for kind, kw in kinds:
        outs = alloc_filled_outputs(c.n_traces)
        before = rta.rta_launch_count()
        if kind == "fixed":
            rta.rta_extract_fixed(d_wf, c.n_events, c.n_pixels, c.n_samples, d_ped, d_gain, c.W,
                                  torch.from_numpy(start).cuda(), *outs)
        elif kind == "local_peak":
            rta.rta_extract_local_peak(d_wf, c.n_events, c.n_pixels, c.n_samples, d_ped, d_gain,
                                       c.W, 2, *outs)
        else:
            rta.rta_extract_fir(d_wf, c.n_events, c.n_pixels, c.n_samples, d_ped, d_gain, taps, *outs)
        torch.cuda.synchronize()
        assert rta.rta_launch_count() == before + 1
        results[kind] = outs
    # one pass over the input slabs serves the three extractors
    for e0, k in slabs(c.n_events, c.n_pixels * c.n_samples * 2):
        wf = d_wf[e0:e0 + k].cpu().numpy().view(np.uint16)
        lo, hi = e0 * c.n_pixels, (e0 + k) * c.n_pixels
        for kind, kw in kinds:
            want = split_events(k, lambda a, b: want_family(kind, wf[a:b], ped, gain, **kw))
            got = tuple(o[lo:hi].cpu().numpy() for o in results[kind])
            assert bits_equal(got, want), "%s %s events %d..%d: %s" % (
                name, kind, e0, e0 + k, first_mismatch(got, want))
