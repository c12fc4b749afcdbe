"""Pins for the window-family oracle (oracle/rta_oracle_windows.cpp; CPU only).

The paper names the family in one sentence (§5) and ref [13] is
not available, so the definitions are DESIGN.md readings R22-R24. They are
pinned to: hand-worked fixtures (tests/golden/hand_worked_windows.json), closed
forms, numpy restatements written here (slicing / argmax / np.correlate), and
reductions to the already pinned sliding-window oracle. No expected value comes
from the oracle under test or from the CUDA path.
"""
import itertools
import json
import os

import numpy as np
import pytest

import oracle
from tests._checks import np_window_outputs, np_fixed, np_local_peak, np_fir

GOLD = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_windows.json")
f32 = np.float32


def _one(kind, tr, ped, gain, **kw):
    wf = np.asarray(tr, np.uint16).reshape(1, 1, -1)
    p, g = np.array([ped], np.int32), np.array([gain], np.float32)
    if kind == "fixed":
        r = oracle.extract_fixed(wf, p, g, kw["W"], [kw["window_start"]])
    elif kind == "local_peak":
        r = oracle.extract_local_peak(wf, p, g, kw["W"], kw["shift"])
    else:
        r = oracle.extract_fir(wf, p, g, kw["taps"])
    return int(r[0][0]), int(r[1][0]), f32(r[2][0]), f32(r[3][0])


def test_hand_worked_window_fixtures():
    cases = json.load(open(GOLD))["cases"]
    assert {c["kind"] for c in cases} == {"fixed", "local_peak", "fir"}
    for c in cases:
        kw = {k: c[k] for k in ("W", "window_start", "shift", "taps") if k in c}
        s, t, q, tm = _one(c["kind"], c["wf"], c["pedestal"], c["gain"], **kw)
        assert (s, t) == (c["out_sum"], c["out_start"]), c["name"]
        assert q == f32(c["out_charge"]), c["name"]
        assert tm == f32(np.float64(c["time_num"]) / np.float64(c["time_den"])), c["name"]


# ------------------------------------------------------------------ fixed ----
@pytest.mark.parametrize("S,W", [(30, 7), (25, 4), (128, 8), (5, 5), (9, 1)])
def test_fixed_constant_trace_and_clamping(S, W):
    ped, c, gain = 400, 437, 1.0625
    for t0 in (-1000, -1, 0, 1, S - W - 1, S - W, S - W + 1, S, 10 ** 6):
        s, t, q, tm = _one("fixed", [c] * S, ped, gain, W=W, window_start=t0)
        want_t = min(max(t0, 0), S - W)
        assert t == want_t and s == W * (c - ped) and q == f32(W * (c - ped) * gain)
        assert tm == f32(want_t + (W - 1) / 2)            # equal weights -> centre


@pytest.mark.parametrize("S,W", [(12, 3), (40, 7)])
def test_fixed_delta_inside_and_outside_the_window(S, W):
    ped, A = 300, 57
    for k in range(S):
        tr = [ped] * S
        tr[k] = ped + A
        for t0 in range(S - W + 1):
            s, t, q, tm = _one("fixed", tr, ped, 0.75, W=W, window_start=t0)
            assert t == t0
            if t0 <= k < t0 + W:
                assert s == A and tm == f32(k) and q == f32(A * 0.75)
            else:
                assert s == 0 and tm == f32(t0 + (W - 1) / 2) and q == 0


def test_fixed_start_is_per_pixel_not_per_event():
    rng = np.random.default_rng(1)
    E, P, S, W = 5, 7, 20, 4
    wf = rng.integers(0, 4096, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(300, 500, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    start = rng.integers(-3, S + 3, P).astype(np.int32)
    got = oracle.extract_fixed(wf, ped, gain, W, start)
    ref = np_fixed(wf, ped, gain, W, start)
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)
    assert (got[1].reshape(E, P) == np.clip(start, 0, S - W)[None, :]).all()


@pytest.mark.parametrize("name", ["C1"])
def test_fixed_at_the_sliding_start_reproduces_the_sliding_extractor(name):
    """Reduction to the pinned oracle: one pixel per 'camera' so that the
    per-pixel start can be set trace by trace."""
    import dl0gen
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 0, 2, threads=2)                       # [2][P][S]
    ref = oracle.extract(wf, ped, gain, c.W)
    flat = wf.reshape(1, -1, c.n_samples)                            # 1 event, 2P pixels
    got = oracle.extract_fixed(flat, np.tile(ped, 2), np.tile(gain, 2), c.W, ref[1])
    for a, b in zip(got, ref):
        assert np.array_equal(a.view(np.int32), b.view(np.int32))


# ------------------------------------------------------------- local peak ----
@pytest.mark.parametrize("S,W,shift", [(30, 7, 3), (25, 4, 1), (16, 5, 0), (16, 5, -2), (9, 1, 0)])
def test_local_peak_delta_every_position(S, W, shift):
    ped, A = 300, 57
    for k in range(S):
        tr = [ped] * S
        tr[k] = ped + A
        s, t, q, tm = _one("local_peak", tr, ped, 1.0, W=W, shift=shift)
        want_t = min(max(k - shift, 0), S - W)
        assert t == want_t
        if want_t <= k < want_t + W:
            assert s == A and tm == f32(k)
        else:                                             # shift moved the window off the pulse
            assert s == 0 and tm == f32(want_t + (W - 1) / 2)


def test_local_peak_ties_take_the_earliest_maximum():
    tr = [10, 50, 20, 50, 50, 10, 10, 10]
    s, t, q, tm = _one("local_peak", tr, 10, 1.0, W=2, shift=0)
    assert (s, t) == (40 + 10, 1)
    tr[3] = 51
    s, t, q, tm = _one("local_peak", tr, 10, 1.0, W=2, shift=0)
    assert (s, t) == (41 + 40, 3)


def test_local_peak_W1_shift0_is_the_sliding_extractor_with_W1():
    rng = np.random.default_rng(6)
    wf = rng.integers(0, 50, size=(7, 11, 19)).astype(np.uint16)     # many ties
    ped = rng.integers(0, 20, 11).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, 11).astype(np.float32)
    a = oracle.extract_local_peak(wf, ped, gain, 1, 0)
    b = oracle.extract(wf, ped, gain, 1)
    for u, v in zip(a, b):
        assert np.array_equal(u.view(np.int32), v.view(np.int32))


@pytest.mark.parametrize("E,P,S,W,shift,hi", [
    (9, 13, 30, 7, 3, 4096), (5, 8, 40, 7, 2, 4096), (6, 10, 25, 4, 1, 4096),
    (3, 5, 128, 8, 3, 4096), (4, 6, 31, 5, -4, 65536), (4, 9, 17, 6, 20, 6)])
def test_local_peak_numpy_restatement(E, P, S, W, shift, hi):
    rng = np.random.default_rng(S * 31 + W)
    wf = rng.integers(0, hi, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(0, max(2, hi // 8), P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    got = oracle.extract_local_peak(wf, ped, gain, W, shift)
    ref = np_local_peak(wf, ped, gain, W, shift)
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)


def test_local_peak_pedestal_invariance():
    rng = np.random.default_rng(13)
    wf = rng.integers(300, 3000, size=(4, 17, 30)).astype(np.uint16)
    ped = rng.integers(280, 420, 17).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, 17).astype(np.float32)
    a = oracle.extract_local_peak(wf, ped, gain, 7, 3)
    b = oracle.extract_local_peak(wf + np.uint16(1000), ped + 1000, gain, 7, 3)
    for u, v in zip(a, b):
        assert np.array_equal(u, v)


# -------------------------------------------------------------------- FIR ----
@pytest.mark.parametrize("E,P,S,W", [(9, 13, 30, 7), (5, 8, 40, 7), (6, 10, 25, 4), (3, 5, 128, 8),
                                      (4, 6, 9, 9), (4, 6, 9, 1)])
def test_fir_all_ones_is_the_sliding_extractor(E, P, S, W):
    rng = np.random.default_rng(S + W)
    wf = rng.integers(0, 4096, size=(E, P, S)).astype(np.uint16)
    wf[0] = rng.integers(0, 3, size=(P, S))                          # tie-heavy event
    ped = rng.integers(0, 2000, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    a = oracle.extract_fir(wf, ped, gain, np.ones(W, np.int32))
    b = oracle.extract(wf, ped, gain, W)
    for u, v in zip(a, b):
        assert np.array_equal(u.view(np.int32), v.view(np.int32))


def test_fir_scaling_the_taps_scales_the_sum_only():
    rng = np.random.default_rng(3)
    wf = rng.integers(0, 4096, size=(6, 9, 30)).astype(np.uint16)
    ped = rng.integers(300, 2500, 9).astype(np.int32)
    gain = np.ones(9, np.float32)
    taps = np.array([1, 3, 5, 3, 1], np.int32)
    a = oracle.extract_fir(wf, ped, gain, taps)
    b = oracle.extract_fir(wf, ped, gain, 3 * taps)
    assert np.array_equal(3 * a[0], b[0]) and np.array_equal(a[1], b[1])
    assert np.array_equal(a[3], b[3])                     # (3 num)/(3 sum) is the same real number
    assert np.array_equal(b[2], (3 * a[0]).astype(np.float32))


def test_fir_single_shifted_tap_finds_the_peak_sample():
    """taps [0,0,1]: y(t) = x[t+2], so t* = (first argmax of x[2:]) and the time
    is exactly the index of that sample."""
    rng = np.random.default_rng(4)
    S = 20
    wf = rng.integers(500, 4000, size=(5, 6, S)).astype(np.uint16)
    ped = np.full(6, 400, np.int32)                       # x > 0 everywhere
    s, t, q, tm = oracle.extract_fir(wf, ped, np.ones(6, np.float32), [0, 0, 1])
    x = wf.astype(np.int64).reshape(-1, S) - 400
    pk = x[:, 2:].argmax(-1)
    assert np.array_equal(t, pk) and np.array_equal(s, x[np.arange(len(x)), pk + 2])
    assert np.array_equal(tm, (pk + 2).astype(np.float32))


def test_fir_difference_filter_on_a_ramp():
    a, ped, S = 3, 50, 12
    s, t, q, tm = _one("fir", [ped + a * i for i in range(S)], ped, 1.0, taps=[-1, 1])
    assert (s, t) == (a, 0)                               # y(t) = a for every t -> earliest
    assert tm == f32(1.0)                                 # num = 0*(-1)*0 + 1*1*a, den = a


def test_fir_negated_unit_tap_picks_the_earliest_minimum():
    tr = [9, 4, 7, 4, 8]
    s, t, q, tm = _one("fir", tr, 5, 1.0, taps=[-1])
    assert (s, t) == (1, 1) and tm == f32(1)              # y = -(4-5) = 1 > 0: num/den = 1*(-1)*(-1)/1
    s, t, q, tm = _one("fir", tr, 2, 1.0, taps=[-1])
    assert (s, t) == (-2, 1) and tm == f32(1)             # y <= 0 -> centre of a width-1 support


@pytest.mark.parametrize("taps", [[1, -2, 1], [2, 1], [1, 2, 3, 2, 1], [-1, 0, 1], [5]])
def test_fir_exhaustive_small_alphabet_against_numpy(taps):
    S = 6
    tr = np.array(list(itertools.product([9, 10, 11], repeat=S)), np.uint16)   # 729 traces
    wf = tr.reshape(243, 3, S)
    ped = np.array([10, 9, 12], np.int32)
    gain = np.array([1.0, 0.5, 1.0625], np.float32)
    got = oracle.extract_fir(wf, ped, gain, taps)
    ref = np_fir(wf, ped, gain, taps)
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("E,P,S,K,hi", [(9, 13, 30, 7, 4096), (5, 8, 40, 7, 4096), (6, 10, 25, 4, 4096),
                                         (3, 5, 128, 8, 4096), (4, 6, 31, 16, 65536)])
def test_fir_numpy_restatement_random(E, P, S, K, hi):
    rng = np.random.default_rng(S * 17 + K)
    wf = rng.integers(0, hi, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(0, max(2, hi // 8), P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    taps = rng.integers(-4, 9, K).astype(np.int32)
    got = oracle.extract_fir(wf, ped, gain, taps)
    ref = np_fir(wf, ped, gain, taps)
    for a, b in zip(got, ref):
        assert np.array_equal(a, b)


def test_window_family_error_paths_and_empty():
    wf = np.zeros((2, 3, 5), np.uint16)
    ped, g = np.zeros(3, np.int32), np.ones(3, np.float32)
    with pytest.raises(ValueError):
        oracle.extract_fixed(wf, ped, g, 6, [0, 0, 0])
    with pytest.raises(ValueError):
        oracle.extract_local_peak(wf, ped, g, 0, 0)
    with pytest.raises(ValueError):
        oracle.extract_fir(wf, ped, g, np.ones(6, np.int32))
    with pytest.raises(ValueError):
        oracle.extract_fixed(wf, ped, g, 2, [0, 0])                  # start must be [n_pixels]
    empty = np.zeros((0, 3, 5), np.uint16)
    assert all(len(o) == 0 for o in oracle.extract_fir(empty, ped, g, [1, 1]))
