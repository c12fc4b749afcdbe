"""Pins for the oracle (CPU only): what the definition and the mathematics fix.

The paper prints no algorithm and no numbers for this step (§5),
so the oracle is pinned to BASELINE.json:north_star's own checks — the constant
trace and single-sample delta closed forms, brute force over all windows on
tiny inputs, the invariant out_sum = sum of the selected samples — expanded to
SURVEY.md §8(c) pins P1..P16. Expected values below are closed forms typed
from the mathematics, never produced by the oracle or by the CUDA path.
"""
import itertools
import json
import os

import numpy as np
import pytest

import oracle
from tests._checks import check_invariants, np_extract, prefix_extract_ints

GOLD = os.path.join(os.path.dirname(__file__), "golden", "hand_worked.json")


def run1(trace, ped, gain, W):
    """One trace -> python scalars (sum, start, charge, time)."""
    wf = np.asarray(trace, np.uint16).reshape(1, 1, -1)
    s, t, q, tm = oracle.extract(wf, np.array([ped], np.int32),
                                 np.array([gain], np.float32), W)
    return int(s[0]), int(t[0]), np.float32(q[0]), np.float32(tm[0])


def f32(x):
    return np.float32(x)


# ---------------------------------------------------------------- golden ----
def test_hand_worked_fixtures():
    cases = json.load(open(GOLD))["cases"]
    assert len(cases) >= 8
    for c in cases:
        E, P, S = c["n_events"], c["n_pixels"], c["n_samples"]
        wf = np.array(c["wf"], np.uint16).reshape(E, P, S)
        s, t, q, tm = oracle.extract(wf, np.array(c["pedestal"], np.int32),
                                     np.array(c["gain"], np.float32), c["W"])
        assert s.tolist() == c["out_sum"], c["name"]
        assert t.tolist() == c["out_start"], c["name"]
        assert q.tolist() == [float(f32(v)) for v in c["out_charge"]], c["name"]
        want = [f32(np.float64(n) / np.float64(d))
                for n, d in zip(c["time_num"], c["time_den"])]
        assert tm.tolist() == [float(v) for v in want], c["name"]


# ---------------------------------------------------------- closed forms ----
@pytest.mark.parametrize("S,W", [(30, 7), (40, 7), (25, 4), (128, 8), (5, 5), (9, 1)])
@pytest.mark.parametrize("c,ped", [(500, 400), (400, 400), (390, 400), (4095, 0), (0, 7)])
def test_P1_constant_trace(S, W, c, ped):
    gain = 1.0625  # exactly representable, so the product below is exact
    s, t, q, tm = run1([c] * S, ped, gain, W)
    assert t == 0                                   # every window ties -> earliest
    assert s == W * (c - ped)
    assert q == f32(W * (c - ped) * gain)
    assert tm == f32((W - 1) / 2)                   # equal weights, or R7 centre


@pytest.mark.parametrize("S,W", [(30, 7), (25, 4), (12, 12), (10, 1), (128, 8)])
def test_P2_positive_delta_every_position(S, W):
    ped, A, gain = 300, 57, 0.75
    for k in range(S):
        tr = [ped] * S
        tr[k] = ped + A
        s, t, q, tm = run1(tr, ped, gain, W)
        assert s == A
        assert t == max(0, k - W + 1)               # earliest window containing k
        assert tm == f32(k)                         # peak time == its index (R9)
        assert q == f32(A * gain)


@pytest.mark.parametrize("S,W", [(10, 3), (9, 4), (6, 6), (7, 1)])
def test_P3_negative_delta(S, W):
    ped, A = 100, -40
    for k in range(S):
        tr = [ped] * S
        tr[k] = ped + A
        s, t, q, tm = run1(tr, ped, 1.0, W)
        free = [u for u in range(S - W + 1) if not (u <= k <= u + W - 1)]
        if free:                                    # some window avoids the dip
            assert s == 0 and t == free[0]
        else:                                       # every window contains it
            assert s == A and t == 0
        assert tm == f32(t + (W - 1) / 2)           # R7, both branches (sum <= 0)


def test_P4_two_equal_deltas_first_wins():
    S, W, ped, A = 40, 7, 400, 90
    tr = [ped] * S
    tr[10] = ped + A
    tr[10 + W + 3] = ped + A
    s, t, q, tm = run1(tr, ped, 1.0, W)
    assert (s, t) == (A, 10 - W + 1) and tm == f32(10)
    tr[10 + W + 3] = ped + A + 1                    # now the later one is larger
    s, t, q, tm = run1(tr, ped, 1.0, W)
    assert (s, t) == (A + 1, 10 + 3 + 1) and tm == f32(10 + W + 3)


@pytest.mark.parametrize("S,W,a", [(30, 7, 3), (25, 4, 1), (16, 5, 11)])
def test_P5_ramps(S, W, a):
    ped = 50
    up = [ped + a * s for s in range(S)]
    s, t, q, tm = run1(up, ped, 1.0, W)
    t0 = S - W
    assert t == t0 and s == a * (W * t0 + W * (W - 1) // 2)
    idx = np.arange(t0, t0 + W, dtype=np.float64)
    assert tm == f32((idx * idx).sum() / idx.sum())
    ped2 = 4000
    down = [ped2 - a * s for s in range(S)]         # x = -a*s: maximum at t=0
    s, t, q, tm = run1(down, ped2, 1.0, W)
    assert t == 0 and s == -a * (W * (W - 1) // 2)
    assert tm == f32((W - 1) / 2)                   # sum <= 0 -> centre (W>1), R7


def test_P6_W1_is_first_argmax():
    rng = np.random.default_rng(6)
    wf = rng.integers(0, 50, size=(7, 11, 19)).astype(np.uint16)  # many ties
    ped = rng.integers(0, 20, 11).astype(np.int32)
    s, t, q, tm = oracle.extract(wf, ped, np.ones(11, np.float32), 1)
    x = wf.astype(np.int64) - ped[None, :, None]
    assert (t.reshape(7, 11) == x.argmax(-1)).all()
    assert (s.reshape(7, 11) == x.max(-1)).all()
    pos = s > 0
    assert (tm[pos] == t[pos].astype(np.float32)).all()
    assert (tm[~pos] == t[~pos].astype(np.float32)).all()  # centre of width 1 == start


def test_P7_W_equals_S_global_mean():
    rng = np.random.default_rng(7)
    wf = rng.integers(100, 4096, size=(3, 5, 17)).astype(np.uint16)
    ped = np.full(5, 100, np.int32)
    s, t, q, tm = oracle.extract(wf, ped, np.ones(5, np.float32), 17)
    x = wf.astype(np.float64) - 100.0
    assert (t == 0).all()
    assert (s == x.sum(-1).ravel()).all()
    want = (x * np.arange(17)).sum(-1) / x.sum(-1)
    assert (tm == want.astype(np.float32).ravel()).all()


# ---------------------------------------------- brute force on tiny inputs ----
def _all_traces(values, S):
    return np.array(list(itertools.product(values, repeat=S)), np.uint16)


@pytest.mark.parametrize("S,Ws,values,ped", [
    (4, [2], [9, 10, 11], 10),                      # 3^4 traces around the pedestal
    (5, [1, 2, 3, 4, 5], [0, 1, 2, 3], 1),          # 4^5 traces, every W
    (12, [3], [0, 1], 0),                           # 2^12 binary traces
])
def test_P10_exhaustive(S, Ws, values, ped):
    tr = _all_traces(values, S)
    n = len(tr)
    P = 4 if n % 4 == 0 else 3 if n % 3 == 0 else 1 # also exercises e*P+p indexing
    wf = tr.reshape(n // P, P, S)
    pedv = np.full(P, ped, np.int32)
    gain = np.linspace(0.9, 1.1, P).astype(np.float32)
    for W in Ws:
        got = oracle.extract(wf, pedv, gain, W)
        ref = np_extract(wf, pedv, gain, W)
        pre = prefix_extract_ints(wf, pedv, W)
        assert (got[0] == ref[0]).all() and (got[1] == ref[1]).all()
        assert (got[0] == pre[0]).all() and (got[1] == pre[1]).all()
        assert (got[2] == ref[2]).all()
        assert (got[3] == ref[3]).all()
        check_invariants(wf, pedv, gain, W, *got)


# --------------------------------------------- library restatement, random ----
@pytest.mark.parametrize("E,P,S,W,hi", [
    (16, 37, 30, 7, 4096), (9, 50, 40, 7, 4096), (11, 33, 25, 4, 4096),
    (5, 21, 128, 8, 4096), (6, 13, 31, 5, 65536), (4, 9, 64, 16, 8),
])
def test_P11_numpy_restatement_random(E, P, S, W, hi):
    rng = np.random.default_rng(E * 1000 + S)
    wf = rng.integers(0, hi, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(0, max(2, hi // 8), P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    got = oracle.extract(wf, ped, gain, W)
    ref = np_extract(wf, ped, gain, W)
    for a, b in zip(got, ref):
        assert (a == b).all()
    check_invariants(wf, ped, gain, W, *got)


# ------------------------------------------------------------- invariants ----
def test_P12_shift_equivariance():
    S, W, ped = 40, 7, 400
    rng = np.random.default_rng(12)
    core = (ped + rng.integers(1, 200, 9)).tolist()   # strictly above pedestal
    base = None
    for d in range(0, S - len(core) - 2 * W):
        tr = [ped] * S
        lo = W + d                                    # keep away from both edges
        tr[lo:lo + len(core)] = core
        s, t, q, tm = run1(tr, ped, 1.0, W)
        if base is None:
            base = (s, t, float(tm))
        assert s == base[0] and t == base[1] + d
        assert abs(float(tm) - (base[2] + d)) < 1e-5


def test_P13_pedestal_invariance():
    rng = np.random.default_rng(13)
    wf = rng.integers(300, 3000, size=(4, 17, 30)).astype(np.uint16)
    ped = rng.integers(280, 420, 17).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, 17).astype(np.float32)
    a = oracle.extract(wf, ped, gain, 7)
    b = oracle.extract(wf + np.uint16(1000), ped + 1000, gain, 7)
    for u, v in zip(a, b):
        assert (u == v).all()


def test_P14_gain():
    rng = np.random.default_rng(14)
    wf = rng.integers(0, 4096, size=(3, 8, 25)).astype(np.uint16)
    ped = rng.integers(200, 2500, 8).astype(np.int32)   # sums of both signs
    one = oracle.extract(wf, ped, np.ones(8, np.float32), 4)
    assert (one[2] == one[0].astype(np.float32)).all()   # gain 1 -> bit-exact cast
    zero = oracle.extract(wf, ped, np.zeros(8, np.float32), 4)
    assert (zero[2] == 0).all()
    two = oracle.extract(wf, ped, np.full(8, 2.0, np.float32), 4)
    assert (two[2] == 2 * one[2]).all()                  # exact doubling
    for k in (0, 1, 3):                                  # gain never touches the rest
        assert (one[k] == two[k]).all() and (one[k] == zero[k]).all()
    half = oracle.extract(wf, ped, np.linspace(0.9, 1.1, 8).astype(np.float32), 4)
    g64 = np.tile(np.linspace(0.9, 1.1, 8).astype(np.float32).astype(np.float64), 3)
    assert (half[2] == (one[0] * g64).astype(np.float32)).all()


def test_P15_time_inside_window_when_weights_nonnegative():
    rng = np.random.default_rng(15)
    wf = rng.integers(400, 4096, size=(5, 40, 40)).astype(np.uint16)
    ped = np.full(40, 400, np.int32)                     # x >= 0 everywhere
    s, t, q, tm = oracle.extract(wf, ped, np.ones(40, np.float32), 7)
    pos = s > 0
    assert pos.any()
    assert (tm[pos] >= t[pos]).all() and (tm[pos] <= t[pos] + 6).all()


def test_P16_saturation_plateau():
    S, W, ped = 30, 7, 400
    tr = [ped + 3] * S
    for k in range(9, 9 + W + 3):                        # W+3 clamped samples
        tr[k] = 4095
    s, t, q, tm = run1(tr, ped, 1.0, W)
    assert t == 9 and s == W * (4095 - ped)              # first of 4 tied windows
    assert tm == f32(9 + (W - 1) / 2)


def test_negative_x_and_uint16_extremes():
    # R13: any uint16 value; R2: pedestal above the samples
    s, t, q, tm = run1([65535] * 4 + [0] * 4, 70000, 1.0, 4)
    assert (s, t) == (4 * (65535 - 70000), 0) and tm == f32(1.5)
    s, t, q, tm = run1([0, 65535, 65535, 0], 0, 1.0, 2)
    assert (s, t) == (131070, 1) and tm == f32(1.5)


def test_P17_error_paths_and_empty():
    wf = np.zeros((2, 3, 5), np.uint16)
    ped = np.zeros(3, np.int32)
    g = np.ones(3, np.float32)
    with pytest.raises(ValueError):
        oracle.extract(wf, ped, g, 6)                    # W > S
    with pytest.raises(ValueError):
        oracle.extract(wf, ped, g, 0)                    # W < 1
    out = oracle.extract(np.zeros((0, 3, 5), np.uint16), ped, g, 2)
    assert all(len(o) == 0 for o in out)                 # R17


def test_threads_variant_is_the_same_function():
    rng = np.random.default_rng(99)
    wf = rng.integers(0, 4096, size=(13, 7, 30)).astype(np.uint16)
    ped = rng.integers(380, 421, 7).astype(np.int32)
    g = rng.uniform(0.9, 1.1, 7).astype(np.float32)
    a = oracle.extract(wf, ped, g, 7)
    b = oracle.extract_threads(wf, ped, g, 7, 4)
    for u, v in zip(a, b):
        assert (u == v).all()
