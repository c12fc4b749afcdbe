"""Independent checkers used by the pins and by the GPU parity tests.

Nothing here calls ``oracle/`` or the CUDA path: these are separate numpy
restatements of what BASELINE.json:north_star sentence 2 defines, written so a
mistake in either implementation shows up against them.
"""
from __future__ import annotations

import numpy as np
from numpy.lib.stride_tricks import sliding_window_view


def np_extract(wf, pedestal, gain, W):
    """numpy restatement (pin P11): sliding_window_view + argmax, whose
    first-maximum rule is exactly "earliest on ties". int64 / float64 inside."""
    wf = np.asarray(wf)
    E, P, S = wf.shape
    x = wf.astype(np.int64) - np.asarray(pedestal, np.int64)[None, :, None]
    win = sliding_window_view(x, W, axis=2)              # [E][P][S-W+1][W]
    sums = win.sum(-1)
    start = sums.argmax(-1)                               # first maximum
    best = np.take_along_axis(sums, start[..., None], -1)[..., 0]
    idx = start[..., None] + np.arange(W)[None, None, :]
    xs = np.take_along_axis(x, idx, -1)
    num = (idx * xs).sum(-1)
    g = np.asarray(gain, np.float32).astype(np.float64)[None, :]
    charge = (best.astype(np.float64) * g).astype(np.float32)
    with np.errstate(divide="ignore", invalid="ignore"):
        t_pos = num.astype(np.float64) / best.astype(np.float64)
    t_deg = start.astype(np.float64) + 0.5 * (W - 1)
    time = np.where(best > 0, t_pos, t_deg).astype(np.float32)
    return (best.astype(np.int32).ravel(), start.astype(np.int32).ravel(),
            charge.ravel(), time.ravel())


def prefix_extract_ints(wf, pedestal, W):
    """Second independent integer implementation (pin P10): prefix sums,
    scanning windows from the LAST to the first with '>=' so that the earliest
    maximum survives — a different tie mechanism from the oracle's strict '>'."""
    wf = np.asarray(wf)
    E, P, S = wf.shape
    x = wf.astype(np.int64) - np.asarray(pedestal, np.int64)[None, :, None]
    c = np.concatenate([np.zeros((E, P, 1), np.int64), np.cumsum(x, -1)], -1)
    nwin = S - W + 1
    best = c[..., nwin - 1 + W] - c[..., nwin - 1]
    start = np.full((E, P), nwin - 1, np.int64)
    for t in range(nwin - 2, -1, -1):
        s = c[..., t + W] - c[..., t]
        take = s >= best
        best = np.where(take, s, best)
        start = np.where(take, t, start)
    return best.astype(np.int32).ravel(), start.astype(np.int32).ravel()


def check_invariants(wf, pedestal, gain, W, out_sum, out_start, out_charge,
                     out_time, time_atol=1e-4, charge_rtol=1e-6):
    """Pins P8 + P9 (+ float consistency): properties that fully characterise
    the integer outputs and hold at any size. Raises AssertionError."""
    wf = np.asarray(wf)
    E, P, S = wf.shape
    n = E * P
    x = (wf.astype(np.int64) - np.asarray(pedestal, np.int64)[None, :, None]).reshape(n, S)
    out_sum = np.asarray(out_sum).astype(np.int64)
    out_start = np.asarray(out_start).astype(np.int64)
    assert out_sum.shape == (n,) and out_start.shape == (n,)
    assert (out_start >= 0).all() and (out_start <= S - W).all(), "start outside [0, S-W]"
    c = np.concatenate([np.zeros((n, 1), np.int64), np.cumsum(x, -1)], -1)
    rows = np.arange(n)
    # P8: out_sum is the sum of the selected W pedestal-subtracted samples
    sel = c[rows, out_start + W] - c[rows, out_start]
    assert (sel == out_sum).all(), "P8: out_sum != sum of selected window"
    # P9: maximal, and strictly greater than every earlier window
    allsums = c[:, W:] - c[:, :S - W + 1]
    assert (allsums <= out_sum[:, None]).all(), "P9: a window beats out_sum"
    earlier = np.arange(S - W + 1)[None, :] < out_start[:, None]
    assert (~earlier | (allsums < out_sum[:, None])).all(), "P9: an earlier window ties"
    # charge: one rounding of the exact product (R10)
    g = np.tile(np.asarray(gain, np.float32).astype(np.float64), E)
    want_q = (out_sum.astype(np.float64) * g).astype(np.float32)
    q = np.asarray(out_charge, np.float32)
    ok = np.isclose(q, want_q, rtol=charge_rtol, atol=0.0) | (q == want_q)
    assert ok.all(), "charge outside rel 1e-6"
    # time: weighted mean over the selected window, or the centre (R7)
    idx = out_start[:, None] + np.arange(W)[None, :]
    xs = np.take_along_axis(x, idx, 1)
    num = (idx * xs).sum(1)
    with np.errstate(divide="ignore", invalid="ignore"):
        t_pos = num / out_sum.astype(np.float64)
    want_t = np.where(out_sum > 0, t_pos, out_start + 0.5 * (W - 1))
    tt = np.asarray(out_time, np.float32).astype(np.float64)
    err = np.abs(tt - want_t)
    # R12: beyond |t| = 1024 FP32 spacing exceeds 1e-4 — compare to RN32 there
    big = np.abs(want_t) > 1024.0
    assert (err[~big] <= time_atol).all(), "time outside abs 1e-4"
    if big.any():
        assert (np.asarray(out_time, np.float32)[big]
                == want_t[big].astype(np.float32)).all(), "time != RN32(exact)"


# ---- window family (oracle/rta_oracle_windows.cpp): numpy restatements -------
def np_window_outputs(x, start, gain_per_trace, weights):
    """Outputs of every trace given its window start: x int64 [n][S], start
    int64 [n], weights int64 [W] (ones for a plain window)."""
    n, S = x.shape
    W = len(weights)
    idx = start[:, None] + np.arange(W)[None, :]
    xs = np.take_along_axis(x, idx, 1) * weights[None, :]
    s = xs.sum(1)
    num = (idx * xs).sum(1)
    charge = (s.astype(np.float64) * gain_per_trace).astype(np.float32)
    with np.errstate(divide="ignore", invalid="ignore"):
        t_pos = num.astype(np.float64) / s.astype(np.float64)
    time = np.where(s > 0, t_pos, start + 0.5 * (W - 1)).astype(np.float32)
    return s.astype(np.int32), start.astype(np.int32), charge, time


def _flat(wf, pedestal, gain):
    wf = np.asarray(wf)
    E, P, S = wf.shape
    x = (wf.astype(np.int64) - np.asarray(pedestal, np.int64)[None, :, None]).reshape(E * P, S)
    g = np.tile(np.asarray(gain, np.float32).astype(np.float64), E)
    return E, P, S, x, g


def np_fixed(wf, pedestal, gain, W, window_start):
    E, P, S, x, g = _flat(wf, pedestal, gain)
    start = np.tile(np.clip(np.asarray(window_start, np.int64), 0, S - W), E)
    return np_window_outputs(x, start, g, np.ones(W, np.int64))


def np_local_peak(wf, pedestal, gain, W, shift):
    E, P, S, x, g = _flat(wf, pedestal, gain)
    start = np.clip(x.argmax(1) - int(shift), 0, S - W)               # argmax: first maximum
    return np_window_outputs(x, start, g, np.ones(W, np.int64))


def np_fir(wf, pedestal, gain, taps):
    E, P, S, x, g = _flat(wf, pedestal, gain)
    c = np.asarray(taps, np.int64)
    y = np.stack([np.correlate(row, c, mode="valid") for row in x])   # y[t] = sum_k c[k] x[t+k]
    return np_window_outputs(x, y.argmax(1), g, c)
