"""Pins for the mixed-camera (ragged) oracle (oracle/rta_oracle_ragged.cpp; CPU
only). The paper has three telescope sizes, sub-arrays
 and an event builder that merges telescopes but no
layout; the layout is DESIGN.md readings R28-R30. Pinned to: a hand-assembled
batch of hand-worked traces (tests/golden/ragged.json), an independent numpy
restatement applied block by block, closed forms per block, invariance under
block order / gaps / output placement, reduction of a uniform batch to the
(pinned) uniform oracle, and mutation checks. No expected value comes from the
CUDA path."""
import json
import os

import numpy as np
import pytest

import oracle
from tests._checks import np_extract
from tests._ragged import make_batch

GOLD = os.path.join(os.path.dirname(__file__), "golden", "ragged.json")


def run(b, **kw):
    return oracle.extract_ragged(b.wf, *b.tables(), b.pedestal, b.gain, b.n_out, **kw)


def np_ragged(b):
    """numpy restatement: slice every block out and apply tests/_checks.np_extract."""
    outs = (np.full(b.n_out, -1, np.int32), np.full(b.n_out, -1, np.int32),
            np.full(b.n_out, np.nan, np.float32), np.full(b.n_out, np.nan, np.float32))
    for k, w0, o0 in zip(b.blk_tel, b.blk_wf_offset, b.blk_out_offset):
        P, S, W, c = b.tel_n_pixels[k], b.tel_n_samples[k], b.tel_W[k], b.tel_calib_offset[k]
        blk = b.wf[w0:w0 + P * S].reshape(1, P, S)
        r = np_extract(blk, b.pedestal[c:c + P], b.gain[c:c + P], W)
        for o, v in zip(outs, r):
            o[o0:o0 + P] = v
    return outs


def same(a, b):
    return all(np.array_equal(x.view(np.int32), y.view(np.int32)) for x, y in zip(a, b))


def test_hand_assembled_fixture():
    g = json.load(open(GOLD))
    s, t, q, tm = oracle.extract_ragged(
        g["wf"], g["tel_n_pixels"], g["tel_n_samples"], g["tel_W"], g["tel_calib_offset"],
        g["blk_tel"], g["blk_wf_offset"], g["blk_out_offset"], g["pedestal"], g["gain"], g["n_out"])
    n = len(g["out_sum"])
    assert s[:n].tolist() == g["out_sum"] and t[:n].tolist() == g["out_start"]
    assert q[:n].tolist() == g["out_charge"]
    want_t = [float(np.float32(np.float64(a) / np.float64(b))) for a, b in zip(g["time_num"], g["time_den"])]
    assert tm[:n].tolist() == want_t
    assert s[n] == -1 and t[n] == -1 and np.isnan(q[n]) and np.isnan(tm[n])   # never written


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_numpy_restatement_block_by_block(seed):
    b = make_batch([((5, 9, 3), 2), ((3, 4, 4), 1), ((17, 30, 7), 2), ((8, 25, 4), 1), ((2, 128, 8), 1)],
                   n_events=9, seed=seed, gap=5, shuffle_out=True)
    assert same(run(b), np_ragged(b))


def test_config_cameras_numpy_restatement():
    b = make_batch([("C1", 1), ("C3", 1)], n_events=2, seed=3, trigger=1.0)
    assert same(run(b), np_ragged(b))


def test_closed_forms_per_block():
    """Constant blocks: every trace gives start 0, sum W(c-ped), time (W-1)/2 — with each
    block's own W and calibration; a delta at sample k gives time k exactly."""
    b = make_batch([((4, 12, 5), 1), ((3, 7, 2), 1), ((6, 40, 7), 1)], n_events=3, seed=5, trigger=1.0)
    wf = b.wf.copy()
    consts = {}
    for i, (k, w0) in enumerate(zip(b.blk_tel, b.blk_wf_offset)):
        P, S = b.tel_n_pixels[k], b.tel_n_samples[k]
        consts[i] = 700 + 10 * i
        wf[w0:w0 + P * S] = consts[i]
    s, t, q, tm = oracle.extract_ragged(wf, *b.tables(), b.pedestal, b.gain, b.n_out)
    for i, (k, o0) in enumerate(zip(b.blk_tel, b.blk_out_offset)):
        P, W, c = b.tel_n_pixels[k], b.tel_W[k], b.tel_calib_offset[k]
        ped, gain = b.pedestal[c:c + P].astype(np.int64), b.gain[c:c + P]
        assert (t[o0:o0 + P] == 0).all()
        assert (s[o0:o0 + P] == W * (consts[i] - ped)).all()
        assert (tm[o0:o0 + P] == np.float32((W - 1) / 2)).all()
        assert (q[o0:o0 + P] == (W * (consts[i] - ped) * gain.astype(np.float64)).astype(np.float32)).all()
    # delta: pedestal everywhere, +A at sample kpos of every trace of block 1
    k = b.blk_tel[1]
    P, S, W, c = b.tel_n_pixels[k], b.tel_n_samples[k], b.tel_W[k], b.tel_calib_offset[k]
    for kpos in range(S):
        blk = np.repeat(b.pedestal[c:c + P].astype(np.uint16)[:, None], S, 1)
        blk[:, kpos] += 9
        w0 = b.blk_wf_offset[1]
        wf[w0:w0 + P * S] = blk.ravel()
        s, t, q, tm = oracle.extract_ragged(wf, *b.tables(), b.pedestal, b.gain, b.n_out)
        o0 = b.blk_out_offset[1]
        assert (s[o0:o0 + P] == 9).all() and (t[o0:o0 + P] == max(0, kpos - W + 1)).all()
        assert (tm[o0:o0 + P] == np.float32(kpos)).all()


def test_block_order_gaps_and_output_placement_do_not_matter():
    tels = [((5, 9, 3), 2), ((17, 30, 7), 1), ((8, 25, 4), 2)]
    a = make_batch(tels, n_events=6, seed=11)
    ra = run(a)
    # the same blocks listed in reverse order: identical outputs
    b = make_batch(tels, n_events=6, seed=11)
    b.blk_tel, b.blk_wf_offset, b.blk_out_offset = b.blk_tel[::-1], b.blk_wf_offset[::-1], b.blk_out_offset[::-1]
    assert same(run(b), ra)
    # the same blocks moved apart in the waveform buffer (junk in between)
    c = make_batch(tels, n_events=6, seed=11)
    wf, offs, pos = [], [], 0
    rng = np.random.default_rng(1)
    for k, w0 in zip(c.blk_tel, c.blk_wf_offset):
        n = c.tel_n_pixels[k] * c.tel_n_samples[k]
        junk = rng.integers(0, 65536, int(rng.integers(0, 9))).astype(np.uint16)
        wf += [junk, c.wf[w0:w0 + n]]
        offs.append(pos + junk.size)
        pos += junk.size + n
    c.wf, c.blk_wf_offset = np.concatenate(wf), offs
    assert same(run(c), ra)
    # outputs scattered: each block's results land at its own offset
    d = make_batch(tels, n_events=6, seed=11, shuffle_out=True)
    rd = run(d)
    for k, oa, od in zip(a.blk_tel, a.blk_out_offset, d.blk_out_offset):
        P = a.tel_n_pixels[k]
        for x, y in zip(ra, rd):
            assert np.array_equal(x[oa:oa + P].view(np.int32), y[od:od + P].view(np.int32))


def test_uniform_batch_reduces_to_the_uniform_oracle():
    rng = np.random.default_rng(4)
    E, P, S, W = 7, 13, 30, 7
    wf = rng.integers(0, 4096, (E, P, S)).astype(np.uint16)
    ped = rng.integers(300, 500, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    want = oracle.extract(wf, ped, gain, W)
    got = oracle.extract_ragged(wf, [P], [S], [W], [0], [0] * E, [e * P * S for e in range(E)],
                                [e * P for e in range(E)], ped, gain, E * P)
    assert same(got, want)


def test_mutations_fail_the_fixture():
    """A plausible wrong reading of the tables must not reproduce the hand-assembled batch."""
    g = json.load(open(GOLD))
    base = dict(wf=g["wf"], tp=g["tel_n_pixels"], ts=g["tel_n_samples"], tw=g["tel_W"],
                tc=g["tel_calib_offset"], bt=g["blk_tel"], bw=g["blk_wf_offset"], bo=g["blk_out_offset"])

    def go(**kw):
        a = dict(base, **kw)
        wf = np.concatenate([np.array(a["wf"], np.uint16), np.zeros(64, np.uint16)])
        r = oracle.extract_ragged(wf, a["tp"], a["ts"], a["tw"], a["tc"], a["bt"], a["bw"], a["bo"],
                                  g["pedestal"] + [0] * 8, g["gain"] + [1.0] * 8, 16)
        return r[0][:6].tolist(), r[1][:6].tolist()
    good = (g["out_sum"], g["out_start"])
    assert go() == good
    assert go(tc=[0, 2, 4]) != good                         # calibration offsets taken in telescope order
    assert go(bw=[2 * x for x in g["blk_wf_offset"]]) != good   # offsets in bytes instead of samples
    assert go(tw=[3, 2, 2]) != good                         # windows swapped between telescopes
    assert go(bt=[1, 0, 2, 2]) != good                      # wrong telescope for the last block


def test_bad_tables_are_rejected():
    with pytest.raises(ValueError):
        oracle.extract_ragged([1, 2, 3, 4], [1], [4], [2], [0], [1], [0], [0], [0], [1.0], 1)   # tel out of range
    with pytest.raises(ValueError):
        oracle.extract_ragged([1, 2, 3, 4], [1], [4], [5], [0], [0], [0], [0], [0], [1.0], 1)   # W > S
    with pytest.raises(ValueError):
        oracle.extract_ragged([1, 2, 3], [1], [4], [2], [0], [0], [0], [0], [0], [1.0], 1)      # block leaves wf
