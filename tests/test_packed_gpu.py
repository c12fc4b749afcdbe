"""GPU parity of the packed 12-bit ingest: the CUDA
path decodes a P12 stream inside the extraction kernel; the oracle decodes it
bit by bit (oracle/rta_oracle_packed.cpp) and then applies the sliding-window
definition. Same bar as the uint16 path: integers bit-exact, charge relative
1e-6, time absolute 1e-4 — and in fact bit-identical floats.

Inputs are packed by dl0gen's encoder or by the big-integer encoder written in
this file; expected values come from the oracle or from the fixtures of
tests/golden/packed12.json (hand-worked), never from the CUDA path."""
import itertools
import json
import os

import numpy as np
import pytest

import dl0gen
import oracle
from tests._checks import check_invariants
from tests._full import alloc_filled_outputs, compare_every_event, slabs
from tests._gpu import alloc_outputs, assert_parity, bit_identical

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden", "packed12.json")
SHAPES = [(30, 7), (40, 7), (25, 4), (128, 8)]          # specialised tile12 kernels


def py_pack12(samples, pad_nibble=0):
    """big-integer encoder (independent of dl0gen's): the stream is one
    little-endian integer, 12 bits per sample."""
    big = 0
    for i, v in enumerate(samples):
        big |= (int(v) & 0xFFF) << (12 * i)
    n = len(samples)
    nb = (12 * n + 7) // 8
    if n % 2:
        big |= (pad_nibble & 0xF) << (12 * n)
    return np.frombuffer(big.to_bytes(nb, "little"), np.uint8).copy()


def run_packed(packed, E, P, S, ped, gain, W, generic=False, offset=0):
    """packed: host uint8 stream. offset: byte offset of the device copy from a
    256-byte-aligned allocation (0 -> staged kernels, odd -> generic12)."""
    import torch
    import paper_1307_6489_b200 as rta
    buf = torch.zeros(packed.size + offset + 16, dtype=torch.uint8, device="cuda")
    buf[offset:offset + packed.size] = torch.from_numpy(packed).cuda()
    view = buf[offset:offset + packed.size]
    d_ped = torch.from_numpy(np.ascontiguousarray(ped, np.int32)).cuda()
    d_gain = torch.from_numpy(np.ascontiguousarray(gain, np.float32)).cuda()
    outs = alloc_outputs(E * P)
    try:
        rta.rta_debug_force_generic(generic)
        rta.rta_extract_packed12(view, E, P, S, d_ped, d_gain, W, *outs)
        torch.cuda.synchronize()
    finally:
        rta.rta_debug_force_generic(False)
    return tuple(o.cpu().numpy() for o in outs)


def all_paths(wf12, ped, gain, W):
    """wf12: uint16 [E][P][S] with 12-bit values. Oracle on the packed bytes vs
    the staged kernel, the generic kernel and an odd-byte-aligned stream."""
    E, P, S = wf12.shape
    packed = dl0gen.pack12_cpu(wf12)
    want = oracle.extract_packed12(packed, E, ped, gain, S, W)
    # decode-then-extract equals extraction of the unpacked samples (oracle vs oracle's own parts
    # is not a pin; it is here to keep the two test inputs in step)
    assert bit_identical(want, oracle.extract(wf12, ped, gain, W))
    for kw in ({}, {"generic": True}, {"offset": 1}, {"offset": 7}):
        got = run_packed(packed, E, P, S, ped, gain, W, **kw)
        assert_parity(got, want, str(kw))
        assert bit_identical(got, want), kw
    import paper_1307_6489_b200 as rta
    if rta.rta_kernel_name_packed12(S, W) == "tile12<jit>":
        # a shape without an ahead-of-time kernel: the run above took the run-time specialisation;
        # without it (no libnvrtc) the same call takes generic12
        rta.rta_debug_jit(False)
        try:
            assert rta.rta_kernel_name_packed12(S, W) == "generic12"
            assert bit_identical(run_packed(packed, E, P, S, ped, gain, W), want), "jit off"
        finally:
            rta.rta_debug_jit(True)
    return want


def test_hand_worked_byte_fixtures_decode_on_gpu():
    """One trace per sample (S = 1, W = 1, pedestal 0, gain 1): out_sum IS the
    decoded sample, so the hand-worked bytes pin the device decoder directly."""
    for c in json.load(open(GOLD))["cases"]:
        n = len(c["samples"])
        packed = np.array(c["bytes"], np.uint8)
        ped, gain = np.zeros(n, np.int32), np.ones(n, np.float32)
        for kw in ({}, {"offset": 3}):
            s, t, q, tm = run_packed(packed, 1, n, 1, ped, gain, 1, **kw)
            assert s.tolist() == c["samples"], c["name"]
            assert (t == 0).all() and q.tolist() == [float(v) for v in c["samples"]]


def test_every_12bit_value_at_both_nibble_phases():
    vals = np.arange(4096, dtype=np.uint16)
    for lead in (0, 1):                                   # even / odd position of value v
        samples = np.concatenate([np.zeros(lead, np.uint16), vals, vals[::-1]])
        samples = np.concatenate([samples, np.zeros(-samples.size % 12, np.uint16)])
        n = samples.size
        packed = py_pack12(samples.tolist())
        ped, gain = np.zeros(n, np.int32), np.ones(n, np.float32)
        s, _, _, _ = run_packed(packed, 1, n, 1, ped, gain, 1)
        assert (s == samples).all()
        # the same stream as 12-sample-wide traces through a window
        wf = samples.reshape(1, n // 12, 12)
        ped2 = np.zeros(n // 12, np.int32)
        want = oracle.extract(wf, ped2, np.ones(n // 12, np.float32), 3)
        got = run_packed(packed, 1, n // 12, 12, ped2, np.ones(n // 12, np.float32), 3)
        assert bit_identical(got, want)


def test_padding_nibble_of_an_odd_stream_is_ignored():
    rng = np.random.default_rng(3)
    E, P, S, W = 1, 3, 25, 4                               # 75 samples: odd
    wf = rng.integers(0, 4096, (E, P, S)).astype(np.uint16)
    ped = np.array([100, 2000, 4000], np.int32)
    gain = np.array([1.0, 0.9, 1.1], np.float32)
    want = oracle.extract(wf, ped, gain, W)
    for pad in (0x0, 0xF, 0x5):
        packed = py_pack12(wf.ravel().tolist(), pad_nibble=pad)
        assert bit_identical(oracle.extract_packed12(packed, E, ped, gain, S, W), want)
        for kw in ({}, {"generic": True}, {"offset": 5}):
            assert bit_identical(run_packed(packed, E, P, S, ped, gain, W, **kw), want)


@pytest.mark.parametrize("S,W", SHAPES)
def test_exhaustive_tie_patterns_in_specialised_shapes(S, W):
    pats = np.array(list(itertools.product([0, 1], repeat=12)), np.uint16)  # 4096
    for off in (0, (S - 12) // 2, S - 12):
        tr = np.full((4096, S), 100, np.uint16)
        tr[:, off:off + 12] += pats * 5
        wf = tr.reshape(64, 64, S)
        ped = np.full(64, 100, np.int32)
        ped[::3] = 101
        all_paths(wf, ped, np.linspace(0.9, 1.1, 64).astype(np.float32), W)


@pytest.mark.parametrize("S,W", SHAPES)
def test_closed_forms_in_specialised_shapes(S, W):
    P = 3
    ped = np.array([400, 0, 4095], np.int32)
    gain = np.array([1.0, 0.5, 1.0625], np.float32)
    for c in (0, 400, 4095):                               # P1 constant traces
        wf = np.full((5, P, S), c, np.uint16)
        s, t, q, tm = run_packed(dl0gen.pack12_cpu(wf), 5, P, S, ped, gain, W)
        assert (t == 0).all()
        assert (s.reshape(5, P) == W * (c - ped.astype(np.int64))).all()
        assert (tm == np.float32((W - 1) / 2)).all()
        assert (q.reshape(5, P) == (W * (c - ped.astype(np.float64)) * gain).astype(np.float32)).all()
    A = 57                                                 # P2 delta at every position
    ped = np.array([400, 0, 4000], np.int32)
    wf = np.broadcast_to(ped.astype(np.uint16)[None, :, None], (S, P, S)).copy()
    for k in range(S):
        wf[k, :, k] += A
    s, t, q, tm = run_packed(dl0gen.pack12_cpu(wf), S, P, S, ped, gain, W)
    ks = np.repeat(np.arange(S), P)
    assert (s == A).all() and (t == np.maximum(0, ks - W + 1)).all()
    assert (tm == ks.astype(np.float32)).all()
    all_paths(wf, ped, gain, W)


@pytest.mark.parametrize("S,W", SHAPES + [(31, 5), (64, 16), (7, 7), (9, 1), (200, 3), (1, 1)])
@pytest.mark.parametrize("n_traces_shape", [(1, 1), (3, 5), (7, 37), (2, 129), (5, 257), (4, 1031), (3, 683)])
def test_random_12bit_and_ragged_sizes(S, W, n_traces_shape):
    """Full 12-bit range, sizes around the tile boundaries, odd sample totals,
    pedestals of both signs and beyond the samples."""
    E, P = n_traces_shape
    rng = np.random.default_rng(S * 7919 + W * 31 + E * P)
    wf = rng.integers(0, 4096, size=(E, P, S)).astype(np.uint16)
    wf[rng.random((E, P)) < 0.2] = 4095                   # saturated traces: every window ties
    ped = rng.integers(-70000, 70000, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    all_paths(wf, ped, gain, W)


@pytest.mark.parametrize("S,W", SHAPES)
def test_extreme_pedestals_and_gains(S, W):
    rng = np.random.default_rng(S)
    E, P = 3, 300
    wf = rng.integers(0, 4096, size=(E, P, S)).astype(np.uint16)
    ped = rng.integers(-2 ** 30, 2 ** 30, P).astype(np.int32)
    gain = rng.uniform(-3, 3, P).astype(np.float32)
    gain[0], gain[1], gain[2] = np.float32("nan"), np.float32("inf"), np.float32(1e-42)
    packed = dl0gen.pack12_cpu(wf)
    want = oracle.extract_packed12(packed, E, ped, gain, S, W)
    got = run_packed(packed, E, P, S, ped, gain, W)
    assert (got[0] == want[0]).all() and (got[1] == want[1]).all()
    assert bit_identical(got, want)


def test_C1_full_parity_packed():
    c = dl0gen.CONFIGS["C1"]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, threads=4)
    want = all_paths(wf, ped, gain, c.W)
    check_invariants(wf, ped, gain, c.W, *want)


@pytest.mark.parametrize("name,n_ev", [("C2", 23), ("C3", 19), ("C4", 11)])
def test_config_models_small_batches_packed(name, n_ev):
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, 100, n_ev, threads=4)
    all_paths(wf, ped, gain, c.W)


def test_device_encoder_matches_host_encoder():
    """dl0gen's two P12 encoders (input preparation) write the same bytes."""
    import torch
    c = dl0gen.CONFIGS["C3"]
    wf = dl0gen.events_cpu(c, 7, 5, threads=4)             # 5 * 1764 * 25 samples
    d_wf = torch.from_numpy(wf.view(np.int16)).cuda()
    nb = dl0gen.packed12_nbytes(wf.size)
    d_pk = torch.zeros(nb, dtype=torch.uint8, device="cuda")
    dl0gen.pack12_cuda(d_wf.data_ptr(), wf.size, d_pk.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert (d_pk.cpu().numpy() == dl0gen.pack12_cpu(wf)).all()
    assert (oracle.unpack12(d_pk.cpu().numpy(), wf.size) == wf.ravel()).all()


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_full_size_configs_packed_every_event_against_oracle(name):
    """BASELINE.json's full sizes as bench.py's packed leg runs them: generate
    on the GPU, pack on the GPU, one rta_extract_packed12 over the whole stream
    into sentinel-filled outputs; EVERY event against the oracle's bit-by-bit
    decoder + extraction on the packed bytes copied back in slabs (all host
    cores). A few blocks are also regenerated and packed on the host (device
    bytes == host packer's bytes) and put through the invariants."""
    import torch
    import paper_1307_6489_b200 as rta
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    st = torch.cuda.current_stream().cuda_stream
    n_samples_total = c.n_traces * c.n_samples
    d_wf = torch.empty((c.n_events, c.n_pixels, c.n_samples), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(c, d_wf.data_ptr(), 0, c.n_events, st)
    d_pk = torch.empty(dl0gen.packed12_nbytes(n_samples_total), dtype=torch.uint8, device="cuda")
    dl0gen.pack12_cuda(d_wf.data_ptr(), n_samples_total, d_pk.data_ptr(), st)
    torch.cuda.synchronize()
    del d_wf
    outs = alloc_filled_outputs(c.n_traces)
    before = rta.rta_launch_count()
    rta.rta_extract_packed12(d_pk, c.n_events, c.n_pixels, c.n_samples, torch.from_numpy(ped).cuda(),
                             torch.from_numpy(gain).cuda(), c.W, *outs)
    torch.cuda.synchronize()
    assert rta.rta_launch_count() == before + 1
    ev_samples = c.n_pixels * c.n_samples
    assert ev_samples % 2 == 0                              # every event starts on a byte
    ev_bytes = ev_samples * 3 // 2
    n = compare_every_event(
        c.n_events, c.n_pixels, slabs(c.n_events, ev_bytes, 256 << 20),
        lambda e0, k: d_pk[e0 * ev_bytes:(e0 + k) * ev_bytes].cpu().numpy(),
        lambda pk, a, b: oracle.extract_packed12(pk[a * ev_bytes:b * ev_bytes], b - a, ped, gain,
                                                 c.n_samples, c.W), outs)
    assert n == c.n_events
    rng = np.random.default_rng(6)
    for e0 in [0, c.n_events - 12] + sorted(rng.integers(12, c.n_events - 24, 2).tolist()):
        wf = dl0gen.events_cpu(c, e0, 12, threads=4)
        pk = dl0gen.pack12_cpu(wf)
        assert (d_pk[e0 * ev_bytes:e0 * ev_bytes + pk.size].cpu().numpy() == pk).all()
        lo, hi = e0 * c.n_pixels, (e0 + 12) * c.n_pixels
        got = tuple(o[lo:hi].cpu().numpy() for o in outs)
        assert_parity(got, oracle.extract_packed12(pk, 12, ped, gain, c.n_samples, c.W),
                      "%s events %d.." % (name, e0))
        check_invariants(wf, ped, gain, c.W, *got)


# ---- host-fed packed path ---------------------------------------------------
def _small_case(name="C5", n_ev=41, first=1234):
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    wf = dl0gen.events_cpu(c, first, n_ev, threads=4)
    pk = dl0gen.pack12_cpu(wf)
    return c, ped, gain, wf, pk, oracle.extract_packed12(pk, n_ev, ped, gain, c.n_samples, c.W)


@pytest.mark.parametrize("pinned", [True, False])
@pytest.mark.parametrize("name,chunk_events", [("C5", 1), ("C5", 7), ("C5", 40), ("C5", 41), ("C5", 1000),
                                               ("C3", 9), ("C3", 33), ("C1", 5)])
def test_stream_packed_small_odd_chunking(pinned, name, chunk_events):
    """Chunks are whole events starting on 16-byte boundaries of the stream
    (C5/C1: multiples of 4 events; C3 (1764 x 25): multiples of 8)."""
    import torch
    import paper_1307_6489_b200 as rta
    c, ped, gain, wf, pk, want = _small_case(name)
    n_ev = wf.shape[0]
    host = torch.from_numpy(pk)
    if pinned:
        host = host.pin_memory()
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    outs = alloc_outputs(n_ev * c.n_pixels)
    ev_bytes = c.n_pixels * c.n_samples * 3 // 2
    cb = chunk_events * ev_bytes + 17
    before = rta.rta_launch_count()
    rta.rta_extract_stream_packed12(host, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs,
                                    chunk_bytes=cb)
    torch.cuda.synchronize()
    ce = rta.rta_chunk_events(n_ev, c.n_pixels, c.n_samples, cb, 12)
    assert rta.rta_launch_count() - before == -(-n_ev // ce)
    got = tuple(o.cpu().numpy() for o in outs)
    assert_parity(got, want)
    assert bit_identical(got, want)
    rta.rta_extract_stream_packed12(host, n_ev, c.n_pixels, c.n_samples, d_ped, d_gain, c.W, *outs,
                                    chunk_bytes=3 * ev_bytes)
    torch.cuda.synchronize()
    assert bit_identical(tuple(o.cpu().numpy() for o in outs), want)


@pytest.mark.parametrize("chunk_events", [0, 5, 64])
def test_extract_host_packed_end_to_end(chunk_events):
    import paper_1307_6489_b200 as rta
    c, ped, gain, wf, pk, want = _small_case(n_ev=37, first=77)
    n = 37 * c.n_pixels
    outs = (np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.float32),
            np.zeros(n, np.float32))
    rta.rta_extract_host_packed12(pk, 37, c.n_pixels, c.n_samples, ped, gain, c.W, *outs,
                                  chunk_bytes=chunk_events * c.n_pixels * c.n_samples * 3 // 2)
    assert bit_identical(outs, want)
    # 16-bit and 12-bit calls share one workspace: alternate them
    outs16 = tuple(np.zeros_like(o) for o in outs)
    rta.rta_extract_host(wf, 37, c.n_pixels, c.n_samples, ped, gain, c.W, *outs16, chunk_bytes=1 << 20)
    assert bit_identical(outs16, want)
    outs2 = tuple(np.zeros_like(o) for o in outs)
    rta.rta_extract_host_packed12(pk, 37, c.n_pixels, c.n_samples, ped, gain, c.W, *outs2)
    assert bit_identical(outs2, want)


@pytest.mark.parametrize("S,W,P", [(60, 7, 1855), (31, 5, 333), (96, 8, 512)])
def test_stream_and_host_variants_on_shapes_without_an_ahead_of_time_kernel(S, W, P):
    """The host-fed P12 calls on shapes that take the run-time specialisation of the P12
    kernel (or generic12 without the compiler): several chunks, every chunk a kernel launch on
    a 16-byte-aligned slice of the stream, against the bit-by-bit oracle."""
    import torch
    import paper_1307_6489_b200 as rta
    rng = np.random.default_rng(S * 100 + W)
    n_ev = 37
    wf = rng.integers(0, 4096, size=(n_ev, P, S)).astype(np.uint16)
    wf[rng.random((n_ev, P)) < 0.1] = 4095
    ped = rng.integers(0, 600, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    pk = dl0gen.pack12_cpu(wf)
    want = oracle.extract_packed12(pk, n_ev, ped, gain, S, W)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    ev_bytes = P * S * 3 // 2
    for chunk_events in (5, 16, 1000):
        outs = alloc_outputs(n_ev * P)
        rta.rta_extract_stream_packed12(torch.from_numpy(pk).pin_memory(), n_ev, P, S, d_ped, d_gain, W, *outs,
                                        chunk_bytes=chunk_events * ev_bytes + 3)
        torch.cuda.synchronize()
        assert bit_identical(tuple(o.cpu().numpy() for o in outs), want), chunk_events
    rta.rta_debug_jit(False)
    try:
        outs = alloc_outputs(n_ev * P)
        rta.rta_extract_stream_packed12(torch.from_numpy(pk), n_ev, P, S, d_ped, d_gain, W, *outs,
                                        chunk_bytes=9 * ev_bytes)
        torch.cuda.synchronize()
        assert bit_identical(tuple(o.cpu().numpy() for o in outs), want), "jit off"
    finally:
        rta.rta_debug_jit(True)
