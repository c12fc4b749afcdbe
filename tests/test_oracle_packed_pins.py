"""Pins for the packed-sample oracle (oracle/rta_oracle_packed.cpp; CPU only).

The paper only says the DL0 data travel as "a logical sequence of bits"
(§5); the P12 format is DESIGN.md readings R25-R27. The decoder is
pinned to: hand-worked byte fixtures (tests/golden/packed12.json), a numpy
bit-level restatement written here (np.unpackbits, little-endian bit order), a
pure-Python big-integer restatement, every 12-bit value at both nibble phases,
closed-form byte patterns, and mutation checks (a plausible wrong format fails
the fixtures). No expected value comes from the oracle, from dl0gen's encoder
or from the CUDA path.
"""
import json
import os

import numpy as np
import pytest

import oracle
from tests._checks import np_extract

GOLD = os.path.join(os.path.dirname(__file__), "golden", "packed12.json")


def np_unpack12(packed, n):
    """numpy restatement: the stream as a little-endian bit string, 12 bits per sample."""
    bits = np.unpackbits(np.asarray(packed, np.uint8), bitorder="little")[: 12 * n]
    return (bits.reshape(n, 12).astype(np.uint32) << np.arange(12, dtype=np.uint32)).sum(1).astype(np.uint16)


def py_unpack12(packed, n):
    """big-integer restatement: the whole stream is one little-endian integer."""
    big = int.from_bytes(bytes(bytearray(int(b) for b in packed)), "little")
    return [(big >> (12 * i)) & 0xFFF for i in range(n)]


def py_pack12(samples):
    """big-integer encoder, used only to build inputs for the pins below."""
    big = 0
    for i, v in enumerate(samples):
        big |= (int(v) & 0xFFF) << (12 * i)
    return np.frombuffer(big.to_bytes((12 * len(samples) + 7) // 8, "little"), np.uint8)


def test_hand_worked_fixtures():
    cases = json.load(open(GOLD))["cases"]
    assert len(cases) >= 10
    for c in cases:
        got = oracle.unpack12(np.array(c["bytes"], np.uint8), len(c["samples"]))
        assert got.tolist() == c["samples"], c["name"]


def test_plausible_wrong_formats_fail_the_fixtures():
    """A big-endian nibble order, or swapping the two samples of a pair, cannot
    reproduce the fixtures: they do discriminate."""
    cases = json.load(open(GOLD))["cases"]

    def big_endian(b, n):       # a = b0<<4 | b1>>4 ; b = (b1&0xF)<<8 | b2
        out = []
        for k in range(0, n, 2):
            b0, b1 = b[3 * k // 2], b[3 * k // 2 + 1]
            out.append((b0 << 4) | (b1 >> 4))
            if k + 1 < n:
                out.append(((b1 & 0xF) << 8) | b[3 * k // 2 + 2])
        return out

    def swapped(b, n):
        good = py_unpack12(b + [0], n + (n & 1))
        return [good[i ^ 1] for i in range(n - (n & 1))] + ([good[n - 1]] if n & 1 else [])

    for wrong in (big_endian, swapped):
        assert any(wrong(c["bytes"], len(c["samples"])) != c["samples"] for c in cases)


def test_every_value_at_both_nibble_phases():
    v = np.arange(4096)
    for other in (0, 0xFFF, 0x5A5):
        even = np.stack([v, np.full(4096, other)], 1).ravel()     # value in the 'a' slot
        odd = np.stack([np.full(4096, other), v], 1).ravel()      # value in the 'b' slot
        for s in (even, odd):
            p = py_pack12(s.tolist())
            assert (oracle.unpack12(p, s.size) == s).all()
            assert (np_unpack12(p, s.size) == s).all()


def test_closed_form_byte_patterns():
    n = 64
    assert (oracle.unpack12(np.full(96, 0xFF, np.uint8), n) == 0xFFF).all()
    assert (oracle.unpack12(np.zeros(96, np.uint8), n) == 0).all()
    # FF 0F 00 repeated = (0xFFF, 0) pairs; 00 F0 FF = (0, 0xFFF) pairs
    assert oracle.unpack12(np.tile(np.array([0xFF, 0x0F, 0x00], np.uint8), 32), n).tolist() == [0xFFF, 0] * 32
    assert oracle.unpack12(np.tile(np.array([0x00, 0xF0, 0xFF], np.uint8), 32), n).tolist() == [0, 0xFFF] * 32
    # a single set bit b of the stream is bit (b % 12) of sample (b // 12)
    for bit in range(0, 96 * 8, 7):
        raw = np.zeros(96, np.uint8)
        raw[bit // 8] = 1 << (bit % 8)
        got = oracle.unpack12(raw, n)
        want = np.zeros(n, np.uint16)
        want[bit // 12] = 1 << (bit % 12)
        assert (got == want).all(), bit


@pytest.mark.parametrize("n", [0, 1, 2, 3, 7, 8, 31, 100, 1001, 4096])
def test_random_streams_against_numpy_and_bigint(n):
    rng = np.random.default_rng(n)
    raw = rng.integers(0, 256, oracle.packed12_nbytes(n)).astype(np.uint8)   # arbitrary bytes
    got = oracle.unpack12(raw, n)
    assert (got == np_unpack12(raw, n)).all()
    assert got.tolist() == py_unpack12(raw.tolist(), n)
    assert oracle.packed12_nbytes(n) == -(-12 * n // 8)


def test_short_stream_is_rejected():
    with pytest.raises(ValueError):
        oracle.unpack12(np.zeros(2, np.uint8), 2)


@pytest.mark.parametrize("E,P,S,W", [(3, 5, 30, 7), (2, 7, 25, 4), (1, 3, 128, 8), (5, 1, 9, 9), (2, 3, 7, 1)])
def test_extract_packed_equals_numpy_decode_then_numpy_extract(E, P, S, W):
    """decode (numpy bits) -> extract (numpy sliding_window_view): two
    restatements chained, against the oracle's packed entry point."""
    rng = np.random.default_rng(E * 1000 + S)
    wf = rng.integers(0, 4096, (E, P, S)).astype(np.uint16)
    wf[0, 0] = 4095                                   # every window ties
    ped = rng.integers(0, 600, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    packed = py_pack12(wf.ravel().tolist())
    want = np_extract(np_unpack12(packed, wf.size).reshape(E, P, S), ped, gain, W)
    got = oracle.extract_packed12(packed, E, ped, gain, S, W)
    assert (got[0] == want[0]).all() and (got[1] == want[1]).all()
    assert (got[2] == want[2]).all() and (got[3] == want[3]).all()


def test_dl0gen_encoder_round_trips_through_the_pinned_decoder():
    """The input generator's encoder (not part of the method) is checked here
    against the pinned decoder and the big-integer encoder."""
    import dl0gen
    rng = np.random.default_rng(5)
    for n in (0, 1, 2, 5, 64, 999):
        x = rng.integers(0, 4096, n).astype(np.uint16)
        p = dl0gen.pack12_cpu(x)
        assert p.size == oracle.packed12_nbytes(n)
        assert (p == py_pack12(x.tolist())).all()
        assert (oracle.unpack12(p, n) == x).all()
    # values above 12 bits are masked by the encoder
    x = np.array([0xFABC, 0x1123], np.uint16)
    assert oracle.unpack12(dl0gen.pack12_cpu(x), 2).tolist() == [0xABC, 0x123]
