"""GPU parity of the any-shape staged kernel (runtime S and W)
against the oracle, through rta_extract: every combination of the kernel's
cases — word stride odd / 2 mod 4 / 0 mod 4 (lane groups skewed by one word),
units of a multiple of 32 bytes (padded layout, 16-byte cp.async ingest), odd S
(two traces per thread), fewer windows than the skew, W = 1 and W = S, several
tiles per CTA plus a ragged tail, cameras smaller than a unit (the calibration
index wraps inside a unit). The old generic kernel must agree bit for bit."""
import numpy as np
import pytest

import oracle
from tests._gpu import bit_identical, run_gpu

pytestmark = pytest.mark.gpu

# (S, W): words per unit s, g = gcd(s, 32) -> case
SHAPES = [
    (50, 8),     # s = 25, g = 1
    (60, 7),     # s = 30, g = 2
    (20, 3),     # s = 10, g = 2
    (40, 5),     # s = 20, g = 4
    (24, 24),    # s = 12, g = 4, one window
    (40, 38),    # three windows, fewer than the skew of 6
    (200, 9),    # s = 100, g = 4, 128 threads per CTA
    (96, 8),     # 192-byte units: padded layout
    (128, 10),   # 256-byte units: padded layout, 128 threads
    (64, 1),     # padded, W = 1
    (16, 5),     # 32-byte units: padded, 48-byte stride
    (576, 12),   # the largest unit (1152 bytes), 32 threads per CTA
    (33, 5),     # odd S: two traces per thread, s = 33
    (27, 27),    # odd S, one window
    (3, 2), (2, 1), (1, 1),
    (287, 6),    # odd S, 1148-byte units
]


@pytest.mark.parametrize("S,W", SHAPES)
@pytest.mark.parametrize("E,P", [(1, 1), (5, 3), (3, 700), (2, 5000)])
def test_any_shape_random(S, W, E, P):
    import paper_1307_6489_b200 as rta
    jit = 2 * S * (2 if S % 2 else 1) <= 320        # the unit fits a register copy: run-time specialisation
    assert rta.rta_kernel_name(S, W) == ("staged<jit>" if jit else "staged<any>")
    if E * P * S > 3_000_000:
        E = 1
    rng = np.random.default_rng(S * 1009 + W * 31 + E * P)
    full = (S + W) % 2 == 0
    hi = 65536 if full else 4096
    wf = rng.integers(0, hi, size=(E, P, S)).astype(np.uint16)
    wf[rng.random((E, P)) < 0.15] = hi - 1                     # all windows tie
    wf[rng.random((E, P)) < 0.15] //= np.uint16(hi // 2)       # tie-heavy
    ped = (rng.integers(-70000, 70000, P) if full else rng.integers(0, 600, P)).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    want = oracle.extract(wf, ped, gain, W)
    got = run_gpu(wf, ped, gain, W)                  # NVRTC specialisation where eligible
    assert (got[0] == want[0]).all() and (got[1] == want[1]).all()
    assert bit_identical(got, want)
    rta.rta_debug_jit(False)                         # the runtime-shape kernel (no libnvrtc needed)
    try:
        assert rta.rta_kernel_name(S, W) == "staged<any>"
        assert bit_identical(run_gpu(wf, ped, gain, W), want)
    finally:
        rta.rta_debug_jit(True)
    old = run_gpu(wf, ped, gain, W, generic=True)
    assert bit_identical(got, old)


@pytest.mark.parametrize("S,W", [(60, 7), (40, 5), (96, 8), (33, 5)])
def test_any_shape_many_tiles_both_schedules(S, W):
    """Several tiles per CTA, dynamic and static tile schedules, a ragged tail
    of every length class (odd number of traces for the two-traces-per-thread case)."""
    import paper_1307_6489_b200 as rta
    rng = np.random.default_rng(S)
    E, P = 37, 1855 + (S % 2)
    wf = (400 + rng.normal(0, 4, (E, P, S))).round().clip(0, 4095).astype(np.uint16)
    wf[:, ::11, S // 3: S // 3 + 4] += np.uint16(300)
    ped = rng.integers(380, 421, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
    want = oracle.extract(wf, ped, gain, W)
    for jit in (True, False):                        # run-time specialisation / runtime-shape kernel
        for static in (False, True):
            rta.rta_debug_static_schedule(static)
            rta.rta_debug_jit(jit)
            try:
                got = run_gpu(wf, ped, gain, W)
            finally:
                rta.rta_debug_static_schedule(False)
                rta.rta_debug_jit(True)
            assert bit_identical(got, want), (jit, static)


def test_any_shape_closed_forms():
    """Delta at every position and constant traces (SURVEY.md pins P1, P2) for a
    g = 4 shape: earliest of the tied windows through the skewed lane groups."""
    S, W, ped = 40, 5, 100
    wf = np.full((1, S + 1, S), ped, np.uint16)
    for k in range(S):
        wf[0, k, k] = ped + 50
    wf[0, S, :] = 777
    import paper_1307_6489_b200 as rta
    for jit in (True, False):
        rta.rta_debug_jit(jit)
        try:
            got = run_gpu(wf, np.full(S + 1, ped, np.int32), np.ones(S + 1, np.float32), W)
        finally:
            rta.rta_debug_jit(True)
        for k in range(S):
            assert got[0][k] == 50 and got[1][k] == max(0, k - W + 1) and got[3][k] == np.float32(k)
        assert got[0][S] == W * (777 - ped) and got[1][S] == 0 and got[3][S] == np.float32((W - 1) / 2)


@pytest.mark.parametrize("S,W", [(30, 7), (40, 7), (25, 4), (60, 7), (50, 8), (200, 9), (33, 5), (128, 8), (96, 8)])
@pytest.mark.parametrize("off", [1, 2, 3, 5, 7])
def test_unaligned_base_pointers(S, W, off):
    """A waveform pointer `off` halfwords past a 16-byte boundary: dense layouts
    (the specialised shapes included) take the runtime-shape kernel with the tile
    landing `mis` bytes into the stage, padded layouts the generic kernel. The
    buffer ends exactly at the last sample and is followed by a guard whose value
    must not matter; numbers of traces with and without a ragged tail."""
    import torch
    import paper_1307_6489_b200 as rta
    from tests._gpu import alloc_outputs
    rng = np.random.default_rng(S * 10 + off)
    padded = (2 * S * (2 if S % 2 else 1)) % 32 == 0
    assert rta.rta_kernel_name(S, W, aligned16=False) == ("generic" if padded else "staged<any>")
    for E, P in ((3, 1855), (2, 512), (1, 5)):
        wf = rng.integers(0, 4096, size=(E, P, S)).astype(np.uint16)
        ped = rng.integers(0, 600, P).astype(np.int32)
        gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
        want = oracle.extract(wf, ped, gain, W)
        for guard in (0, -1):
            buf = torch.full((wf.size + off + 16,), guard, dtype=torch.int16, device="cuda")
            assert buf.data_ptr() % 16 == 0
            buf[off:off + wf.size] = torch.from_numpy(wf.reshape(-1).view(np.int16)).cuda()
            view = buf[off:off + wf.size]
            outs = alloc_outputs(E * P)
            rta.rta_extract(view, E, P, S, torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda(),
                            W, *outs)
            torch.cuda.synchronize()
            assert bit_identical(tuple(o.cpu().numpy() for o in outs), want), (E, P, guard)


# ---- several lanes per trace (shuffle prefix sums): long traces, and any S % 8 == 0 on request
def _tie_heavy(rng, E, P, S, hi):
    wf = rng.integers(0, hi, size=(E, P, S)).astype(np.uint16)
    wf[rng.random((E, P)) < 0.15] = hi - 1                     # all windows tie
    wf[rng.random((E, P)) < 0.15] //= np.uint16(hi // 2)       # tie-heavy
    return wf


@pytest.mark.parametrize("S,W", [(584, 9), (1000, 32), (2048, 12), (2048, 1), (4096, 7), (8192, 3), (800, 40),
                                 (1024, 1024 // 512), (578, 9), (289, 9), (601, 2), (1001, 30), (3000, 10),
                                 (20000, 1), (16000, 2), (2050, 15), (2050, 12), (2052, 9)])
def test_long_traces_take_a_thread_per_segment(S, W):
    """Units above 1152 bytes: the segment kernel (a thread per run of window starts, keys of
    a trace merged by a shared-memory atomicMax) instead of the strided generic kernel, for
    any n_samples (odd ones included: the tile then holds a multiple of 8 traces); both
    against the oracle, full uint16 range where the ABI guard allows; trace counts that
    leave the last tile partly empty and not a multiple of 16 bytes long."""
    import paper_1307_6489_b200 as rta
    assert rta.rta_kernel_name(S, W) == "segments"
    rng = np.random.default_rng(S + W)
    for E, P in ((1, 1), (3, 37), (2, 700), (1, 67)):
        if E * P * S > 3_000_000:
            P = max(1, 3_000_000 // (E * S))
        hi = 65536 if S * W * 65535 < 2 ** 31 and W % 2 else 4096
        if S * W * (hi - 1) >= 2 ** 31:
            hi = max(2, (2 ** 31 - 1) // (S * W))
        wf = _tie_heavy(rng, E, P, S, hi)
        ped = rng.integers(0, 600, P).astype(np.int32)
        gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
        want = oracle.extract(wf, ped, gain, W)
        assert bit_identical(run_gpu(wf, ped, gain, W), want), (E, P)
        for static in (True,):
            rta.rta_debug_static_schedule(static)
            try:
                assert bit_identical(run_gpu(wf, ped, gain, W), want), (E, P, "static")
            finally:
                rta.rta_debug_static_schedule(False)
        assert bit_identical(run_gpu(wf, ped, gain, W, generic=True), want), (E, P)


@pytest.mark.parametrize("L,TR,NT,ST", [(34, 8, 128, 2), (66, 0, 0, 0), (130, 16, 256, 4), (2, 8, 32, 3), (6, 64, 64, 2),
                                         (258, 0, 0, 0), (66, 1, 32, 4)])
@pytest.mark.parametrize("S,W", [(128, 8), (40, 7), (25, 4), (33, 33), (96, 1), (1000, 32), (2048, 12)])
def test_segment_kernel_on_any_shape(L, TR, NT, ST, S, W):
    """The segment kernel forced onto shapes that normally take a thread per trace, with
    segment lengths from 2 window starts (every segment is one or two windows) to more
    than a trace (one segment), several traces per thread pass, tiles of 1 to 64 traces, two
    to four stages; n_samples a multiple of 8 (one bulk copy per trace, padded stride) or not
    (dense tiles)."""
    import paper_1307_6489_b200 as rta
    rng = np.random.default_rng(L * 1000 + S)
    for E, P in ((1, 1), (2, 37), (3, 1855)):
        if E * P * S > 3_000_000:
            P = max(1, 3_000_000 // (E * S))
        wf = _tie_heavy(rng, E, P, S, 4096)
        ped = rng.integers(-70000, 70000, P).astype(np.int32)
        gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
        want = oracle.extract(wf, ped, gain, W)
        rta.rta_debug_seg_tuning(L, TR, NT, ST)
        try:
            got = run_gpu(wf, ped, gain, W)
        finally:
            rta.rta_debug_seg_tuning(0, 0, 0, 0)
        assert bit_identical(got, want), (E, P)


@pytest.mark.parametrize("lpt", [4, 8, 16, 32])
@pytest.mark.parametrize("S,W", [(128, 8), (40, 7), (8, 8), (16, 1), (96, 9), (256, 20)])
def test_lanes_per_trace_on_short_traces(lpt, S, W):
    """The same kernel with 4, 8, 16 or 32 lanes per trace on shapes that normally take a
    thread per trace (the measurement of DESIGN.md section 5g): bit-identical to the oracle,
    trace counts that leave groups and warps partly empty."""
    import paper_1307_6489_b200 as rta
    rng = np.random.default_rng(lpt * 1000 + S)
    for E, P in ((1, 1), (2, 37), (3, 1855)):
        wf = _tie_heavy(rng, E, P, S, 4096)
        ped = rng.integers(-70000, 70000, P).astype(np.int32)
        gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
        want = oracle.extract(wf, ped, gain, W)
        rta.rta_debug_lanes_per_trace(lpt)
        try:
            got = run_gpu(wf, ped, gain, W)
        finally:
            rta.rta_debug_lanes_per_trace(0)
        assert bit_identical(got, want), (E, P)
