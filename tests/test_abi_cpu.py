"""CPU-only checks of the boundary: librta.so builds, loads, exports every
symbol include/rta.h declares, and rejects bad arguments before touching CUDA
(pin P17). No compute call is made here."""
import ctypes
import os
import re

import pytest

import paper_1307_6489_b200 as rta

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rta.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rta_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = rta.lib()
    names = declared_symbols()
    assert {"rta_extract", "rta_extract_stream", "rta_extract_host", "rta_strerror",
            "rta_last_cuda_error", "rta_kernel_name", "rta_launch_count",
            "rta_shutdown"} <= set(names)
    for n in names:
        assert hasattr(L, n), n


def test_shipped_library_exports_exactly_the_header():
    """librta.so is built with hidden visibility: its defined dynamic function
    symbols are the functions include/rta.h declares, no test hook, no internal
    C++ symbol. The hooks exist in librta_testing.so only."""
    import subprocess
    from paper_1307_6489_b200 import build as b

    def exported(path):
        out = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True,
                             text=True, check=True).stdout
        return sorted(f[2] for f in (ln.split() for ln in out.splitlines())
                      if len(f) == 3 and f[1] == "T")
    rta.lib()
    assert exported(b.LIB) == declared_symbols()
    hooks = {"rta_extract_generic", "rta_extract_image_generic", "rta_debug_force_generic",
             "rta_debug_static_schedule", "rta_debug_serial_ragged", "rta_debug_general_cleaning",
             "rta_debug_jit", "rta_debug_lanes_per_trace", "rta_debug_seg_tuning"}
    assert set(exported(b.TEST_LIB)) == set(declared_symbols()) | hooks
    T = rta.testing_lib()
    for n in hooks:
        assert hasattr(T, n) and not hasattr(rta.lib(), n), n


def test_library_links_no_torch():
    import subprocess
    out = subprocess.run(["ldd", rta.lib()._name], capture_output=True, text=True).stdout
    assert "torch" not in out and "c10" not in out


def _call(n_events=1, n_pixels=4, n_samples=30, W=7, wf=0x1000, ped=0x2000, gain=0x3000,
          o=(0x4000, 0x5000, 0x6000, 0x7000)):
    return rta.lib().rta_extract(wf, n_events, n_pixels, n_samples, ped, gain, W, *o, 0)


def test_shape_errors_before_any_cuda_call():
    assert _call(W=0) == rta.RTA_ERR_SHAPE
    assert _call(W=31) == rta.RTA_ERR_SHAPE               # W > S
    assert _call(n_samples=0) == rta.RTA_ERR_SHAPE
    assert _call(n_pixels=0) == rta.RTA_ERR_SHAPE
    assert _call(n_events=-1) == rta.RTA_ERR_SHAPE


def test_unsupported_sizes():
    assert _call(n_events=2 ** 31, n_pixels=1) == rta.RTA_ERR_UNSUPPORTED
    assert _call(n_events=2 ** 20, n_pixels=2 ** 11) == rta.RTA_ERR_UNSUPPORTED
    assert _call(n_samples=2048, W=17) == rta.RTA_ERR_UNSUPPORTED   # 2048*17*65535 >= 2^31
    assert _call(n_samples=182, W=182) == rta.RTA_ERR_UNSUPPORTED


def test_null_and_alignment():
    assert _call(wf=None) == rta.RTA_ERR_NULL
    assert _call(ped=None) == rta.RTA_ERR_NULL
    assert _call(gain=None) == rta.RTA_ERR_NULL
    assert _call(o=(0x4000, None, 0x6000, 0x7000)) == rta.RTA_ERR_NULL
    assert _call(wf=0x1001) == rta.RTA_ERR_ALIGN
    assert _call(o=(0x4002, 0x5000, 0x6000, 0x7000)) == rta.RTA_ERR_ALIGN


def test_empty_input_is_ok_and_touches_nothing():
    # R17: no work -> RTA_OK even with null pointers, nothing enqueued
    before = rta.rta_launch_count()
    assert _call(n_events=0, wf=None, ped=None, gain=None, o=(None,) * 4) == rta.RTA_OK
    L = rta.lib()
    assert L.rta_extract_stream(None, 0, 4, 30, None, None, 7, None, None, None, None, 0, 0) == rta.RTA_OK
    assert L.rta_extract_host(None, 0, 4, 30, None, None, 7, None, None, None, None, 0) == rta.RTA_OK
    assert rta.rta_launch_count() == before


def test_stream_and_host_entry_points_validate_too():
    L = rta.lib()
    assert L.rta_extract_stream(0x1000, 1, 4, 30, 0x2000, 0x3000, 31, 0x4000, 0x5000,
                                0x6000, 0x7000, 0, 0) == rta.RTA_ERR_SHAPE
    assert L.rta_extract_host(0x1000, 1, 4, 30, None, 0x3000, 7, 0x4000, 0x5000,
                              0x6000, 0x7000, 0) == rta.RTA_ERR_NULL


def test_strerror_and_kernel_names():
    for s in range(0, 8):
        assert isinstance(rta.rta_strerror(s), str) and rta.rta_strerror(s)
    assert rta.rta_kernel_name(40, 7) == "tile<S=40,W=7>"
    assert rta.rta_kernel_name(30, 7) == "tile<S=30,W=7>"
    assert rta.rta_kernel_name(25, 4) == "tile<S=25,W=4>"
    assert rta.rta_kernel_name(128, 8) == "tile<S=128,W=8>"
    # a base that is only 2-byte aligned: dense layouts take the runtime-shape kernel,
    # units of a multiple of 32 bytes (padded layout, 16-byte cp.async) the generic one
    assert rta.rta_kernel_name(40, 7, aligned16=False) == "staged<any>"
    assert rta.rta_kernel_name(128, 8, aligned16=False) == "generic"
    # any other shape: units up to 320 bytes are compiled for their (S, W) at first use when
    # libnvrtc can be loaded (staged<jit>); otherwise, and for units up to 1152 bytes, the
    # staged kernel with runtime (S, W)
    assert rta.rta_kernel_name(41, 7) in ("staged<jit>", "staged<any>")
    assert rta.rta_kernel_name(60, 7) == rta.rta_kernel_name(160, 9) == rta.rta_kernel_name(41, 7)
    assert rta.rta_kernel_name(162, 9) == "staged<any>"
    rta.rta_debug_jit(False)
    try:
        assert rta.rta_kernel_name(41, 7) == rta.rta_kernel_name(60, 7) == "staged<any>"
    finally:
        rta.rta_debug_jit(True)
    assert rta.rta_kernel_name(576, 9) == "staged<any>" and rta.rta_kernel_name(287, 9) == "staged<any>"
    # longer traces: a thread per segment of a trace (any S that the ABI guard n_samples * W *
    # 65535 < 2^31 admits; the names below are what the dispatch would pick past that guard)
    assert rta.rta_kernel_name(578, 9) == "segments" and rta.rta_kernel_name(289, 9) == "segments"
    assert rta.rta_kernel_name(584, 9) == "segments" and rta.rta_kernel_name(2048, 12) == "segments"
    assert rta.rta_kernel_name(2048, 1000) == "lanes<32>" and rta.rta_kernel_name(2047, 1000) == "generic"
    assert rta.rta_kernel_name(65536, 4) == "generic" and rta.rta_kernel_name(40000, 4) == "segments"
    assert rta.rta_kernel_name(2048, 12, aligned16=False) == "generic"
    assert rta.rta_kernel_name(60, 7, aligned16=False) == "staged<any>"
    assert rta.rta_kernel_name(96, 8, aligned16=False) == "generic"


def test_binding_raises_on_error_status():
    with pytest.raises(rta.RtaError) as ei:
        rta.rta_extract(0x1000, 1, 4, 30, 0x2000, 0x3000, 99, 0x4000, 0x5000, 0x6000,
                        0x7000, stream=0)
    assert ei.value.status == rta.RTA_ERR_SHAPE


def test_no_cpu_fallback_without_a_device():
    """On a box without a GPU a real compute call must fail loudly."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import numpy as np
    wf = np.zeros((1, 4, 30), np.uint16)
    ped = np.zeros(4, np.int32)
    g = np.ones(4, np.float32)
    outs = [np.zeros(4, np.int32), np.zeros(4, np.int32), np.zeros(4, np.float32),
            np.zeros(4, np.float32)]
    with pytest.raises(rta.RtaError) as ei:
        rta.rta_extract_host(wf, 1, 4, 30, ped, g, 7, *outs)
    assert ei.value.status in (rta.RTA_ERR_CUDA, rta.RTA_ERR_NOMEM)


def test_shard_events_partitions_exactly():
    for n in (0, 1, 7, 10_000, 200_000):
        for w in (1, 2, 3, 8):
            parts = [rta.shard_events(n, w, r) for r in range(w)]
            assert parts[0][0] == 0
            assert sum(c for _, c in parts) == n
            for (a, ca), (b, _) in zip(parts, parts[1:]):
                assert a + ca == b
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1


# ---- extractor family (rta_extract_fixed / _local_peak / _fir) ---------------
def _taps(vals):
    return (ctypes.c_int32 * len(vals))(*vals)


def test_family_entry_points_validate_before_any_cuda_call():
    L = rta.lib()
    o = (0x4000, 0x5000, 0x6000, 0x7000)
    fixed = lambda **k: L.rta_extract_fixed(k.get("wf", 0x1000), k.get("E", 1), 4, 30, 0x2000, 0x3000,
                                            k.get("W", 7), k.get("ws", 0x8000), *o, 0)
    assert fixed(W=31) == rta.RTA_ERR_SHAPE
    assert fixed(ws=None) == rta.RTA_ERR_NULL
    assert fixed(ws=0x8002) == rta.RTA_ERR_ALIGN
    assert fixed(wf=None) == rta.RTA_ERR_NULL
    assert fixed(E=0, wf=None, ws=None) == rta.RTA_OK
    peak = lambda **k: L.rta_extract_local_peak(k.get("wf", 0x1000), k.get("E", 1), 4, 30, 0x2000, 0x3000,
                                                k.get("W", 7), k.get("shift", 3), *o, 0)
    assert peak(W=0) == rta.RTA_ERR_SHAPE
    assert peak(wf=0x1001) == rta.RTA_ERR_ALIGN
    assert peak(E=0, wf=None) == rta.RTA_OK
    fir = lambda taps, S=30, E=1, wf=0x1000: L.rta_extract_fir(
        wf, E, 4, S, 0x2000, 0x3000, _taps(taps) if taps is not None else None,
        len(taps) if taps is not None else 3, *o, 0)
    assert fir([1] * 31) == rta.RTA_ERR_SHAPE              # more taps than samples
    assert fir([1] * 33, S=64) == rta.RTA_ERR_UNSUPPORTED  # more than 32 taps
    assert fir(None) == rta.RTA_ERR_NULL
    assert fir([20000, -20000], S=30) == rta.RTA_ERR_UNSUPPORTED   # 30*40000*65535 >= 2^31
    assert fir([1, 2, 1], wf=None) == rta.RTA_ERR_NULL
    assert fir([1, 2, 1], E=0, wf=None) == rta.RTA_OK


# ---- packed 12-bit ingest (rta_extract_packed12 and the host-fed variants) ----
def test_packed12_entry_points_validate_before_any_cuda_call():
    L = rta.lib()
    o = (0x4000, 0x5000, 0x6000, 0x7000)
    dev = lambda **k: L.rta_extract_packed12(k.get("wf", 0x1001), k.get("E", 1), k.get("P", 4),
                                             k.get("S", 30), k.get("ped", 0x2000), 0x3000,
                                             k.get("W", 7), *k.get("o", o), 0)
    assert dev(W=31) == rta.RTA_ERR_SHAPE
    assert dev(W=0) == rta.RTA_ERR_SHAPE
    assert dev(P=0) == rta.RTA_ERR_SHAPE
    assert dev(E=-1) == rta.RTA_ERR_SHAPE
    assert dev(E=2 ** 31, P=1) == rta.RTA_ERR_UNSUPPORTED
    assert dev(wf=None) == rta.RTA_ERR_NULL
    assert dev(ped=None) == rta.RTA_ERR_NULL
    assert dev(ped=0x2002) == rta.RTA_ERR_ALIGN
    assert dev(o=(0x4001, 0x5000, 0x6000, 0x7000)) == rta.RTA_ERR_ALIGN
    assert dev(E=0, wf=None, ped=None) == rta.RTA_OK
    # a P12 stream may start on any byte: an odd address is not an alignment error
    # (without a device the call then fails in CUDA, never in validation)
    import torch
    if not torch.cuda.is_available():
        assert dev(wf=0x1001) in (rta.RTA_ERR_CUDA, rta.RTA_ERR_NOMEM)
    assert L.rta_extract_stream_packed12(0x1001, 1, 4, 30, 0x2000, 0x3000, 31, *o, 0, 0) == rta.RTA_ERR_SHAPE
    assert L.rta_extract_stream_packed12(None, 1, 4, 30, 0x2000, 0x3000, 7, *o, 0, 0) == rta.RTA_ERR_NULL
    assert L.rta_extract_stream_packed12(None, 0, 4, 30, None, None, 7, None, None, None, None, 0, 0) == rta.RTA_OK
    assert L.rta_extract_host_packed12(0x1001, 1, 4, 30, None, 0x3000, 7, *o, 0) == rta.RTA_ERR_NULL
    assert L.rta_extract_host_packed12(None, 0, 4, 30, None, None, 7, None, None, None, None, 0) == rta.RTA_OK


def test_packed12_kernel_names():
    assert rta.rta_kernel_name_packed12(40, 7) == "tile12<S=40,W=7>"
    assert rta.rta_kernel_name_packed12(30, 7) == "tile12<S=30,W=7>"
    assert rta.rta_kernel_name_packed12(25, 4) == "tile12<S=25,W=4>"
    assert rta.rta_kernel_name_packed12(128, 8) == "tile12<S=128,W=8>"
    assert rta.rta_kernel_name_packed12(40, 7, aligned16=False) == "generic12"
    assert rta.rta_kernel_name_packed12(41, 7) in ("tile12<jit>", "generic12")   # with / without libnvrtc
    assert rta.rta_kernel_name_packed12(300, 7) == "generic12"                   # 450-byte units: no register copy
    rta.rta_debug_jit(False)
    try:
        assert rta.rta_kernel_name_packed12(41, 7) == "generic12"
    finally:
        rta.rta_debug_jit(True)


def test_chunk_events_planning():
    """Host logic of the host-fed calls (R21, R27): whole events, rounded
    down, at least one; P12 chunks start on a 16-byte boundary of the stream."""
    ce = rta.rta_chunk_events
    # BASELINE.json:configs[4]: 1 GiB chunks of 1855 x 40 uint16 events -> 7235 events, 28 chunks
    assert ce(200_000, 1855, 40, 1 << 30, 16) == 7235
    assert ce(200_000, 1855, 40, 0, 16) == 7235                       # 0 = 1 GiB
    assert -(-200_000 // 7235) == 28
    # the same events as P12: 111 300 B each -> 9647 fit; 1855*40 = 8 * 9275 -> multiples of 4
    assert (1 << 30) // 111_300 == 9647
    assert ce(200_000, 1855, 40, 1 << 30, 12) == 9644
    for (P, S) in [(1855, 40), (1855, 30), (1764, 25), (2048, 128), (3, 5), (1, 1), (7, 32)]:
        import math
        m = 32 // math.gcd(P * S, 32)
        for bits in (16, 12):
            ev_bits = P * S * bits
            for cb in (1, 100, ev_bits // 8, 10 * ev_bits // 8 + 5, 1 << 20, 1 << 30):
                for E in (0, 1, 5, 1000, 200_000):
                    got = ce(E, P, S, cb, bits)
                    fit = (8 * cb) // ev_bits
                    if bits == 12:
                        fit -= fit % m
                        fit = max(fit, m)
                    want = max(1, min(max(fit, 1), E)) if E > 0 else 1
                    assert got == want, (P, S, bits, cb, E, got, want)
                    if bits == 12 and got < E:                       # every later chunk starts aligned
                        assert (got * ev_bits) % 128 == 0
    assert ce(-1, 4, 30, 0, 16) == -1 and ce(1, 4, 30, 0, 8) == -1 and ce(1, 0, 30, 0, 12) == -1


# ---- mixed-camera (ragged) plans: validation is pure host logic ----------------
def _plan_status(tp, ts, tw, tc, bt, bw, bo):
    L = rta.lib()
    a32 = lambda v: (ctypes.c_int32 * max(1, len(v)))(*v)
    a64 = lambda v: (ctypes.c_int64 * max(1, len(v)))(*v)
    plan = ctypes.c_void_p()
    rc = L.rta_ragged_plan_create(len(tp), ctypes.cast(a32(tp), ctypes.c_void_p), ctypes.cast(a32(ts), ctypes.c_void_p),
                                  ctypes.cast(a32(tw), ctypes.c_void_p), ctypes.cast(a64(tc), ctypes.c_void_p),
                                  len(bt), ctypes.cast(a32(bt), ctypes.c_void_p), ctypes.cast(a64(bw), ctypes.c_void_p),
                                  ctypes.cast(a64(bo), ctypes.c_void_p), ctypes.byref(plan))
    if rc == rta.RTA_OK:
        L.rta_ragged_plan_destroy(plan)
    else:
        assert plan.value is None
    return rc


def test_ragged_plan_validation_before_any_cuda_call():
    ok = ([4], [30], [7], [0])
    assert _plan_status(*ok, [], [], []) == rta.RTA_OK                       # empty plan, no device needed
    assert _plan_status([0], [30], [7], [0], [], [], []) == rta.RTA_ERR_SHAPE
    assert _plan_status([4], [30], [31], [0], [], [], []) == rta.RTA_ERR_SHAPE   # W > S
    assert _plan_status([4], [30], [0], [0], [], [], []) == rta.RTA_ERR_SHAPE
    assert _plan_status([4], [30], [7], [-1], [], [], []) == rta.RTA_ERR_SHAPE
    assert _plan_status([4], [2048], [17], [0], [], [], []) == rta.RTA_ERR_UNSUPPORTED
    assert _plan_status(*ok, [1], [0], [0]) == rta.RTA_ERR_SHAPE              # telescope index out of range
    assert _plan_status(*ok, [-1], [0], [0]) == rta.RTA_ERR_SHAPE
    assert _plan_status(*ok, [0], [-2], [0]) == rta.RTA_ERR_SHAPE
    assert _plan_status(*ok, [0], [0], [-2]) == rta.RTA_ERR_SHAPE
    assert _plan_status(*ok, [0], [0], [2 ** 31 - 2]) == rta.RTA_ERR_UNSUPPORTED
    assert _plan_status(*ok, [0], [2 ** 47], [0]) == rta.RTA_ERR_UNSUPPORTED
    L = rta.lib()
    assert L.rta_ragged_plan_create(0, None, None, None, None, 0, None, None, None, None) == rta.RTA_ERR_NULL
    assert L.rta_extract_ragged(None, 0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000, 0x7000, 0) == rta.RTA_ERR_NULL
    assert L.rta_ragged_plan_info(None, 0) == -1
    L.rta_ragged_plan_destroy(None)
    # an empty plan extracts to RTA_OK with null pointers and launches nothing
    plan = rta.rta_ragged_plan_create([4], [30], [7], [0], [], [], [])
    before = rta.rta_launch_count()
    assert L.rta_extract_ragged(plan, None, None, None, None, None, None, None, 0) == rta.RTA_OK
    assert rta.rta_launch_count() == before
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_TILES) == 0
    assert rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_LAUNCHES) == 0
    assert rta.rta_ragged_plan_info(plan, 99) == -1
    rta.rta_ragged_plan_destroy(plan)


def test_prepare_validates_before_any_cuda_call():
    """include/rta.h:rta_prepare: argument errors and the ahead-of-time shapes are decided
    on the host; only a shape that needs compiling reaches CUDA (and fails here, without a
    device, as every compute call does)."""
    L = rta.lib()
    assert L.rta_prepare(0, 1, rta.RTA_EXTRACTOR_SLIDING, 16) == rta.RTA_ERR_SHAPE
    assert L.rta_prepare(30, 31, rta.RTA_EXTRACTOR_SLIDING, 16) == rta.RTA_ERR_SHAPE
    assert L.rta_prepare(30, 7, 4, 16) == rta.RTA_ERR_SHAPE          # no such extractor
    assert L.rta_prepare(30, 7, -1, 16) == rta.RTA_ERR_SHAPE
    assert L.rta_prepare(30, 7, rta.RTA_EXTRACTOR_SLIDING, 8) == rta.RTA_ERR_SHAPE
    assert L.rta_prepare(2048, 17, rta.RTA_EXTRACTOR_SLIDING, 16) == rta.RTA_ERR_UNSUPPORTED
    assert L.rta_prepare(36, 5, rta.RTA_EXTRACTOR_FIXED, 12) == rta.RTA_ERR_UNSUPPORTED
    assert L.rta_prepare(64, 33, rta.RTA_EXTRACTOR_FIR, 16) == rta.RTA_ERR_UNSUPPORTED
    for S, W in ((30, 7), (40, 7), (25, 4), (128, 8)):               # built with the library
        for bits in (16, 12):
            assert L.rta_prepare(S, W, rta.RTA_EXTRACTOR_SLIDING, bits) == rta.RTA_OK
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if not has_gpu:
        assert L.rta_prepare(36, 5, rta.RTA_EXTRACTOR_SLIDING, 16) in (
            rta.RTA_ERR_CUDA, rta.RTA_ERR_NOMEM, rta.RTA_ERR_UNSUPPORTED)
