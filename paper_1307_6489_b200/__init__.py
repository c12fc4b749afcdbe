"""paper_1307_6489_b200 — thin Python binding of librta.so (include/rta.h).

Argument marshalling only: every step of the extraction runs in the CUDA
kernels of ``csrc/``. PyTorch is used by callers for device memory and streams;
this module only turns tensors into raw pointers for the C ABI. There is no CPU
fallback — if the library cannot be built or loaded, importing the entry points
raises.
"""
from __future__ import annotations

import ctypes
import os
import threading

RTA_OK = 0
RTA_ERR_NULL = 1
RTA_ERR_SHAPE = 2
RTA_ERR_UNSUPPORTED = 3
RTA_ERR_ALIGN = 4
RTA_ERR_CUDA = 5
RTA_ERR_NOMEM = 6
RTA_ERR_TOO_LARGE = 7
RTA_NOALLOC_MAX_TRACES = 1 << 20   # include/rta.h

_HERE = os.path.dirname(os.path.abspath(__file__))
_lock = threading.Lock()
_lib = None
_test_lib = None
_hooks_on: set = set()     # names of the rta_debug_* switches that are on (tests only)

_VP = ctypes.c_void_p
_EXTRACT_ARGS = [_VP, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, _VP, _VP,
                 ctypes.c_int32, _VP, _VP, _VP, _VP]


class RtaError(RuntimeError):
    def __init__(self, status: int, message: str, cuda_error: int = 0):
        super().__init__("rta: %s (status %d, cudaError %d)" % (message, status, cuda_error))
        self.status = status
        self.cuda_error = cuda_error


def _declare(L: ctypes.CDLL, testing: bool) -> ctypes.CDLL:
    for name in ("rta_extract",) + (("rta_extract_generic",) if testing else ()):
        fn = getattr(L, name)
        fn.restype = ctypes.c_int
        fn.argtypes = _EXTRACT_ARGS + [_VP]
    L.rta_extract_stream.restype = ctypes.c_int
    L.rta_extract_stream.argtypes = _EXTRACT_ARGS + [ctypes.c_size_t, _VP]
    L.rta_extract_host.restype = ctypes.c_int
    L.rta_extract_host.argtypes = _EXTRACT_ARGS + [ctypes.c_size_t]
    L.rta_extract_packed12.restype = ctypes.c_int
    L.rta_extract_packed12.argtypes = _EXTRACT_ARGS + [_VP]
    L.rta_extract_stream_packed12.restype = ctypes.c_int
    L.rta_extract_stream_packed12.argtypes = _EXTRACT_ARGS + [ctypes.c_size_t, _VP]
    L.rta_extract_host_packed12.restype = ctypes.c_int
    L.rta_extract_host_packed12.argtypes = _EXTRACT_ARGS + [ctypes.c_size_t]
    L.rta_kernel_name_packed12.restype = ctypes.c_char_p
    L.rta_kernel_name_packed12.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int]
    L.rta_extract_fixed.restype = ctypes.c_int
    L.rta_extract_fixed.argtypes = _EXTRACT_ARGS[:7] + [_VP] + [_VP] * 4 + [_VP]
    L.rta_extract_local_peak.restype = ctypes.c_int
    L.rta_extract_local_peak.argtypes = _EXTRACT_ARGS[:7] + [ctypes.c_int32] + [_VP] * 4 + [_VP]
    L.rta_extract_fir.restype = ctypes.c_int
    L.rta_extract_fir.argtypes = _EXTRACT_ARGS[:6] + [_VP, ctypes.c_int32] + [_VP] * 4 + [_VP]
    L.rta_strerror.restype = ctypes.c_char_p
    L.rta_strerror.argtypes = [ctypes.c_int]
    L.rta_last_cuda_error.restype = ctypes.c_int
    L.rta_last_cuda_error.argtypes = []
    L.rta_kernel_name.restype = ctypes.c_char_p
    L.rta_kernel_name.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int]
    L.rta_ragged_plan_create.restype = ctypes.c_int
    L.rta_ragged_plan_create.argtypes = ([ctypes.c_int32] + [_VP] * 4 + [ctypes.c_int64]
                                         + [_VP] * 3 + [ctypes.POINTER(_VP)])
    L.rta_extract_ragged.restype = ctypes.c_int
    L.rta_extract_ragged.argtypes = [_VP] * 9
    L.rta_ragged_plan_info.restype = ctypes.c_int64
    L.rta_ragged_plan_info.argtypes = [_VP, ctypes.c_int32]
    L.rta_ragged_plan_destroy.restype = None
    L.rta_ragged_plan_destroy.argtypes = [_VP]
    _CAM = [_VP, _VP, _VP, ctypes.c_float, ctypes.c_float]
    _IMG_OUT = [_VP, _VP, _VP]
    L.rta_image_moments.restype = ctypes.c_int
    L.rta_image_moments.argtypes = ([_VP, _VP, ctypes.c_int64, ctypes.c_int32] + _CAM
                                    + _IMG_OUT + [_VP])
    for name in ("rta_extract_image", "rta_extract_image_noalloc") + (
            ("rta_extract_image_generic",) if testing else ()):
        fn = getattr(L, name)
        fn.restype = ctypes.c_int
        fn.argtypes = _EXTRACT_ARGS[:7] + _CAM + _IMG_OUT + [_VP]
    L.rta_extract_image_stream.restype = ctypes.c_int
    L.rta_extract_image_stream.argtypes = (_EXTRACT_ARGS[:7] + _CAM + _IMG_OUT
                                           + [ctypes.c_size_t, _VP])
    L.rta_extract_image_host.restype = ctypes.c_int
    L.rta_extract_image_host.argtypes = (_EXTRACT_ARGS[:7] + _CAM + _IMG_OUT
                                         + [ctypes.c_size_t])
    L.rta_image_kernel_name.restype = ctypes.c_char_p
    L.rta_image_kernel_name.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                        ctypes.c_int]
    L.rta_image_max_pixels.restype = ctypes.c_int32
    L.rta_image_max_pixels.argtypes = []
    L.rta_prepare.restype = ctypes.c_int
    L.rta_prepare.argtypes = [ctypes.c_int32] * 4
    L.rta_chunk_events.restype = ctypes.c_int64
    L.rta_chunk_events.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32,
                                   ctypes.c_size_t, ctypes.c_int32]
    L.rta_launch_count.restype = ctypes.c_uint64
    L.rta_launch_count.argtypes = []
    L.rta_shutdown.restype = None
    L.rta_shutdown.argtypes = []
    if testing:
        for name in ("rta_debug_force_generic", "rta_debug_static_schedule",
                     "rta_debug_serial_ragged", "rta_debug_general_cleaning", "rta_debug_jit",
                     "rta_debug_lanes_per_trace"):
            fn = getattr(L, name)
            fn.restype = None
            fn.argtypes = [ctypes.c_int]
        L.rta_debug_seg_tuning.restype = None
        L.rta_debug_seg_tuning.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    return L


def _load(testing: bool) -> ctypes.CDLL:
    from . import build as _build
    # RTA_LIBRARY: load a prebuilt library (a -DRTA_TESTING build serves both roles)
    # instead of building in-tree
    path = os.environ.get("RTA_LIBRARY")
    if not path:
        path = _build.build()
        if testing:
            path = _build.TEST_LIB
    if not os.path.exists(path):
        raise ImportError("%s is missing and could not be built" % path)
    return _declare(ctypes.CDLL(path), testing)


def lib() -> ctypes.CDLL:
    """Load (building in-tree if stale) librta.so and declare its symbols: the
    ABI of include/rta.h, nothing else. While a test hook is switched on (see
    :func:`testing_lib`) every call is routed to librta_testing.so instead."""
    global _lib
    if _hooks_on:
        return testing_lib()
    with _lock:
        if _lib is None:
            _lib = _load(False)
    return _lib


def testing_lib() -> ctypes.CDLL:
    """librta_testing.so: the same sources built with -DRTA_TESTING, which adds
    the entry points the tests need and the shipped library does not export
    (rta_extract_generic, rta_extract_image_generic, rta_debug_*). The two
    libraries share no state."""
    global _test_lib
    with _lock:
        if _test_lib is None:
            _test_lib = _load(True)
    return _test_lib


def _ptr(x) -> int | None:
    """torch tensor / numpy array / int / None -> raw address."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError("expected a tensor, an array, an int address or None")


def _check(status: int) -> None:
    if status != RTA_OK:
        L = lib()
        raise RtaError(status, L.rta_strerror(status).decode(), L.rta_last_cuda_error())


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def rta_extract(wf, n_events, n_pixels, n_samples, pedestal, gain, W,
                out_sum, out_start, out_charge, out_time, stream=None, *,
                generic: bool = False) -> None:
    """include/rta.h:rta_extract. Device pointers (tensors or addresses);
    asynchronous on ``stream`` (default: torch's current stream)."""
    fn = testing_lib().rta_extract_generic if generic else lib().rta_extract
    _check(fn(_ptr(wf), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
              _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
              _stream_handle(stream)))


def rta_extract_fixed(wf, n_events, n_pixels, n_samples, pedestal, gain, W, window_start,
                      out_sum, out_start, out_charge, out_time, stream=None) -> None:
    """include/rta.h:rta_extract_fixed. ``window_start`` is a device int32 [n_pixels]."""
    _check(lib().rta_extract_fixed(
        _ptr(wf), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
        _ptr(window_start), _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
        _stream_handle(stream)))


def rta_extract_local_peak(wf, n_events, n_pixels, n_samples, pedestal, gain, W, shift,
                           out_sum, out_start, out_charge, out_time, stream=None) -> None:
    """include/rta.h:rta_extract_local_peak."""
    _check(lib().rta_extract_local_peak(
        _ptr(wf), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W, int(shift),
        _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
        _stream_handle(stream)))


def rta_extract_fir(wf, n_events, n_pixels, n_samples, pedestal, gain, taps,
                    out_sum, out_start, out_charge, out_time, stream=None) -> None:
    """include/rta.h:rta_extract_fir. ``taps`` is a host sequence of ints."""
    taps = [int(t) for t in taps]
    arr = (ctypes.c_int32 * max(1, len(taps)))(*taps)
    _check(lib().rta_extract_fir(
        _ptr(wf), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain),
        ctypes.cast(arr, _VP) if taps else None, len(taps),
        _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
        _stream_handle(stream)))


def rta_extract_stream(wf_host, n_events, n_pixels, n_samples, pedestal, gain, W,
                       out_sum, out_start, out_charge, out_time, chunk_bytes=0,
                       stream=None) -> None:
    """include/rta.h:rta_extract_stream. ``wf_host`` is host memory; the rest
    are device pointers. Outputs valid after ``stream`` is synchronised."""
    _check(lib().rta_extract_stream(
        _ptr(wf_host), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
        _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
        int(chunk_bytes), _stream_handle(stream)))


def rta_extract_host(wf_host, n_events, n_pixels, n_samples, pedestal_host, gain_host,
                     W, out_sum_host, out_start_host, out_charge_host, out_time_host,
                     chunk_bytes=0) -> None:
    """include/rta.h:rta_extract_host. Every pointer is host memory;
    synchronous."""
    _check(lib().rta_extract_host(
        _ptr(wf_host), n_events, n_pixels, n_samples, _ptr(pedestal_host),
        _ptr(gain_host), W, _ptr(out_sum_host), _ptr(out_start_host),
        _ptr(out_charge_host), _ptr(out_time_host), int(chunk_bytes)))


def rta_extract_packed12(packed, n_events, n_pixels, n_samples, pedestal, gain, W,
                         out_sum, out_start, out_charge, out_time, stream=None) -> None:
    """include/rta.h:rta_extract_packed12. ``packed`` is a device P12 byte stream."""
    _check(lib().rta_extract_packed12(
        _ptr(packed), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
        _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
        _stream_handle(stream)))


def rta_extract_stream_packed12(packed_host, n_events, n_pixels, n_samples, pedestal, gain, W,
                                out_sum, out_start, out_charge, out_time, chunk_bytes=0,
                                stream=None) -> None:
    """include/rta.h:rta_extract_stream_packed12. ``packed_host`` is a host P12
    byte stream; calibration and outputs are device pointers."""
    _check(lib().rta_extract_stream_packed12(
        _ptr(packed_host), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
        _ptr(out_sum), _ptr(out_start), _ptr(out_charge), _ptr(out_time),
        int(chunk_bytes), _stream_handle(stream)))


def rta_extract_host_packed12(packed_host, n_events, n_pixels, n_samples, pedestal_host,
                              gain_host, W, out_sum_host, out_start_host, out_charge_host,
                              out_time_host, chunk_bytes=0) -> None:
    """include/rta.h:rta_extract_host_packed12. Every pointer is host memory; synchronous."""
    _check(lib().rta_extract_host_packed12(
        _ptr(packed_host), n_events, n_pixels, n_samples, _ptr(pedestal_host),
        _ptr(gain_host), W, _ptr(out_sum_host), _ptr(out_start_host),
        _ptr(out_charge_host), _ptr(out_time_host), int(chunk_bytes)))


RTA_RAGGED_N_LAUNCHES = 0
RTA_RAGGED_N_TILES = 1
RTA_RAGGED_N_TRACES = 2
RTA_RAGGED_WF_BYTES = 3
RTA_RAGGED_WF_END_BYTES = 4
RTA_RAGGED_OUT_END = 5


def _host_array(seq, ctype):
    seq = [int(v) for v in seq]
    return (ctype * max(1, len(seq)))(*seq), len(seq)


def rta_ragged_plan_create(tel_n_pixels, tel_n_samples, tel_W, tel_calib_offset,
                           blk_tel, blk_wf_offset, blk_out_offset) -> int:
    """include/rta.h:rta_ragged_plan_create. The tables are host sequences of
    ints; returns the opaque plan handle (an address)."""
    tp, n_tel = _host_array(tel_n_pixels, ctypes.c_int32)
    ts, n1 = _host_array(tel_n_samples, ctypes.c_int32)
    tw, n2 = _host_array(tel_W, ctypes.c_int32)
    tc, n3 = _host_array(tel_calib_offset, ctypes.c_int64)
    bt, n_blk = _host_array(blk_tel, ctypes.c_int32)
    bw, m1 = _host_array(blk_wf_offset, ctypes.c_int64)
    bo, m2 = _host_array(blk_out_offset, ctypes.c_int64)
    if not (n_tel == n1 == n2 == n3 and n_blk == m1 == m2):
        raise ValueError("table lengths differ")
    plan = _VP()
    _check(lib().rta_ragged_plan_create(
        n_tel, ctypes.cast(tp, _VP), ctypes.cast(ts, _VP), ctypes.cast(tw, _VP),
        ctypes.cast(tc, _VP), n_blk, ctypes.cast(bt, _VP), ctypes.cast(bw, _VP),
        ctypes.cast(bo, _VP), ctypes.byref(plan)))
    return plan.value


def rta_extract_ragged(plan, wf, pedestal, gain, out_sum, out_start, out_charge, out_time,
                       stream=None) -> None:
    """include/rta.h:rta_extract_ragged. Device pointers; asynchronous on ``stream``."""
    _check(lib().rta_extract_ragged(
        plan, _ptr(wf), _ptr(pedestal), _ptr(gain), _ptr(out_sum), _ptr(out_start),
        _ptr(out_charge), _ptr(out_time), _stream_handle(stream)))


def rta_ragged_plan_info(plan, what: int) -> int:
    return int(lib().rta_ragged_plan_info(plan, int(what)))


def rta_ragged_plan_destroy(plan) -> None:
    lib().rta_ragged_plan_destroy(plan)


def rta_image_moments(charge, time, n_events, n_pixels, pix_x, pix_y, neighbors, thr_picture,
                      thr_boundary, out_n_pix, out_params, out_mask=None, stream=None) -> None:
    """include/rta.h:rta_image_moments. Device pointers; asynchronous on ``stream``."""
    _check(lib().rta_image_moments(
        _ptr(charge), _ptr(time), n_events, n_pixels, _ptr(pix_x), _ptr(pix_y), _ptr(neighbors),
        float(thr_picture), float(thr_boundary), _ptr(out_n_pix), _ptr(out_params),
        _ptr(out_mask), _stream_handle(stream)))


def rta_extract_image(wf, n_events, n_pixels, n_samples, pedestal, gain, W, pix_x, pix_y,
                      neighbors, thr_picture, thr_boundary, out_n_pix, out_params,
                      out_mask=None, stream=None, *, generic: bool = False) -> None:
    """include/rta.h:rta_extract_image. Device pointers; asynchronous on ``stream``."""
    fn = testing_lib().rta_extract_image_generic if generic else lib().rta_extract_image
    _check(fn(_ptr(wf), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
              _ptr(pix_x), _ptr(pix_y), _ptr(neighbors), float(thr_picture),
              float(thr_boundary), _ptr(out_n_pix), _ptr(out_params), _ptr(out_mask),
              _stream_handle(stream)))


def rta_extract_image_noalloc(wf, n_events, n_pixels, n_samples, pedestal, gain, W, pix_x, pix_y,
                              neighbors, thr_picture, thr_boundary, out_n_pix, out_params,
                              out_mask=None, stream=None) -> None:
    """include/rta.h:rta_extract_image_noalloc: rta_extract_image for callers that must
    not allocate device memory (fixed scratch inside the library, at most
    RTA_NOALLOC_MAX_TRACES traces per call, calls that overlap on the GPU race).
    Device pointers; asynchronous on ``stream``."""
    _check(lib().rta_extract_image_noalloc(
        _ptr(wf), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
        _ptr(pix_x), _ptr(pix_y), _ptr(neighbors), float(thr_picture), float(thr_boundary),
        _ptr(out_n_pix), _ptr(out_params), _ptr(out_mask), _stream_handle(stream)))


def rta_extract_image_stream(wf_host, n_events, n_pixels, n_samples, pedestal, gain, W, pix_x,
                             pix_y, neighbors, thr_picture, thr_boundary, out_n_pix, out_params,
                             out_mask=None, chunk_bytes=0, stream=None) -> None:
    """include/rta.h:rta_extract_image_stream. ``wf_host`` is host memory; the
    rest are device pointers."""
    _check(lib().rta_extract_image_stream(
        _ptr(wf_host), n_events, n_pixels, n_samples, _ptr(pedestal), _ptr(gain), W,
        _ptr(pix_x), _ptr(pix_y), _ptr(neighbors), float(thr_picture), float(thr_boundary),
        _ptr(out_n_pix), _ptr(out_params), _ptr(out_mask), int(chunk_bytes),
        _stream_handle(stream)))


def rta_extract_image_host(wf_host, n_events, n_pixels, n_samples, pedestal_host, gain_host, W,
                           pix_x_host, pix_y_host, neighbors_host, thr_picture, thr_boundary,
                           out_n_pix_host, out_params_host, out_mask_host=None,
                           chunk_bytes=0) -> None:
    """include/rta.h:rta_extract_image_host. Every pointer is host memory; synchronous."""
    _check(lib().rta_extract_image_host(
        _ptr(wf_host), n_events, n_pixels, n_samples, _ptr(pedestal_host), _ptr(gain_host), W,
        _ptr(pix_x_host), _ptr(pix_y_host), _ptr(neighbors_host), float(thr_picture),
        float(thr_boundary), _ptr(out_n_pix_host), _ptr(out_params_host), _ptr(out_mask_host),
        int(chunk_bytes)))


def rta_image_kernel_name(n_pixels: int, n_samples: int, W: int, aligned16: bool = True) -> str:
    return lib().rta_image_kernel_name(n_pixels, n_samples, W, 1 if aligned16 else 0).decode()


def rta_image_max_pixels() -> int:
    return int(lib().rta_image_max_pixels())


RTA_EXTRACTOR_SLIDING, RTA_EXTRACTOR_FIXED, RTA_EXTRACTOR_LOCAL_PEAK, RTA_EXTRACTOR_FIR = 0, 1, 2, 3


def rta_prepare(n_samples: int, W: int, extractor: int = RTA_EXTRACTOR_SLIDING,
                sample_bits: int = 16) -> bool:
    """include/rta.h:rta_prepare. True: a kernel specialised for the shape is ready on the
    current device (nothing will be compiled on the data path); False: the shape has no
    specialisation and runs the runtime-shape kernels. Other statuses raise."""
    st = lib().rta_prepare(n_samples, W, extractor, sample_bits)
    if st == RTA_ERR_UNSUPPORTED:
        return False
    _check(st)
    return True


def rta_strerror(status: int) -> str:
    return lib().rta_strerror(status).decode()


def rta_last_cuda_error() -> int:
    return lib().rta_last_cuda_error()


def rta_kernel_name(n_samples: int, W: int, aligned16: bool = True) -> str:
    return lib().rta_kernel_name(n_samples, W, 1 if aligned16 else 0).decode()


def rta_kernel_name_packed12(n_samples: int, W: int, aligned16: bool = True) -> str:
    return lib().rta_kernel_name_packed12(n_samples, W, 1 if aligned16 else 0).decode()


def rta_chunk_events(n_events: int, n_pixels: int, n_samples: int, chunk_bytes: int = 0,
                     sample_bits: int = 16) -> int:
    """include/rta.h:rta_chunk_events."""
    return int(lib().rta_chunk_events(n_events, n_pixels, n_samples, int(chunk_bytes), sample_bits))


def rta_launch_count() -> int:
    return int(lib().rta_launch_count())


def rta_shutdown() -> None:
    lib().rta_shutdown()


def _hook(name: str, on: bool) -> None:
    getattr(testing_lib(), name)(1 if on else 0)
    (_hooks_on.add if on else _hooks_on.discard)(name)


def rta_debug_force_generic(on: bool) -> None:
    """Test hook (librta_testing.so): route rta_extract_fixed/_local_peak/_fir/_packed12
    to the generic kernel."""
    _hook("rta_debug_force_generic", on)


def rta_debug_static_schedule(on: bool) -> None:
    """Test hook (librta_testing.so): force the static round-robin tile schedule of the
    staged kernels (default is dynamic). Results are identical either way."""
    _hook("rta_debug_static_schedule", on)


def rta_debug_serial_ragged(on: bool) -> None:
    """Test hook (librta_testing.so): rta_extract_ragged issues its launches one after
    the other on the caller's stream instead of forking side streams. Same results."""
    _hook("rta_debug_serial_ragged", on)


def rta_debug_general_cleaning(on: bool) -> None:
    """Test hook (librta_testing.so): the image cleaning runs the two steps of its
    definition even when the neighbour table is symmetric (same masks either way)."""
    _hook("rta_debug_general_cleaning", on)


def rta_debug_jit(on: bool) -> None:
    """Test hook (librta_testing.so): False = no run-time (NVRTC) specialisations, so that
    unspecialised shapes take the runtime-shape kernel, as without libnvrtc; True = default."""
    testing_lib().rta_debug_jit(1 if on else 0)
    (_hooks_on.discard if on else _hooks_on.add)("rta_debug_jit")


def rta_debug_lanes_per_trace(lpt: int) -> None:
    """Test / measurement hook (librta_testing.so): 4, 8, 16 or 32 = rta_extract runs the
    several-lanes-per-trace kernel with that many lanes wherever it can; 0 = normal dispatch."""
    testing_lib().rta_debug_lanes_per_trace(int(lpt))
    (_hooks_on.add if lpt else _hooks_on.discard)("rta_debug_lanes_per_trace")


def rta_debug_seg_tuning(L: int = 0, TR: int = 0, NT: int = 0, stages: int = 0) -> None:
    """Test / measurement hook (librta_testing.so): window starts per segment (2 * odd), traces
    per tile, threads per CTA and ring stages of the segment kernel (0 = chosen per shape). A non-zero L
    sends every sliding rta_extract on a 16-byte-aligned base to that kernel."""
    testing_lib().rta_debug_seg_tuning(int(L), int(TR), int(NT), int(stages))
    (_hooks_on.add if (L or TR or NT or stages) else _hooks_on.discard)("rta_debug_seg_tuning")


def shard_events(n_events: int, world_size: int, rank: int) -> tuple[int, int]:
    """Contiguous event range [first, first+count) of ``rank`` when a batch is
    split over ``world_size`` independent GPUs (traces are
    independent, so there is no exchange step and no collective)."""
    if world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad rank/world_size")
    first = n_events * rank // world_size
    last = n_events * (rank + 1) // world_size
    return first, last - first
