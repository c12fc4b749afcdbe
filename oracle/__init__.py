"""oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes loader for ``oracle/rta_oracle.cpp``: the plain single-threaded C++
definition of sliding-window signal extraction (BASELINE.json:north_star
sentence 2; §5 names the step, nothing more).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package. It never
imports ``paper_1307_6489_b200`` and shares no code with it. numpy arrays in,
numpy arrays out; no torch, no CUDA.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rta_oracle.cpp")
_SRCS = [_SRC, os.path.join(_HERE, "rta_oracle_windows.cpp"),
         os.path.join(_HERE, "rta_oracle_packed.cpp"),
         os.path.join(_HERE, "rta_oracle_ragged.cpp"),
         os.path.join(_HERE, "rta_oracle_image.cpp")]
# RTA_ORACLE_SANITIZE=1: an instrumented build (-fsanitize=address,undefined) beside
# the plain one, for a memory-safety pass of the CPU tests:
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
#   RTA_ORACLE_SANITIZE=1 python -m pytest tests -q -m "not gpu"
_SANITIZE = os.environ.get("RTA_ORACLE_SANITIZE", "") not in ("", "0")
_LIB = os.path.join(_HERE, "librta_oracle_san.so" if _SANITIZE else "librta_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (single-threaded, no fast-math)."""
    with _lock:
        stale = (not os.path.exists(_LIB)
                 or any(os.path.getmtime(_LIB) < os.path.getmtime(f) for f in _SRCS))
        if force or stale:
            tmp = _LIB + ".tmp%d" % os.getpid()
            san = (["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"]
                   if _SANITIZE else [])
            subprocess.check_call(
                ["g++", "-std=c++17", "-O2", "-fPIC", "-shared",
                 "-ffp-contract=off"] + san + ["-o", tmp] + _SRCS)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.rta_oracle_extract.restype = ctypes.c_int
        lib.rta_oracle_extract.argtypes = [
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        common = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32,
                  ctypes.c_void_p, ctypes.c_void_p]
        outs = [ctypes.c_void_p] * 4
        lib.rta_oracle_extract_fixed.restype = ctypes.c_int
        lib.rta_oracle_extract_fixed.argtypes = common + [ctypes.c_int32, ctypes.c_void_p] + outs
        lib.rta_oracle_extract_local_peak.restype = ctypes.c_int
        lib.rta_oracle_extract_local_peak.argtypes = common + [ctypes.c_int32, ctypes.c_int32] + outs
        lib.rta_oracle_extract_fir.restype = ctypes.c_int
        lib.rta_oracle_extract_fir.argtypes = common + [ctypes.c_void_p, ctypes.c_int32] + outs
        lib.rta_oracle_unpack12.restype = ctypes.c_int
        lib.rta_oracle_unpack12.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p]
        lib.rta_oracle_extract_packed12.restype = ctypes.c_int
        lib.rta_oracle_extract_packed12.argtypes = lib.rta_oracle_extract.argtypes
        lib.rta_oracle_extract_ragged.restype = ctypes.c_int
        lib.rta_oracle_extract_ragged.argtypes = (
            [ctypes.c_void_p, ctypes.c_int32] + [ctypes.c_void_p] * 4 + [ctypes.c_int64]
            + [ctypes.c_void_p] * 3 + [ctypes.c_void_p] * 2 + [ctypes.c_void_p] * 4)
        lib.rta_oracle_image_moments.restype = ctypes.c_int
        lib.rta_oracle_image_moments.argtypes = (
            [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32] + [ctypes.c_void_p] * 3
            + [ctypes.c_float, ctypes.c_float] + [ctypes.c_void_p] * 3)
        _lib = lib
    return _lib


def _prep(wf, pedestal, gain):
    wf = np.ascontiguousarray(wf, dtype=np.uint16)
    if wf.ndim != 3:
        raise ValueError("wf must be [n_events][n_pixels][n_samples]")
    E, P, S = wf.shape
    pedestal = np.ascontiguousarray(pedestal, dtype=np.int32)
    gain = np.ascontiguousarray(gain, dtype=np.float32)
    if pedestal.shape != (P,) or gain.shape != (P,):
        raise ValueError("pedestal and gain must be [n_pixels]")
    n = E * P
    outs = (np.empty(n, np.int32), np.empty(n, np.int32), np.empty(n, np.float32),
            np.empty(n, np.float32))
    return wf, pedestal, gain, outs


def extract_fixed(wf, pedestal, gain, W: int, window_start):
    """Fixed-window extractor (rta_oracle_windows.cpp, reading R22)."""
    wf, pedestal, gain, outs = _prep(wf, pedestal, gain)
    E, P, S = wf.shape
    ws = np.ascontiguousarray(window_start, dtype=np.int32)
    if ws.shape != (P,):
        raise ValueError("window_start must be [n_pixels]")
    rc = _load().rta_oracle_extract_fixed(
        wf.ctypes.data, E, P, S, pedestal.ctypes.data, gain.ctypes.data, int(W), ws.ctypes.data,
        *[o.ctypes.data for o in outs])
    if rc != 0:
        raise ValueError("rta_oracle_extract_fixed: bad shape")
    return outs


def extract_local_peak(wf, pedestal, gain, W: int, shift: int):
    """Local-peak extractor (rta_oracle_windows.cpp, reading R23)."""
    wf, pedestal, gain, outs = _prep(wf, pedestal, gain)
    E, P, S = wf.shape
    rc = _load().rta_oracle_extract_local_peak(
        wf.ctypes.data, E, P, S, pedestal.ctypes.data, gain.ctypes.data, int(W), int(shift),
        *[o.ctypes.data for o in outs])
    if rc != 0:
        raise ValueError("rta_oracle_extract_local_peak: bad shape")
    return outs


def extract_fir(wf, pedestal, gain, taps):
    """FIR / matched-filter extractor (rta_oracle_windows.cpp, reading R24)."""
    wf, pedestal, gain, outs = _prep(wf, pedestal, gain)
    E, P, S = wf.shape
    taps = np.ascontiguousarray(taps, dtype=np.int32)
    if taps.ndim != 1:
        raise ValueError("taps must be 1-D")
    rc = _load().rta_oracle_extract_fir(
        wf.ctypes.data, E, P, S, pedestal.ctypes.data, gain.ctypes.data, taps.ctypes.data,
        int(taps.size), *[o.ctypes.data for o in outs])
    if rc != 0:
        raise ValueError("rta_oracle_extract_fir: bad shape")
    return outs


def extract(wf: np.ndarray, pedestal: np.ndarray, gain: np.ndarray, W: int):
    """Run the oracle on ``wf[E][P][S]`` (uint16).

    Returns ``(out_sum int32[E*P], out_start int32[E*P], out_charge
    float32[E*P], out_time float32[E*P])``.
    """
    wf = np.ascontiguousarray(wf, dtype=np.uint16)
    if wf.ndim != 3:
        raise ValueError("wf must be [n_events][n_pixels][n_samples]")
    E, P, S = wf.shape
    pedestal = np.ascontiguousarray(pedestal, dtype=np.int32)
    gain = np.ascontiguousarray(gain, dtype=np.float32)
    if pedestal.shape != (P,) or gain.shape != (P,):
        raise ValueError("pedestal and gain must be [n_pixels]")
    n = E * P
    out_sum = np.empty(n, np.int32)
    out_start = np.empty(n, np.int32)
    out_charge = np.empty(n, np.float32)
    out_time = np.empty(n, np.float32)
    rc = _load().rta_oracle_extract(
        wf.ctypes.data, E, P, S, pedestal.ctypes.data, gain.ctypes.data, int(W),
        out_sum.ctypes.data, out_start.ctypes.data, out_charge.ctypes.data,
        out_time.ctypes.data)
    if rc != 0:
        raise ValueError("rta_oracle_extract: bad shape (S=%d, W=%d)" % (S, W))
    return out_sum, out_start, out_charge, out_time


def packed12_nbytes(n_total: int) -> int:
    """Bytes of a P12 stream holding ``n_total`` samples: ceil(12 n / 8)."""
    return (12 * int(n_total) + 7) // 8


def unpack12(packed, n_total: int) -> np.ndarray:
    """Decode ``n_total`` samples of a P12 stream (rta_oracle_packed.cpp, readings R25-R27)."""
    packed = np.ascontiguousarray(packed, dtype=np.uint8).ravel()
    if packed.size < packed12_nbytes(n_total):
        raise ValueError("P12 stream too short: %d bytes for %d samples" % (packed.size, n_total))
    out = np.empty(int(n_total), np.uint16)
    if _load().rta_oracle_unpack12(packed.ctypes.data, int(n_total), out.ctypes.data) != 0:
        raise ValueError("rta_oracle_unpack12: bad size")
    return out


def extract_packed12(packed, n_events: int, pedestal, gain, n_samples: int, W: int):
    """Sliding-window extraction of a P12 stream of ``n_events x len(pedestal) x n_samples``."""
    pedestal = np.ascontiguousarray(pedestal, dtype=np.int32)
    gain = np.ascontiguousarray(gain, dtype=np.float32)
    P = pedestal.size
    packed = np.ascontiguousarray(packed, dtype=np.uint8).ravel()
    if packed.size < packed12_nbytes(n_events * P * n_samples):
        raise ValueError("P12 stream too short")
    n = int(n_events) * P
    outs = (np.empty(n, np.int32), np.empty(n, np.int32), np.empty(n, np.float32),
            np.empty(n, np.float32))
    rc = _load().rta_oracle_extract_packed12(
        packed.ctypes.data, int(n_events), P, int(n_samples), pedestal.ctypes.data,
        gain.ctypes.data, int(W), *[o.ctypes.data for o in outs])
    if rc != 0:
        raise ValueError("rta_oracle_extract_packed12: bad shape")
    return outs


def extract_ragged(wf, tel_n_pixels, tel_n_samples, tel_W, tel_calib_offset, blk_tel,
                   blk_wf_offset, blk_out_offset, pedestal, gain, n_out: int, fill=None):
    """Mixed-camera batch (rta_oracle_ragged.cpp, readings R28-R30). ``wf`` is the
    flat uint16 waveform buffer; the tables are sequences. Returns the four flat
    output arrays of length ``n_out``; entries no block writes keep ``fill``
    (default: -1 / -1 / NaN / NaN)."""
    wf = np.ascontiguousarray(wf, dtype=np.uint16).ravel()
    tp = np.ascontiguousarray(tel_n_pixels, dtype=np.int32)
    ts = np.ascontiguousarray(tel_n_samples, dtype=np.int32)
    tw = np.ascontiguousarray(tel_W, dtype=np.int32)
    tc = np.ascontiguousarray(tel_calib_offset, dtype=np.int64)
    bt = np.ascontiguousarray(blk_tel, dtype=np.int32)
    bw = np.ascontiguousarray(blk_wf_offset, dtype=np.int64)
    bo = np.ascontiguousarray(blk_out_offset, dtype=np.int64)
    pedestal = np.ascontiguousarray(pedestal, dtype=np.int32)
    gain = np.ascontiguousarray(gain, dtype=np.float32)
    if not (tp.shape == ts.shape == tw.shape == tc.shape and bt.shape == bw.shape == bo.shape):
        raise ValueError("table lengths differ")
    for b in range(bt.size):                       # bounds (the C function trusts them)
        k = int(bt[b])
        if not 0 <= k < tp.size:
            raise ValueError("block %d: telescope %d out of range" % (b, k))
        if bw[b] < 0 or bw[b] + int(tp[k]) * int(ts[k]) > wf.size:
            raise ValueError("block %d leaves the waveform buffer" % b)
        if bo[b] < 0 or bo[b] + int(tp[k]) > n_out:
            raise ValueError("block %d leaves the output arrays" % b)
        if tc[k] < 0 or tc[k] + int(tp[k]) > pedestal.size or tc[k] + int(tp[k]) > gain.size:
            raise ValueError("telescope %d leaves the calibration arrays" % k)
    f = (-1, -1, np.nan, np.nan) if fill is None else fill
    outs = (np.full(n_out, f[0], np.int32), np.full(n_out, f[1], np.int32),
            np.full(n_out, f[2], np.float32), np.full(n_out, f[3], np.float32))
    rc = _load().rta_oracle_extract_ragged(
        wf.ctypes.data, int(tp.size), tp.ctypes.data, ts.ctypes.data, tw.ctypes.data,
        tc.ctypes.data, int(bt.size), bt.ctypes.data, bw.ctypes.data, bo.ctypes.data,
        pedestal.ctypes.data, gain.ctypes.data, *[o.ctypes.data for o in outs])
    if rc != 0:
        raise ValueError("rta_oracle_extract_ragged: bad table")
    return outs


def image_moments(charge, time, pix_x, pix_y, neighbors, thr_picture: float, thr_boundary: float):
    """Cleaning + image moments per event (rta_oracle_image.cpp, readings R31-R35).
    ``charge``/``time``: float32 [E][P]. Returns (n_pix int32[E], params float32[E][8],
    mask uint8[E][P]); params = size, cog_x, cog_y, length, width, psi, t_mean, q_max."""
    charge = np.ascontiguousarray(charge, dtype=np.float32)
    time = np.ascontiguousarray(time, dtype=np.float32)
    if charge.ndim != 2 or time.shape != charge.shape:
        raise ValueError("charge and time must be [n_events][n_pixels]")
    E, P = charge.shape
    pix_x = np.ascontiguousarray(pix_x, dtype=np.float32)
    pix_y = np.ascontiguousarray(pix_y, dtype=np.float32)
    neighbors = np.ascontiguousarray(neighbors, dtype=np.int32)
    if pix_x.shape != (P,) or pix_y.shape != (P,) or neighbors.shape != (P, 6):
        raise ValueError("geometry must be x[P], y[P], neighbors[P][6]")
    npix = np.empty(E, np.int32)
    params = np.empty((E, 8), np.float32)
    mask = np.empty((E, P), np.uint8)
    rc = _load().rta_oracle_image_moments(
        charge.ctypes.data, time.ctypes.data, E, P, pix_x.ctypes.data, pix_y.ctypes.data,
        neighbors.ctypes.data, float(thr_picture), float(thr_boundary), npix.ctypes.data,
        params.ctypes.data, mask.ctypes.data)
    if rc != 0:
        raise ValueError("rta_oracle_image_moments: bad shape")
    return npix, params, mask


def extract_threads(wf, pedestal, gain, W, threads: int):
    """The unmodified oracle function run on disjoint event ranges, one per
    thread (ctypes releases the GIL). Used only for the all-cores CPU figure."""
    from concurrent.futures import ThreadPoolExecutor
    E = wf.shape[0]
    threads = max(1, min(int(threads), E))
    bounds = [E * i // threads for i in range(threads + 1)]
    _load()
    with ThreadPoolExecutor(threads) as ex:
        parts = list(ex.map(
            lambda i: extract(wf[bounds[i]:bounds[i + 1]], pedestal, gain, W),
            range(threads)))
    return tuple(np.concatenate([p[k] for p in parts]) for k in range(4))
