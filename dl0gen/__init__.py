"""dl0gen — seeded synthetic DL0 camera waveforms (the inputs, nothing else).

Stands in for the paper's "Prod2" simulation (§5), which is not
available; the five workloads are BASELINE.json:configs[0..4] (C1..C5). This
package holds none of the extraction arithmetic. It serves both the oracle
side and the CUDA side of the tests and the bench: ``events_cpu`` (gcc build)
and ``events_cuda`` (nvcc build) write byte-identical waveforms, so any event
range generated on the GPU at bench scale can be regenerated on the host for
the oracle.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CPU_LIB = os.path.join(_HERE, "libdl0gen_cpu.so")
_CUDA_LIB = os.path.join(_HERE, "libdl0gen_cuda.so")
_lock = threading.Lock()
_cpu = None
_cuda = None


class Params(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64),
        ("n_pixels", ctypes.c_int32), ("n_samples", ctypes.c_int32),
        ("ped_lo", ctypes.c_int32), ("ped_hi", ctypes.c_int32),
        ("adc_max", ctypes.c_int32),
        ("gain_lo", ctypes.c_float), ("gain_hi", ctypes.c_float),
        ("noise_sigma", ctypes.c_float),
        ("pulse_frac", ctypes.c_float), ("pulse_sigma", ctypes.c_float),
        ("peak_lo", ctypes.c_float), ("peak_hi", ctypes.c_float),
        ("amp_mu", ctypes.c_float), ("amp_sigma", ctypes.c_float),
    ]


@dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json:configs."""
    name: str
    label: str
    seed: int
    n_events: int
    n_pixels: int
    n_samples: int
    W: int
    ped_lo: int
    ped_hi: int
    noise_sigma: float
    pulse_frac: float
    pulse_sigma: float
    peak_lo: float
    peak_hi: float
    amp_mu: float
    amp_sigma: float
    gain_lo: float = 0.9
    gain_hi: float = 1.1
    adc_max: int = 4095

    @property
    def n_traces(self) -> int:
        return self.n_events * self.n_pixels

    @property
    def trace_bytes(self) -> int:
        return 2 * self.n_samples

    @property
    def input_bytes(self) -> int:
        return self.n_traces * self.trace_bytes

    @property
    def output_bytes(self) -> int:
        return self.n_traces * 16

    def with_events(self, n_events: int) -> "Config":
        d = dict(self.__dict__)
        d["n_events"] = int(n_events)
        return Config(**d)

    def params(self) -> Params:
        return Params(self.seed, self.n_pixels, self.n_samples, self.ped_lo,
                      self.ped_hi, self.adc_max, self.gain_lo, self.gain_hi,
                      self.noise_sigma, self.pulse_frac, self.pulse_sigma,
                      self.peak_lo, self.peak_hi, self.amp_mu, self.amp_sigma)


# BASELINE.json:configs[0..4]; seeds: C1 = 0 as stated, C2..C5 = 1..4 (unstated).
CONFIGS = {
    "C1": Config("C1", "tiny LST-like 64x1855x30 W=7", 0, 64, 1855, 30, 7,
                 380, 420, 4.0, 0.05, 1.5, 8.0, 22.0, 3.0, 1.0),
    "C2": Config("C2", "LST-like 10000x1855x40 W=7", 1, 10_000, 1855, 40, 7,
                 380, 420, 4.0, 0.08, 1.5, 12.0, 28.0, 3.5, 1.2),
    "C3": Config("C3", "MST-like 20000x1764x25 W=4", 2, 20_000, 1764, 25, 4,
                 280, 320, 3.0, 0.05, 1.2, 6.0, 18.0, 3.0, 1.0),
    "C4": Config("C4", "SST-like 20000x2048x128 W=8", 3, 20_000, 2048, 128, 8,
                 480, 520, 5.0, 0.03, 3.0, 30.0, 100.0, 3.5, 1.3),
    "C5": Config("C5", "sustained stream 200000x1855x40 W=7", 4, 200_000, 1855,
                 40, 7, 380, 420, 4.0, 0.08, 1.5, 12.0, 28.0, 3.5, 1.2),
}


def _stale(lib, srcs):
    return (not os.path.exists(lib)
            or any(os.path.getmtime(lib) < os.path.getmtime(s) for s in srcs))


def build_cpu(force: bool = False) -> str:
    srcs = [os.path.join(_HERE, "dl0gen_cpu.c"), os.path.join(_HERE, "dl0gen_core.h")]
    with _lock:
        if force or _stale(_CPU_LIB, srcs):
            tmp = _CPU_LIB + ".tmp%d" % os.getpid()
            subprocess.check_call(
                ["gcc", "-std=c11", "-O2", "-fPIC", "-shared", "-ffp-contract=off",
                 "-fno-fast-math", "-o", tmp, srcs[0], "-lm"])
            os.replace(tmp, _CPU_LIB)
    return _CPU_LIB


def build_cuda(force: bool = False) -> str:
    srcs = [os.path.join(_HERE, "dl0gen_cuda.cu"), os.path.join(_HERE, "dl0gen_core.h")]
    with _lock:
        if force or _stale(_CUDA_LIB, srcs):
            tmp = _CUDA_LIB + ".tmp%d" % os.getpid()
            subprocess.check_call(
                ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3",
                 "-lineinfo", "-fmad=false", "-shared", "-Xcompiler", "-fPIC",
                 "-o", tmp, srcs[0]])
            os.replace(tmp, _CUDA_LIB)
    return _CUDA_LIB


def _cpu_lib():
    global _cpu
    if _cpu is None:
        lib = ctypes.CDLL(build_cpu())
        lib.dl0gen_calib.restype = None
        lib.dl0gen_calib.argtypes = [ctypes.POINTER(Params), ctypes.c_void_p, ctypes.c_void_p]
        lib.dl0gen_events_cpu.restype = None
        lib.dl0gen_events_cpu.argtypes = [ctypes.POINTER(Params), ctypes.c_int64,
                                          ctypes.c_int64, ctypes.c_void_p]
        lib.dl0gen_pack12_cpu.restype = None
        lib.dl0gen_pack12_cpu.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p]
        _cpu = lib
    return _cpu


def _cuda_lib():
    global _cuda
    if _cuda is None:
        lib = ctypes.CDLL(build_cuda())
        lib.dl0gen_events_cuda.restype = ctypes.c_int
        lib.dl0gen_events_cuda.argtypes = [ctypes.POINTER(Params), ctypes.c_longlong,
                                           ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.dl0gen_pack12_cuda.restype = ctypes.c_int
        lib.dl0gen_pack12_cuda.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p,
                                           ctypes.c_void_p]
        _cuda = lib
    return _cuda


def calib(cfg: Config):
    """(pedestal int32[P], gain float32[P]) for a config."""
    ped = np.empty(cfg.n_pixels, np.int32)
    gain = np.empty(cfg.n_pixels, np.float32)
    p = cfg.params()
    _cpu_lib().dl0gen_calib(ctypes.byref(p), ped.ctypes.data, gain.ctypes.data)
    return ped, gain


def events_cpu(cfg: Config, first_event: int = 0, n_events: int | None = None,
               threads: int = 1) -> np.ndarray:
    """uint16 [n_events][P][S] for events first_event.. on the host."""
    if n_events is None:
        n_events = cfg.n_events - first_event
    out = np.empty((n_events, cfg.n_pixels, cfg.n_samples), np.uint16)
    p = cfg.params()
    lib = _cpu_lib()
    threads = max(1, min(int(threads), max(1, n_events)))
    if threads == 1:
        lib.dl0gen_events_cpu(ctypes.byref(p), first_event, n_events, out.ctypes.data)
        return out
    from concurrent.futures import ThreadPoolExecutor
    b = [n_events * i // threads for i in range(threads + 1)]
    ev_bytes = cfg.n_pixels * cfg.n_samples * 2

    def work(i):
        lib.dl0gen_events_cpu(ctypes.byref(p), first_event + b[i], b[i + 1] - b[i],
                              out.ctypes.data + b[i] * ev_bytes)
    with ThreadPoolExecutor(threads) as ex:
        list(ex.map(work, range(threads)))
    return out


def events_cuda(cfg: Config, wf_dev_ptr: int, first_event: int, n_events: int,
                stream: int = 0) -> None:
    """Fill a DEVICE buffer (raw pointer) with events first_event.. ; async on
    ``stream``. Byte-identical to :func:`events_cpu`."""
    p = cfg.params()
    rc = _cuda_lib().dl0gen_events_cuda(ctypes.byref(p), first_event, n_events,
                                        ctypes.c_void_p(wf_dev_ptr), ctypes.c_void_p(stream))
    if rc != 0:
        raise RuntimeError("dl0gen_events_cuda: cudaError %d" % rc)


def packed12_nbytes(n_samples_total: int) -> int:
    """Bytes of a P12 stream (12-bit little-endian packed) of that many samples."""
    return (12 * int(n_samples_total) + 7) // 8


def pack12_cpu(wf: np.ndarray) -> np.ndarray:
    """Encode uint16 samples (any shape, flattened in C order, masked to 12 bits)
    as a P12 byte stream. Input preparation only: decoding is the method's step."""
    wf = np.ascontiguousarray(wf, dtype=np.uint16).ravel()
    out = np.empty(packed12_nbytes(wf.size), np.uint8)
    _cpu_lib().dl0gen_pack12_cpu(wf.ctypes.data, wf.size, out.ctypes.data)
    return out


def pack12_cuda(wf_dev_ptr: int, n_samples_total: int, out_dev_ptr: int, stream: int = 0) -> None:
    """Device build of :func:`pack12_cpu` (raw device pointers; async on ``stream``)."""
    rc = _cuda_lib().dl0gen_pack12_cuda(ctypes.c_void_p(wf_dev_ptr), int(n_samples_total),
                                        ctypes.c_void_p(out_dev_ptr), ctypes.c_void_p(stream))
    if rc != 0:
        raise RuntimeError("dl0gen_pack12_cuda: cudaError %d" % rc)


# --------------------------------------------------------------------------- #
# Mixed-camera batches: layout arithmetic only.
class MixedArray:
    """A sub-array of telescopes with the cameras of C2/C3/C4 (LST-, MST-, SST-like;
    PAPER.md:39 names the three sizes), every telescope triggered in every event.
    Event e holds one block per telescope slot, in slot order, each block starting
    on a multiple of ``align`` samples; event e of slot j is event ``j_c * n_events
    + e`` of its camera's config, j_c being the slot's rank among slots of the same
    camera — so any block can be regenerated on the host."""

    def __init__(self, slots=(("C2", 4), ("C3", 10), ("C4", 6)), n_events=1000, align=8):
        self.n_events = int(n_events)
        self.slots = []                                   # (config, rank among its camera)
        for name, count in slots:                         # a config name, or a Config of another shape
            for j in range(count):
                self.slots.append((CONFIGS[name] if isinstance(name, str) else name, j))
        self.tel_n_pixels = [c.n_pixels for c, _ in self.slots]
        self.tel_n_samples = [c.n_samples for c, _ in self.slots]
        self.tel_W = [c.W for c, _ in self.slots]
        self.tel_calib_offset, cal = [], 0
        for c, _ in self.slots:
            self.tel_calib_offset.append(cal)
            cal += c.n_pixels
        self.n_calib = cal
        self.slot_offset, pos = [], 0                     # samples, inside one event
        for c, _ in self.slots:
            pos += -pos % align
            self.slot_offset.append(pos)
            pos += c.n_pixels * c.n_samples
        pos += -pos % align
        self.event_stride = pos                           # samples
        self.traces_per_event = sum(self.tel_n_pixels)
        self.slot_out = [sum(self.tel_n_pixels[:j]) for j in range(len(self.slots))]
        self.blk_tel, self.blk_wf_offset, self.blk_out_offset = [], [], []
        for e in range(self.n_events):
            for j in range(len(self.slots)):
                self.blk_tel.append(j)
                self.blk_wf_offset.append(e * self.event_stride + self.slot_offset[j])
                self.blk_out_offset.append(e * self.traces_per_event + self.slot_out[j])
        self.n_samples_total = self.n_events * self.event_stride
        self.n_traces = self.n_events * self.traces_per_event
        self.wf_bytes = 2 * self.n_events * sum(p * s for p, s in zip(self.tel_n_pixels, self.tel_n_samples))

    def tables(self):
        return (self.tel_n_pixels, self.tel_n_samples, self.tel_W, self.tel_calib_offset,
                self.blk_tel, self.blk_wf_offset, self.blk_out_offset)

    def calib(self):
        peds, gains = zip(*[calib(c) for c, _ in self.slots])
        return np.concatenate(peds), np.concatenate(gains)

    def block_cpu(self, event: int, slot: int) -> np.ndarray:
        """uint16 [P][S] of one block, regenerated on the host."""
        c, j = self.slots[slot]
        return events_cpu(c, j * self.n_events + event, 1)[0]

    def fill_cuda(self, torch, d_flat) -> None:
        """Generate every block into ``d_flat`` (int16 device tensor of
        n_samples_total elements); gaps keep their previous content."""
        st = torch.cuda.current_stream().cuda_stream
        for slot, (c, j) in enumerate(self.slots):
            n = c.n_pixels * c.n_samples
            tmp = torch.empty((self.n_events, n), dtype=torch.int16, device=d_flat.device)
            events_cuda(c, tmp.data_ptr(), j * self.n_events, self.n_events, st)
            view = torch.as_strided(d_flat, (self.n_events, n), (self.event_stride, 1),
                                    self.slot_offset[slot])
            view.copy_(tmp)
            del tmp


# --------------------------------------------------------------------------- #
# Synthetic camera geometry (the real pixel tables are
# not available). Geometry only: no cleaning, no moments.
# Cleaning thresholds (picture, boundary) used with each config's charges by the
# tests and bench.py (inputs of the call, chosen so that most events keep a few
# dozen pixels and a few keep none; charge unit = ADC counts summed over W).
IMAGE_THRESHOLDS = {"C1": (60.0, 30.0), "C2": (60.0, 30.0), "C3": (40.0, 20.0), "C4": (60.0, 30.0),
                    "C5": (60.0, 30.0)}


def hex_camera(n_pixels: int, pitch: float = 0.05):
    """The ``n_pixels`` hexagonal-lattice points nearest the origin (ties broken
    by the integer axial coordinates, so the result is platform-independent).
    Returns (x float32[P], y float32[P], neighbors int32[P][6], -1 = none).
    Axial (a, b): x = pitch (a + b/2), y = pitch (sqrt(3)/2) b; neighbours are the
    six lattice neighbours (+-1,0), (0,+-1), (1,-1), (-1,1) present in the set."""
    n_pixels = int(n_pixels)
    r = 2
    while 3 * r * (r + 1) + 1 < n_pixels:
        r += 1
    r += 2
    pts = [(a * a + a * b + b * b, a, b) for a in range(-r, r + 1) for b in range(-r, r + 1)]
    pts.sort()
    pts = pts[:n_pixels]
    index = {(a, b): i for i, (_, a, b) in enumerate(pts)}
    x = np.array([pitch * (a + 0.5 * b) for _, a, b in pts], np.float64).astype(np.float32)
    y = np.array([pitch * (np.sqrt(3.0) / 2.0) * b for _, a, b in pts], np.float64).astype(np.float32)
    nbr = np.full((n_pixels, 6), -1, np.int32)
    for i, (_, a, b) in enumerate(pts):
        for j, (da, db) in enumerate(((1, 0), (-1, 0), (0, 1), (0, -1), (1, -1), (-1, 1))):
            nbr[i, j] = index.get((a + da, b + db), -1)
    return x, y, nbr
