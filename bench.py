#!/usr/bin/env python
"""bench.py — waveform GB/s extracted on B200 (BASELINE.json:metric).

One "step" is one pass of the whole hot path (ingest,
pedestal, window sums, arg-max, stores, charge, peak time) over one batch of
synthetic camera waveforms, i.e. one rta_extract call through the C ABI.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C3|C4|C1]
  python bench.py --impl reference ...      # the oracle on the host cores

Prints ONE JSON line (rank 0). Keys beyond the driver's contract:
  roofline      dominant kernel against the measured HBM peak
  cpu_baseline  the oracle timed on this box's host cores (N=1, rank 0)
  e2e           same metric through rta_extract_host (pinned host buffers in
                and out, H2D/D2H inside the timed region)
  sustained     BASELINE.json:configs[4] (C5): 29.68 GB of pinned host memory
                fed through rta_extract_stream in 1 GiB chunks, against the
                host-link bandwidth measured in the same run and the paper's
                0.5-8 GB/s array data rate
  configs       kernel-only numbers for the other single-GPU configs (C3, C4) and the
                small case C1 (eager and CUDA-graph replay, L2 flushed and resident)
  family        the other extractors (NEXT-1) on the same batches
  packed12      NEXT-2: the same batches as P12 streams (12 bits per sample),
                decoded inside the extraction kernel; sustained.packed12 is C5
                fed as 22.26 GB of P12 through rta_extract_stream_packed12
  ragged        NEXT-3: a mixed-camera array through rta_extract_ragged
  image         NEXT-4: rta_extract_image (extraction + cleaning + moments in one
                kernel) next to rta_extract followed by rta_image_moments;
                sustained.image is C5 through rta_extract_image_stream
  latency       host wall time per call (p50 / p99) for 1 .. 4096 events of the C2 camera:
                rta_extract eager and as a graph replay, rta_extract_host, rta_extract_image_host
  any_shape     shapes without a specialised kernel (not BASELINE configs) through
                the staged kernel with runtime (n_samples, W), next to the generic one
Secondary legs are single-GPU diagnostics (N = 1 only) and run ten untimed launches first.

`--gpus N` without a torchrun environment re-executes itself under
`python -m torch.distributed.run --standalone --nproc-per-node N` (one rank per
GPU, NCCL for the barrier and the MAX over ranks only; no data-path collective).
At N > 1 every rank also runs the host-fed `sustained` leg on its own pinned
buffer (each GPU has its own host link); `value` there is the aggregate over
ranks on the slowest rank's time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "raw_waveform_GBps_extracted"
UNIT = "GB/s"
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
PAPER_RATE_GBS = (0.5, 8.0)       # PAPER.md:27 / PAPER.md:67, whole-array data rate
ALGO_BYTES_PER_TRACE_OUT = 16     # 2*S read + 16 written per trace


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C2",
                    choices=["C1", "C2", "C3", "C4", "X60", "X40w5", "X96", "X128w10", "X2048"],
                    help="C1..C4: BASELINE.json configs; X*: shapes without a specialised kernel "
                         "(diagnostic runs of the runtime-shape kernel, imply --no-extra)")
    ap.add_argument("--input-format", default="u16", choices=["u16", "p12"],
                    help="u16: BASELINE.json's uint16 waveforms (the headline); p12: the same batch as "
                         "a packed 12-bit stream through rta_extract_packed12 (NEXT-2)")
    ap.add_argument("--path", default="extract", choices=["extract", "image", "moments"],
                    help="main leg: rta_extract (default, the BASELINE metric); 'image' = "
                         "rta_extract_image, 'moments' = rta_image_moments (diagnostic runs "
                         "for profiling, imply --no-extra)")
    ap.add_argument("--extractor", default="sliding", choices=["sliding", "fixed", "local_peak", "fir"],
                    help="main leg with --path extract: rta_extract (default, the BASELINE metric) or one "
                         "of the NEXT-1 extractors (diagnostic / profiling runs; secondary legs are skipped)")
    ap.add_argument("--no-extra", action="store_true", help="skip configs/e2e/sustained/cpu legs")
    ap.add_argument("--no-sustained", action="store_true", help="skip the 29.68 GB C5 leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--legs", default="all",
                    help="comma list of the secondary single-GPU legs to run: configs, family, packed12, "
                         "any_shape, ragged, image (default: all; the profiling commands in profiles/ "
                         "name one leg each)")
    ap.add_argument("--e2e-chunk-mb", type=int, default=64)
    return ap.parse_args()


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def csrc_sha256():
    """Content hash of the kernel sources: ties an ncu capture to the code it measured
    (the GPU box has no .git)."""
    import hashlib
    d = os.path.join(ROOT, "paper_1307_6489_b200", "csrc")
    h = hashlib.sha256()
    for n in sorted(os.listdir(d)):
        if n.endswith((".cu", ".cuh", ".h")):
            h.update(n.encode())
            h.update(open(os.path.join(d, n), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(name):
    """DRAM bytes per launch from the committed ncu --set full capture
    (profiles/traffic.json), or None when the kernel sources have changed since
    that capture. Returns (bytes or None, commit of the capture, stale?)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        t = json.load(open(p))
    except Exception:
        return None, None, None
    stale = t.get("csrc_sha256") != csrc_sha256()
    return (None if stale else t.get("kernels", {}).get(name)), t.get("commit"), stale


def oracle_sample_events(cfg):
    """The ONE sampling rule for timing the oracle (both arms): the whole workload
    when its input is at most 2 GB (C1, C2, C3), else the first 2 GB of events."""
    ev_bytes = cfg.n_pixels * cfg.n_samples * 2
    return min(cfg.n_events, max(1, int(2e9 // ev_bytes)))


def event_slabs(n_events, event_bytes, slab_bytes=1 << 30):
    step = max(1, slab_bytes // event_bytes)
    for e0 in range(0, n_events, step):
        yield e0, min(step, n_events - e0)


def bits_equal(torch, dev_out, want, lo, hi):
    """device outputs [lo, hi) == oracle outputs, bit for bit (floats as int32)."""
    import numpy as np
    return all(np.array_equal(o[lo:hi].cpu().numpy().view(np.int32), w.view(np.int32))
               for o, w in zip(dev_out, want))


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: an NVML
    polling thread (about 1 kHz; the timed region of a default run lasts only a
    few tens of ms), or `nvidia-smi -lms` when NVML cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index, uuid=None):
        self.index = index
        self.uuid = uuid
        self.proc = None
        self.lines = []
        self.nvml = None
        self.samples = []          # (sm_mhz, reasons bitmask)
        self.sm_max = None
        self.stop_flag = threading.Event()
        self.thread = None

    def _nvml_handle(self):
        import pynvml
        pynvml.nvmlInit()
        if self.uuid:
            try:
                u = self.uuid if str(self.uuid).startswith("GPU-") else "GPU-" + str(self.uuid)
                return pynvml, pynvml.nvmlDeviceGetHandleByUUID(u.encode())
            except Exception:
                pass
        return pynvml, pynvml.nvmlDeviceGetHandleByIndex(self.index)

    def start(self):
        try:
            self.nvml, self.handle = self._nvml_handle()
            self.sm_max = float(self.nvml.nvmlDeviceGetMaxClockInfo(self.handle, self.nvml.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _poll(self):
        n = self.nvml
        while not self.stop_flag.is_set():
            try:
                mhz = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                mask = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                try:
                    watts = n.nvmlDeviceGetPowerUsage(self.handle) / 1000.0
                except Exception:
                    watts = None
                self.samples.append((mhz, mask, watts))
            except Exception:
                pass
            time.sleep(0.001)

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def mark(self):
        """Number of samples so far: bracket the timed region with two marks."""
        return len(self.samples) if self.nvml else len(self.lines)

    def window(self, lo, hi):
        """Clocks and power of the samples [lo, hi) of a running sampler (NVML only), for the
        secondary legs: an arithmetic-bound leg late in a long run can meet lower clocks."""
        if not self.nvml or hi <= lo:
            return None
        sel = self.samples[lo:hi]
        sm = [x[0] for x in sel]
        w = [x[2] for x in sel if x[2] is not None]
        cap = self.nvml.nvmlClocksThrottleReasonSwPowerCap
        return {"sm_mhz": statistics.median(sm), "sm_min_mhz": min(sm), "watts_max": max(w) if w else None,
                "sw_power_cap": any(x[1] & cap for x in sel), "samples": len(sm)}

    def stop(self, lo=0, hi=None):
        if self.nvml:
            self.stop_flag.set()
            self.thread.join(timeout=2)
            n = self.nvml
            sel = self.samples[lo:hi] or self.samples
            bits = {"hw_slowdown": n.nvmlClocksThrottleReasonHwSlowdown,
                    "hw_thermal_slowdown": n.nvmlClocksThrottleReasonHwThermalSlowdown,
                    "sw_thermal_slowdown": n.nvmlClocksThrottleReasonSwThermalSlowdown,
                    "sw_power_cap": n.nvmlClocksThrottleReasonSwPowerCap}
            reasons = sorted(k for k, b in bits.items() if any(x[1] & b for x in sel))
            sm = [x[0] for x in sel]
            return {"sm_mhz": statistics.median(sm) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                    "sm_max_mhz": self.sm_max, "samples": len(sm), "source": "nvml, timed region only",
                    "reasons": reasons}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in (self.lines[lo:hi] or self.lines):
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(self.NAMES, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "source": "nvidia-smi -lms 20", "reasons": sorted(reasons)}


# --------------------------------------------------------------------------- #
def reference_arm(args):
    """The oracle, as it stands, on the host cores: same metric and config.
    Each step extracts a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np
    import dl0gen
    import oracle
    cfg = workload(args.workload, dl0gen)
    cores = os.cpu_count() or 1
    ped, gain = dl0gen.calib(cfg)
    n_ev = oracle_sample_events(cfg)      # the same sample as the b200 arm's cpu_baseline
    wf = dl0gen.events_cpu(cfg, 0, n_ev, threads=cores)
    for _ in range(max(1, min(args.warmup, 1))):
        oracle.extract_threads(wf, ped, gain, cfg.W, cores)
    # bounded: at most `steps` passes and about two minutes of oracle time
    steps, t_used = 0, 0.0
    while steps < args.steps and (steps == 0 or t_used < 120.0):
        t0 = time.perf_counter()
        oracle.extract_threads(wf, ped, gain, cfg.W, cores)
        t_used += time.perf_counter() - t0
        steps += 1
    dt = t_used / steps
    val = wf.nbytes / dt / 1e9
    sample = "first %d of %d events of %s per step, %d threads" % (n_ev, cfg.n_events, cfg.name, cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT,
        "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup,
        "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": "%s: %s" % (cfg.name, cfg.label), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
    return 0


# --------------------------------------------------------------------------- #
def time_steps(run, steps, stream):
    """K back-to-back launches with an event between each: per-launch device
    durations on the launching stream; their sum is the timed region."""
    import torch
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for i in range(steps):
        run()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    return [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]


def device_batch(cfg, torch, dl0gen):
    d_wf = torch.empty((cfg.n_events, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(cfg, d_wf.data_ptr(), 0, cfg.n_events, torch.cuda.current_stream().cuda_stream)
    ped, gain = dl0gen.calib(cfg)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    outs = [torch.empty(cfg.n_traces, dtype=dt, device="cuda")
            for dt in (torch.int32, torch.int32, torch.float32, torch.float32)]
    torch.cuda.synchronize()
    return d_wf, d_ped, d_gain, outs, ped, gain


def camera_on_device(cfg, torch, dl0gen):
    x, y, nbr = dl0gen.hex_camera(cfg.n_pixels)
    tp, tb = dl0gen.IMAGE_THRESHOLDS[cfg.name]
    return torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda(), torch.from_numpy(nbr).cuda(), tp, tb


def image_outputs(cfg, torch):
    return (torch.empty(cfg.n_events, dtype=torch.int32, device="cuda"),
            torch.empty((cfg.n_events, 8), dtype=torch.float32, device="cuda"))


def family_runs(cfg, base, outs, stream, torch, rta):
    """The three NEXT-1 extractors on one device batch: per-pixel fixed window starts
    (seeded), local peak with shift W/2, FIR with triangular taps."""
    import numpy as np
    start = torch.from_numpy(np.random.default_rng(cfg.seed).integers(
        0, cfg.n_samples - cfg.W + 1, cfg.n_pixels).astype(np.int32)).cuda()
    taps = [1, 2, 3, 4, 3, 2, 1, 1][:cfg.W]
    runs = {
        "fixed": lambda: rta.rta_extract_fixed(*base, cfg.W, start, *outs, stream=stream),
        "local_peak": lambda: rta.rta_extract_local_peak(*base, cfg.W, cfg.W // 2, *outs, stream=stream),
        "fir": lambda: rta.rta_extract_fir(*base, taps, *outs, stream=stream),
    }
    return runs, start, taps


def fixed_gather_bytes_per_trace(cfg, start):
    """rta_extract_fixed GATHERS for traces longer than 96 bytes (rta_kernels.cu launch_mode): it
    touches only the W-sample window of a trace, so its algorithmic bytes are the 32-byte sectors
    that window overlaps (+ 16 bytes out), not the whole waveform. None when it streams."""
    import numpy as np
    if 2 * cfg.n_samples <= 96:
        return None, None
    st = start.cpu().numpy().astype(np.int64)
    g = np.arange(min(cfg.n_traces, 64 * cfg.n_pixels), dtype=np.int64)
    lo = g * (2 * cfg.n_samples) + 2 * st[g % cfg.n_pixels]
    sectors = (lo + 2 * cfg.W - 1) // 32 - lo // 32 + 1
    return 32.0 * float(sectors.mean()) + ALGO_BYTES_PER_TRACE_OUT, float(sectors.mean())


def kernel_only(cfg, steps, warmup, torch, dl0gen, rta, barrier=None, sampler=None, fmt="u16",
                path="extract", extractor="sliding"):
    d_wf, d_ped, d_gain, outs, ped, gain = device_batch(cfg, torch, dl0gen)
    stream = torch.cuda.current_stream()
    if path in ("image", "moments"):
        cam = camera_on_device(cfg, torch, dl0gen)
        ev_out = image_outputs(cfg, torch)
        if path == "image":
            def run():
                rta.rta_extract_image(d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped,
                                      d_gain, cfg.W, *cam, *ev_out, None, stream=stream)
        else:
            rta.rta_extract(d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain,
                            cfg.W, *outs, stream=stream)

            def run():
                rta.rta_image_moments(outs[2], outs[3], cfg.n_events, cfg.n_pixels, *cam,
                                      *ev_out, None, stream=stream)
    elif fmt == "p12":
        n_total = cfg.n_traces * cfg.n_samples
        d_pk = torch.empty(dl0gen.packed12_nbytes(n_total), dtype=torch.uint8, device="cuda")
        dl0gen.pack12_cuda(d_wf.data_ptr(), n_total, d_pk.data_ptr(), stream.cuda_stream)
        torch.cuda.synchronize()

        def run():
            rta.rta_extract_packed12(d_pk, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped,
                                     d_gain, cfg.W, *outs, stream=stream)
    elif extractor != "sliding":
        runs, fam_start, _ = family_runs(
            cfg, (d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain), outs, stream, torch, rta)
        run = runs[extractor]
    else:
        def run():
            rta.rta_extract(d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain,
                            cfg.W, *outs, stream=stream)
    for _ in range(max(3, warmup)):
        run()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    before = rta.rta_launch_count()
    m0 = sampler.mark() if sampler else 0
    per = time_steps(run, steps, stream)
    m1 = sampler.mark() if sampler else 0
    launches = rta.rta_launch_count() - before
    if barrier:
        barrier()
    checksum = int(d_wf.view(-1)[: min(d_wf.numel(), 1 << 26)].sum(dtype=torch.int64))
    return {"per_launch_ms": per, "launches": launches, "checksum_first_64Mi_samples": checksum,
            "marks": (m0, m1), "fixed_start": fam_start if extractor == "fixed" else None,
            "keep": (d_wf, d_ped, d_gain, outs, ped, gain)}


def summarise(cfg, per_ms, peak):
    tot_ms = sum(per_ms)
    avg = tot_ms / len(per_ms)
    algo = cfg.input_bytes + cfg.output_bytes
    return {
        "workload": "%s: %s" % (cfg.name, cfg.label),
        "ms_avg": avg, "ms_median": statistics.median(per_ms), "ms_best": min(per_ms),
        "waveform_GBps": cfg.input_bytes / avg / 1e6,
        "traces_per_s": cfg.n_traces / avg * 1e3,
        "algorithmic_GBps": algo / avg / 1e6,
        "frac_of_measured_hbm": algo / avg / 1e6 / peak,
        "frac_of_nominal_8TBps": algo / avg / 1e6 / 8000.0,
    }


def family_leg(cfg, steps, peak, torch, dl0gen, rta):
    """Kernel-only throughput of the other extractors (NEXT-1) on the same
    device-resident batch: fixed window, local peak, FIR (triangular taps)."""
    import numpy as np
    d_wf, d_ped, d_gain, outs, ped, gain = device_batch(cfg, torch, dl0gen)
    stream = torch.cuda.current_stream()
    base = (d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain)
    runs, start, taps = family_runs(cfg, base, outs, stream, torch, rta)
    res = {}
    for name, run in runs.items():
        for _ in range(LEG_WARMUP):
            run()
        torch.cuda.synchronize()
        res[name] = summarise(cfg, time_steps(run, steps, stream), peak)
    res["fir"]["taps"] = taps
    per_trace, mean_sectors = fixed_gather_bytes_per_trace(cfg, start)
    if per_trace is not None:
        f = res["fixed"]
        algo = per_trace * cfg.n_traces
        f["route"] = "gather (generic kernel): W samples of each trace from global memory"
        f["bytes_per_trace"] = per_trace
        f["mean_sectors_per_trace"] = mean_sectors
        f["streamed_equivalent_GBps"] = f["algorithmic_GBps"]
        f["algorithmic_GBps"] = algo / f["ms_avg"] / 1e6
        f["frac_of_measured_hbm"] = f["algorithmic_GBps"] / peak
        f["frac_of_nominal_8TBps"] = f["algorithmic_GBps"] / 8000.0
    else:
        res["fixed"]["route"] = "streamed (staged kernel): whole tiles cross HBM"
    return res


def packed_leg(cfg, steps, peak, torch, dl0gen, rta):
    """Kernel-only throughput of rta_extract_packed12 on the batch of `cfg`
    stored as a P12 stream (1.5 bytes per sample instead of 2)."""
    d_wf, d_ped, d_gain, outs, ped, gain = device_batch(cfg, torch, dl0gen)
    stream = torch.cuda.current_stream()
    n_total = cfg.n_traces * cfg.n_samples
    nb = dl0gen.packed12_nbytes(n_total)
    d_pk = torch.empty(nb, dtype=torch.uint8, device="cuda")
    dl0gen.pack12_cuda(d_wf.data_ptr(), n_total, d_pk.data_ptr(), stream.cuda_stream)
    torch.cuda.synchronize()
    del d_wf

    def run():
        rta.rta_extract_packed12(d_pk, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain,
                                 cfg.W, *outs, stream=stream)
    for _ in range(LEG_WARMUP):
        run()
    torch.cuda.synchronize()
    per = time_steps(run, steps, stream)
    avg = sum(per) / len(per)
    algo = nb + cfg.output_bytes
    return {"workload": "%s as P12: %s" % (cfg.name, cfg.label),
            "kernel": rta.rta_kernel_name_packed12(cfg.n_samples, cfg.W, True),
            "ms_avg": avg, "ms_median": statistics.median(per), "ms_best": min(per),
            "packed_input_bytes": nb, "algorithmic_bytes_per_launch": algo,
            "bytes_per_trace": 1.5 * cfg.n_samples + ALGO_BYTES_PER_TRACE_OUT,
            "algorithmic_GBps": algo / avg / 1e6, "frac_of_measured_hbm": algo / avg / 1e6 / peak,
            "packed_GBps": nb / avg / 1e6,
            "waveform_equivalent_GBps": cfg.input_bytes / avg / 1e6,
            "traces_per_s": cfg.n_traces / avg * 1e3}


def ragged_leg(steps, peak, torch, dl0gen, rta, n_events=1000, slots=None, label=None):
    """NEXT-3: a mixed-camera array (4 LST-, 10 MST-, 6 SST-like telescopes, the
    cameras of C2/C3/C4), every event holding one block per telescope, through
    one rta_extract_ragged call (one launch per camera shape). `slots` names
    another array (the second measurement: cameras without a specialised kernel)."""
    m = dl0gen.MixedArray(n_events=n_events) if slots is None else dl0gen.MixedArray(slots, n_events)
    ped, gain = m.calib()
    d_wf = torch.zeros(m.n_samples_total, dtype=torch.int16, device="cuda")
    m.fill_cuda(torch, d_wf)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    outs = [torch.empty(m.n_traces, dtype=dt, device="cuda")
            for dt in (torch.int32, torch.int32, torch.float32, torch.float32)]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    plan = rta.rta_ragged_plan_create(*m.tables())
    t_plan = time.perf_counter() - t0
    stream = torch.cuda.current_stream()

    def run():
        rta.rta_extract_ragged(plan, d_wf, d_ped, d_gain, *outs, stream=stream)
    for _ in range(LEG_WARMUP):
        run()
    torch.cuda.synchronize()
    before = rta.rta_launch_count()
    per = time_steps(run, steps, stream)
    launches = (rta.rta_launch_count() - before) // steps
    avg = sum(per) / len(per)
    algo = m.wf_bytes + 16 * m.n_traces
    res = {"workload": "mixed array: %d events x (%s), %d blocks on 16-byte boundaries" % (
               m.n_events, label or "4 x 1855x40 W7 + 10 x 1764x25 W4 + 6 x 2048x128 W8", len(m.blk_tel)),
           "ms_avg": avg, "ms_median": statistics.median(per), "ms_best": min(per),
           "launches_per_call": launches, "tiles": rta.rta_ragged_plan_info(plan, rta.RTA_RAGGED_N_TILES),
           "waveform_bytes": m.wf_bytes, "algorithmic_bytes_per_call": algo,
           "waveform_GBps": m.wf_bytes / avg / 1e6, "algorithmic_GBps": algo / avg / 1e6,
           "frac_of_measured_hbm": algo / avg / 1e6 / peak, "traces_per_s": m.n_traces / avg * 1e3,
           "plan_create_ms_host": t_plan * 1e3}
    rta.rta_ragged_plan_destroy(plan)
    return res


def extra_shapes(dl0gen):
    """Workloads that are NOT BASELINE configs: C2's and C4's signal models with another
    readout length or window width (shapes without a specialised kernel)."""
    import dataclasses
    c2, c4 = dl0gen.CONFIGS["C2"], dl0gen.CONFIGS["C4"]
    shapes = [dataclasses.replace(c2, name="X60", label="10000x1855x60 W=7", seed=11, n_samples=60,
                                  peak_lo=15.0, peak_hi=45.0),
              dataclasses.replace(c2, name="X40w5", label="10000x1855x40 W=5", seed=12, W=5),
              dataclasses.replace(c4, name="X96", label="10000x2048x96 W=8", seed=13, n_events=10_000,
                                  n_samples=96, peak_lo=25.0, peak_hi=70.0),
              dataclasses.replace(c4, name="X128w10", label="10000x2048x128 W=10", seed=14,
                                  n_events=10_000, W=10),
              # traces too long for one thread (4096 bytes): a warp per trace
              dataclasses.replace(c4, name="X2048", label="1000x2048x2048 W=12", seed=15,
                                  n_events=1000, n_samples=2048, W=12, peak_lo=200.0, peak_hi=1800.0)]
    return {c.name: c for c in shapes}


def workload(name, dl0gen):
    return dl0gen.CONFIGS[name] if name in dl0gen.CONFIGS else extra_shapes(dl0gen)[name]


def any_shape_leg(steps, peak, torch, dl0gen, rta):
    """Shapes without a specialised kernel (not BASELINE configs: C2's and C4's
    signal models with other readout lengths / window widths) through rta_extract:
    the staged kernel with runtime (S, W), next to the old generic kernel."""
    res = {}
    for cfg in extra_shapes(dl0gen).values():
        d_wf, d_ped, d_gain, outs, ped, gain = device_batch(cfg, torch, dl0gen)
        stream = torch.cuda.current_stream()
        base = (d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain, cfg.W)
        r = {"kernel": rta.rta_kernel_name(cfg.n_samples, cfg.W, True)}
        ref = None
        for name, generic in (("staged_any", False), ("generic", True)):
            def run():
                rta.rta_extract(*base, *outs, stream=stream, generic=generic)
            for _ in range(LEG_WARMUP):
                run()
            torch.cuda.synchronize()
            r[name] = summarise(cfg, time_steps(run, steps if not generic else 3, stream), peak)
            got = [o.clone() for o in outs]
            if ref is not None:
                r["both_kernels_bit_identical"] = all(
                    bool((a.view(torch.int32) == b.view(torch.int32)).all()) for a, b in zip(ref, got))
            ref = got
        r["speedup_vs_generic"] = r["generic"]["ms_avg"] / r["staged_any"]["ms_avg"]
        res[cfg.name] = r
        del d_wf, outs, ref, got
        torch.cuda.empty_cache()
    return res


SECONDARY_LEGS = ("configs", "family", "packed12", "any_shape", "ragged", "image", "latency")
EVENT_OUT_BYTES = 36   # n_pix int32 + 8 fp32 parameters per event
LEG_WARMUP = 10        # untimed launches in front of every secondary leg (the GPU idles while a leg sets up)


def image_leg(cfg, steps, peak, torch, dl0gen, rta):
    """NEXT-4: extraction + cleaning + moments. `fused` = rta_extract_image (one
    kernel, 36 bytes per event written); `two_calls` = rta_extract followed by
    rta_image_moments (charge / time cross HBM twice); `moments` = the second
    call alone. GB/s are algorithmic bytes of each leg over its device time."""
    d_wf, d_ped, d_gain, outs, ped, gain = device_batch(cfg, torch, dl0gen)
    cam = camera_on_device(cfg, torch, dl0gen)
    ev_out = image_outputs(cfg, torch)
    stream = torch.cuda.current_stream()
    base = (d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain, cfg.W)

    def fused():
        rta.rta_extract_image(*base, *cam, *ev_out, None, stream=stream)

    def moments():
        rta.rta_image_moments(outs[2], outs[3], cfg.n_events, cfg.n_pixels, *cam, *ev_out, None,
                              stream=stream)

    def two_calls():
        rta.rta_extract(*base, *outs, stream=stream)
        moments()
    ev_bytes = EVENT_OUT_BYTES * cfg.n_events
    algo = {"fused": cfg.input_bytes + ev_bytes,
            "two_calls": cfg.input_bytes + cfg.output_bytes + 4 * cfg.n_traces + ev_bytes,
            "moments": 4 * cfg.n_traces + ev_bytes}
    res = {"workload": "%s: %s; hex camera, thresholds %g / %g" % (
        cfg.name, cfg.label, cam[3], cam[4]),
        "kernel": rta.rta_image_kernel_name(cfg.n_pixels, cfg.n_samples, cfg.W, True)}
    for name, run in (("fused", fused), ("two_calls", two_calls), ("moments", moments)):
        for _ in range(LEG_WARMUP):
            run()
        torch.cuda.synchronize()
        per = time_steps(run, steps, stream)
        avg = sum(per) / len(per)
        res[name] = {"ms_avg": avg, "ms_median": statistics.median(per), "ms_best": min(per),
                     "algorithmic_bytes": algo[name], "algorithmic_GBps": algo[name] / avg / 1e6,
                     "frac_of_measured_hbm": algo[name] / avg / 1e6 / peak,
                     "waveform_GBps": cfg.input_bytes / avg / 1e6,
                     "events_per_s": cfg.n_events / avg * 1e3}
    n = ev_out[0].cpu()
    res["mean_pixels_in_image"] = float(n.float().mean())
    res["empty_events_frac"] = float((n == 0).float().mean())
    res["fused_speedup_vs_two_calls"] = res["two_calls"]["ms_avg"] / res["fused"]["ms_avg"]
    return res


def host_link_bandwidth(torch, nbytes=1 << 30, reps=10):
    """Pinned H2D cudaMemcpyAsync bandwidth, best of `reps` (the H2D-fed roofline)."""
    h = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    best = None
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        d.copy_(h, non_blocking=True)
        b.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b)
        best = ms if best is None else min(best, ms)
    del h, d
    return nbytes / best / 1e6


def e2e_leg(cfg, keep, steps, chunk_mb, torch, rta):
    """Through the public host API: pinned host waveforms in, host results out."""
    d_wf, d_ped, d_gain, outs, ped, gain = keep
    h_wf = torch.empty(d_wf.shape, dtype=torch.int16, pin_memory=True)
    h_wf.copy_(d_wf)
    h_out = [torch.empty(cfg.n_traces, dtype=o.dtype, pin_memory=True) for o in outs]
    torch.cuda.synchronize()
    chunk = chunk_mb << 20

    def run():
        rta.rta_extract_host(h_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, ped, gain,
                             cfg.W, *h_out, chunk_bytes=chunk)
    for _ in range(2):
        run()
    # the host copy of the result equals the device-resident result
    ok = all(bool((ho.cuda() == o).all()) for ho, o in zip(h_out[:2], outs[:2]))
    torch.cuda.synchronize()
    k = max(3, min(steps, 10))
    before = rta.rta_launch_count()
    t0 = time.perf_counter()
    for _ in range(k):
        run()                                    # synchronous by contract
    dt = (time.perf_counter() - t0) / k
    launches = (rta.rta_launch_count() - before) // k
    del h_wf, h_out
    return {"value": cfg.input_bytes / dt / 1e9, "unit": UNIT, "ms_per_step": dt * 1e3,
            "h2d_bytes_per_step": cfg.input_bytes + 8 * cfg.n_pixels,
            "d2h_bytes_per_step": cfg.output_bytes, "steps": k, "chunk_bytes": chunk,
            "launches_per_step": launches, "matches_device_result": ok,
            "api": "rta_extract_host (pinned host in/out, double-buffered H2D, D2H on a third stream)"}


def read_stream_peak(torch, nbytes=2 << 30, reps=10):
    """A read-only stream over 2 GiB (torch.sum over float64 / int64 / float32 views: a library
    reduction, used here as a yardstick only), best of `reps`. The driver's
    MEASURED_PEAKS.json figure is a copy (half reads, half writes); the extraction
    kernels are 5:1 reads, and HBM sustains more on reads than on a 1:1 mix, so their
    fraction of the copy peak can exceed 1. This is the second denominator."""
    x = torch.empty(nbytes, dtype=torch.uint8, device="cuda").random_(0, 255)
    best, how = None, None
    # 8-byte elements read fastest (6.89 TB/s against 6.52 TB/s for float32 on this pool)
    for name, v in (("float64", x.view(torch.float64)), ("int64", x.view(torch.int64)),
                    ("float32", x.view(torch.float32))):
        for _ in range(3):
            torch.sum(v)
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            torch.sum(v)
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            if best is None or ms < best:
                best, how = ms, name
    del x
    return nbytes / best / 1e6, "torch.sum over 2 GiB as %s, best of %d (read-only stream)" % (how, reps)


def small_batch_leg(cfg, steps, peak, torch, dl0gen, rta):
    """BASELINE.json configs[0] (C1, 64 events, 7 MB): launch-latency-bound. Device time
    per launch, eager and as a CUDA-graph replay, with L2 flushed between launches
    (a 256 MB write, outside the event pair) and, for contrast, L2-resident."""
    d_wf, d_ped, d_gain, outs, _, _ = device_batch(cfg, torch, dl0gen)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    side = torch.cuda.Stream()

    def run(stream):
        rta.rta_extract(d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain, cfg.W,
                        *outs, stream=stream)
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for _ in range(LEG_WARMUP):
            run(side)
        side.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            run(side)
    torch.cuda.synchronize()

    def timed(launch, flushed):
        st = torch.cuda.current_stream()
        per = []
        for _ in range(3 + steps):
            if flushed:
                flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            launch(st)
            b.record(st)
            per.append((a, b))
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in per[3:]]
    res = {"workload": "%s: %s" % (cfg.name, cfg.label),
           "l2": "input %.1f MB fits the L2: 'flushed' rows write 256 MB between launches, "
                 "'resident' rows do not" % (cfg.input_bytes / 1e6)}
    for name, launch in (("eager", run), ("graph_replay", lambda st: graph.replay())):
        for flushed in (True, False):
            sm = summarise(cfg, timed(launch, flushed), peak)
            res["%s_%s" % (name, "flushed" if flushed else "resident")] = {
                k: sm[k] for k in ("ms_avg", "ms_median", "ms_best", "waveform_GBps",
                                   "frac_of_measured_hbm")}
    return res


def latency_leg(cfg, torch, dl0gen, rta, sizes=(1, 8, 64, 512, 4096), calls=1000):
    """What ONE call costs on small batches (the RTA works event by event
    during data taking; 30 s alert budget). Host wall time per call, p50 and
    p99 over `calls` calls, for n_events of the C2 camera: (i) rta_extract + stream
    synchronise, eager; (ii) the same launch as a CUDA-graph replay + synchronise;
    (iii) rta_extract_host, pinned host buffers in and out; (iv) rta_extract_image_host.
    The ABI is called through ctypes with the pointers prepared beforehand; `abi_call_us`
    is what an empty call (rta_launch_count) costs that way."""
    import ctypes
    import numpy as np
    L = rta.lib()
    P, S, W = cfg.n_pixels, cfg.n_samples, cfg.W
    n_max = max(sizes)
    d_wf = torch.empty((n_max, P, S), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(cfg, d_wf.data_ptr(), 0, n_max, torch.cuda.current_stream().cuda_stream)
    ped, gain = dl0gen.calib(cfg)
    x, y, nbr = dl0gen.hex_camera(P)
    tp, tb = dl0gen.IMAGE_THRESHOLDS[cfg.name]
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    outs = [torch.empty(n_max * P, dtype=dt, device="cuda")
            for dt in (torch.int32, torch.int32, torch.float32, torch.float32)]
    h_wf = torch.empty(d_wf.shape, dtype=torch.int16, pin_memory=True)
    h_wf.copy_(d_wf)
    h_out = [torch.empty(n_max * P, dtype=o.dtype, pin_memory=True) for o in outs]
    h_np, h_par = (torch.empty(n_max, dtype=torch.int32, pin_memory=True),
                   torch.empty((n_max, 8), dtype=torch.float32, pin_memory=True))
    host = [np.ascontiguousarray(a) for a in (ped, gain, x, y, nbr)]
    hp = [a.ctypes.data for a in host]
    stream = torch.cuda.Stream()
    sh = stream.cuda_stream
    sync = stream.synchronize
    o = [t.data_ptr() for t in outs]
    ho = [t.data_ptr() for t in h_out]
    torch.cuda.synchronize()

    def pct(ns):
        ns = sorted(ns)
        return {"p50_us": ns[len(ns) // 2] / 1e3, "p99_us": ns[(len(ns) * 99) // 100] / 1e3,
                "min_us": ns[0] / 1e3}

    def wall(fn, n):
        for _ in range(20):
            fn()
        t = []
        clock = time.perf_counter_ns
        for _ in range(n):
            t0 = clock()
            fn()
            t.append(clock() - t0)
        return pct(t)
    res = {"calls": calls, "camera": "%d pixels x %d samples, W=%d" % (P, S, W),
           "abi_call_us": wall(lambda: L.rta_launch_count(), calls)["p50_us"],
           "stream_sync_us": wall(sync, calls)["p50_us"]}
    for n in sizes:
        def eager():
            L.rta_extract(d_wf.data_ptr(), n, P, S, d_ped.data_ptr(), d_gain.data_ptr(), W, *o, sh)
            sync()
        with torch.cuda.stream(stream):
            eager()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=stream):
                L.rta_extract(d_wf.data_ptr(), n, P, S, d_ped.data_ptr(), d_gain.data_ptr(), W, *o, sh)

            def replay():
                graph.replay()
                sync()

            def host_call():
                L.rta_extract_host(h_wf.data_ptr(), n, P, S, hp[0], hp[1], W, *ho, 0)

            def image_host():
                L.rta_extract_image_host(h_wf.data_ptr(), n, P, S, hp[0], hp[1], W, hp[2], hp[3], hp[4],
                                         tp, tb, h_np.data_ptr(), h_par.data_ptr(), None, 0)
            k = calls if n <= 512 else max(200, calls // 5)
            res["n%d" % n] = {"input_bytes": n * P * S * 2,
                              "extract_eager": wall(eager, k), "extract_graph_replay": wall(replay, k),
                              "extract_host": wall(host_call, k), "extract_image_host": wall(image_host, k)}
            del graph
    return res


def mem_available_bytes():
    try:
        return 1024 * int([l for l in open("/proc/meminfo") if l.startswith("MemAvailable")][0].split()[1])
    except Exception:
        return 0


def bind_to_gpu_numa_node(torch, local):
    """Best effort: run this rank's host threads (and first-touch its pinned buffer)
    on the NUMA node the GPU hangs off. Returns a note for the JSON line."""
    try:
        bus = torch.cuda.get_device_properties(local).pci_bus_id
        dom = torch.cuda.get_device_properties(local).pci_domain_id
        dev = torch.cuda.get_device_properties(local).pci_device_id
        path = "/sys/bus/pci/devices/%04x:%02x:%02x.0/numa_node" % (dom, bus, dev)
        node = int(open(path).read())
        if node < 0:
            return "numa node unknown"
        cpus = set()
        for part in open("/sys/devices/system/node/node%d/cpulist" % node).read().strip().split(","):
            lo, _, hi = part.partition("-")
            cpus.update(range(int(lo), int(hi or lo) + 1))
        cpus &= os.sched_getaffinity(0)
        if cpus:
            os.sched_setaffinity(0, cpus)
            return "bound to numa node %d (%d cpus)" % (node, len(cpus))
        return "numa node %d has no allowed cpu" % node
    except Exception as ex:
        return "not bound (%s)" % type(ex).__name__


def sustained_leg(torch, dl0gen, rta, link_gbs, world=1, rank=0, dist=None, verify=True):
    """BASELINE.json:configs[4]: C5 in pinned host memory, 1 GiB chunks. At
    world > 1 every rank feeds its own GPU from its own pinned buffer (sized so
    that all ranks fit the host's memory); the aggregate is all ranks' bytes over
    the slowest rank's device time."""
    import numpy as np
    cfg = dl0gen.CONFIGS["C5"]
    ev_bytes = cfg.n_pixels * cfg.n_samples * 2
    avail = mem_available_bytes()
    n_events = cfg.n_events
    if world > 1:
        # every rank's pinned buffer plus slack must fit: at most 70 % of the host's memory in all
        n_events = int(min(cfg.n_events, 0.7 * avail / world / ev_bytes))
        n_events -= n_events % 1000
        t = torch.tensor([n_events], device="cuda", dtype=torch.int64)
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        n_events = int(t.item())
    elif avail < 44 << 30:
        return {"skipped": "needs 29.68 GB of pinned host memory; MemAvailable=%d MB" % (avail >> 20)}
    if n_events < 1000:
        return {"skipped": "host memory too small for %d ranks; MemAvailable=%d MB" % (world, avail >> 20)}
    n_traces = n_events * cfg.n_pixels
    input_bytes = n_events * ev_bytes
    t0 = time.perf_counter()
    host = torch.empty((n_events, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, pin_memory=True)
    t_alloc = time.perf_counter() - t0
    gen_ev = 10_000 if n_events % 10_000 == 0 else 1000
    stage = torch.empty((gen_ev, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    first = rank * n_events                        # every rank streams its own events of C5's model
    for e0 in range(0, n_events, gen_ev):
        dl0gen.events_cuda(cfg, stage.data_ptr(), first + e0, gen_ev, st)
        host[e0:e0 + gen_ev].copy_(stage)
    torch.cuda.synchronize()
    del stage
    ped, gain = dl0gen.calib(cfg)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    outs = [torch.full((n_traces,), f, dtype=dt, device="cuda") for f, dt in
            ((-7, torch.int32), (-7, torch.int32), (-7.0, torch.float32), (-7.0, torch.float32))]
    stream = torch.cuda.current_stream()

    def timed(run, reps=2):
        """device time (CUDA events on the compute stream, which every chunk's kernel and
        therefore every copy is ordered into) and host wall time; best of `reps`; with
        several ranks the MAX over ranks of each repetition"""
        best = None
        for _ in range(reps):
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
                torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            a.record(stream)
            run()
            b.record(stream)
            torch.cuda.synchronize()
            wall = time.perf_counter() - t0
            dev = a.elapsed_time(b) / 1e3
            if dist is not None:
                t = torch.tensor([dev, wall], device="cuda", dtype=torch.float64)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                dev, wall = float(t[0]), float(t[1])
            if best is None or dev < best[0]:
                best = (dev, wall)
        return best

    def run():
        rta.rta_extract_stream(host, n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain,
                               cfg.W, *outs, chunk_bytes=1 << 30, stream=stream)
    run()                                        # warm-up: allocates the workspace
    torch.cuda.synchronize()
    before = rta.rta_launch_count()
    dt, wall = timed(run)
    launches = (rta.rta_launch_count() - before) // 2
    val = world * input_bytes / dt / 1e9
    res = {"workload": "%s: %s" % (cfg.name, cfg.label) + ("" if n_events == cfg.n_events else
                                                         " (%d events per rank)" % n_events),
           "value": val, "unit": UNIT, "ranks": world,
           "seconds": dt, "seconds_wall": wall, "timing": "CUDA events on the compute stream, max over ranks",
           "traces_per_s": world * n_traces / dt, "chunk_bytes": 1 << 30,
           "chunks": launches, "h2d_bytes": world * input_bytes,
           "host_link_GBps_measured": link_gbs, "frac_of_host_link": val / world / link_gbs,
           "paper_array_rate_GBps": list(PAPER_RATE_GBS),
           "x_paper_max_rate": val / PAPER_RATE_GBS[1],
           "pinned_alloc_s": t_alloc, "outputs": "stay on device (%.2f GB per rank)" % (16e-9 * n_traces)}
    if world > 1:                              # the single-rank extras below are N = 1 diagnostics
        del host, outs
        rta.rta_shutdown()
        return res

    h = host.numpy().view(np.uint16)
    if verify:
        # every one of the 200 000 events against the oracle, on the pinned buffer's own bytes
        # (chunk-sized slabs, all host cores): the full-size verification pass of SURVEY.md 8(d)
        import oracle
        cores = os.cpu_count() or 1
        t0 = time.perf_counter()
        ok, done = True, 0
        for e0, k in event_slabs(n_events, ev_bytes):
            want = oracle.extract_threads(h[e0:e0 + k], ped, gain, cfg.W, cores)
            ok = ok and bits_equal(torch, outs, want, e0 * cfg.n_pixels, (e0 + k) * cfg.n_pixels)
            done += k
        tv = time.perf_counter() - t0
        res["verified_events"] = done
        res["all_outputs_bit_identical_to_oracle"] = ok
        res["verify_seconds"] = tv
        res["oracle_all_cores_GBps_incl_compare"] = input_bytes / tv / 1e9
    # the same stream from PAGEABLE host memory (PAPER.md:133 is a page-locked-versus-not
    # transfer test): the first 8 GiB of the buffer copied into ordinary memory
    try:
        n_pg = min(n_events, 8 * ((1 << 30) // ev_bytes))
        pg = np.empty((n_pg, cfg.n_pixels, cfg.n_samples), np.int16)
        pg[...] = host[:n_pg].numpy()
        pg_outs = [torch.empty(n_pg * cfg.n_pixels, dtype=o.dtype, device="cuda") for o in outs]

        def run_pg():
            rta.rta_extract_stream(pg, n_pg, cfg.n_pixels, cfg.n_samples, d_ped, d_gain, cfg.W,
                                   *pg_outs, chunk_bytes=1 << 30, stream=stream)
        run_pg()
        torch.cuda.synchronize()
        same = all(bool((a == b[:a.numel()]).all()) for a, b in zip(pg_outs[:2], outs[:2]))
        dtp, _ = timed(run_pg)
        res["pageable"] = {"value": pg.nbytes / dtp / 1e9, "unit": UNIT, "seconds": dtp,
                           "h2d_bytes": pg.nbytes, "events": n_pg,
                           "frac_of_host_link": pg.nbytes / dtp / 1e9 / link_gbs,
                           "source": "pageable numpy array (staged through library-owned pinned buffers)",
                           "equals_pinned_result": same}
        del pg, pg_outs
    except Exception as ex:
        res["pageable"] = {"error": repr(ex)}
    # NEXT-4: the same pinned buffer through rta_extract_image_stream: waveforms in at
    # link speed, 36 bytes of event parameters per event out (they stay on the device)
    try:
        cam = camera_on_device(cfg, torch, dl0gen)
        n_pix = torch.empty(n_events, dtype=torch.int32, device="cuda")
        par = torch.empty((n_events, 8), dtype=torch.float32, device="cuda")

        def run_img():
            rta.rta_extract_image_stream(host, n_events, cfg.n_pixels, cfg.n_samples, d_ped,
                                         d_gain, cfg.W, *cam, n_pix, par, None,
                                         chunk_bytes=1 << 30, stream=stream)
        run_img()
        torch.cuda.synchronize()
        # every event again from the (verified) per-trace outputs of the uint16 leg above
        n_all = torch.empty(n_events, dtype=torch.int32, device="cuda")
        p_all = torch.empty((n_events, 8), dtype=torch.float32, device="cuda")
        rta.rta_image_moments(outs[2], outs[3], n_events, cfg.n_pixels, *cam, n_all, p_all, None,
                              stream=stream)
        torch.cuda.synchronize()
        same_img = bool((n_pix == n_all).all()) and bool(
            (par.view(torch.int32) == p_all.view(torch.int32)).all())
        dti, _ = timed(run_img)
        res["image"] = {
            "value": input_bytes / dti / 1e9, "unit": UNIT, "seconds": dti,
            "api": "rta_extract_image_stream (extraction + cleaning + moments in one kernel per chunk)",
            "events_per_s": n_events / dti, "frac_of_host_link": input_bytes / dti / 1e9 / link_gbs,
            "result_bytes": EVENT_OUT_BYTES * n_events,
            "mean_pixels_in_image": float(n_pix.float().mean()),
            "all_events_equal_extract_then_moments": same_img}
        del n_pix, par, n_all, p_all
    except Exception as ex:
        res["image"] = {"error": repr(ex)}
    # NEXT-2: the same 200 000 events as a P12 stream (22.26 GB) in the same pinned
    # buffer, through rta_extract_stream_packed12 (chunks of 9644 events = 1.07 GB)
    try:
        ev_samples = cfg.n_pixels * cfg.n_samples
        nb = dl0gen.packed12_nbytes(n_traces * cfg.n_samples)
        hp = host.view(-1).view(torch.uint8)[:nb]
        stage = torch.empty((gen_ev, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, device="cuda")
        stage_pk = torch.empty(gen_ev * ev_samples * 3 // 2, dtype=torch.uint8, device="cuda")
        for e0 in range(0, n_events, gen_ev):
            dl0gen.events_cuda(cfg, stage.data_ptr(), e0, gen_ev, st)
            dl0gen.pack12_cuda(stage.data_ptr(), gen_ev * ev_samples, stage_pk.data_ptr(), st)
            b0 = e0 * ev_samples * 3 // 2
            hp[b0:b0 + stage_pk.numel()].copy_(stage_pk)
        torch.cuda.synchronize()
        del stage, stage_pk
        want = [o.clone() for o in outs]          # the (verified) uint16-path result, every trace
        for o in outs:
            o.zero_()

        def run12():
            rta.rta_extract_stream_packed12(hp, n_events, cfg.n_pixels, cfg.n_samples, d_ped,
                                            d_gain, cfg.W, *outs, chunk_bytes=1 << 30, stream=stream)
        run12()
        torch.cuda.synchronize()
        same = all(bool((o.view(torch.int32) == w.view(torch.int32)).all()) for o, w in zip(outs, want))
        del want
        before = rta.rta_launch_count()
        dt12, _ = timed(run12)
        res["packed12"] = {
            "value": input_bytes / dt12 / 1e9, "unit": UNIT,
            "meaning": "raw-waveform-equivalent GB/s (2 bytes per sample) of the same 200000 events",
            "seconds": dt12, "h2d_bytes": nb, "link_GBps": nb / dt12 / 1e9,
            "frac_of_host_link": nb / dt12 / 1e9 / link_gbs,
            "chunks": (rta.rta_launch_count() - before) // 2,
            "chunk_events": rta.rta_chunk_events(n_events, cfg.n_pixels, cfg.n_samples, 1 << 30, 12),
            "traces_per_s": n_traces / dt12, "x_paper_max_rate": input_bytes / dt12 / 1e9 / PAPER_RATE_GBS[1],
            "speedup_vs_uint16_feed": dt / dt12,
            "all_events_equal_uint16_path": same}
    except Exception as ex:  # the uint16 leg above stands on its own
        res["packed12"] = {"error": repr(ex)}
    del host, outs
    rta.rta_shutdown()
    return res


def cpu_baseline_leg(cfg, keep, dl0gen, torch):
    """The oracle, as it stands, on this box's host cores, on the same bytes the
    GPU extracted: all cores on `oracle_sample_events` events (the whole batch
    for C2: the timing run doubles as the verification pass), one thread on an
    eighth of that. Every event of the batch is then compared with the device
    result (the events beyond the timed sample in untimed slabs)."""
    import numpy as np
    import oracle
    d_wf, _, _, outs, ped, gain = keep
    cores = os.cpu_count() or 1
    ev_bytes = cfg.n_pixels * cfg.n_samples * 2
    n_ev = oracle_sample_events(cfg)
    wf = d_wf[:n_ev].cpu().numpy().view(np.uint16)
    t0 = time.perf_counter()
    rn = oracle.extract_threads(wf, ped, gain, cfg.W, cores)
    tn = time.perf_counter() - t0
    n1 = max(1, n_ev // 8)
    t0 = time.perf_counter()
    oracle.extract(wf[:n1], ped, gain, cfg.W)
    t1 = time.perf_counter() - t0
    n = n_ev * cfg.n_pixels
    ints_equal = bits_equal(torch, outs[:2], rn[:2], 0, n)
    floats_equal = bits_equal(torch, outs[2:], rn[2:], 0, n)
    verified = n_ev
    del wf, rn
    for e0, k in event_slabs(cfg.n_events - n_ev, ev_bytes):      # the rest of the batch, untimed
        e0 += n_ev
        w = d_wf[e0:e0 + k].cpu().numpy().view(np.uint16)
        r = oracle.extract_threads(w, ped, gain, cfg.W, cores)
        lo, hi = e0 * cfg.n_pixels, (e0 + k) * cfg.n_pixels
        ints_equal = ints_equal and bits_equal(torch, outs[:2], r[:2], lo, hi)
        floats_equal = floats_equal and bits_equal(torch, outs[2:], r[2:], lo, hi)
        verified += k
    return {"value": n_ev * ev_bytes / tn / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "first %d of %d events of %s (%.2f GB), same bytes as the GPU run"
                      % (n_ev, cfg.n_events, cfg.name, n_ev * ev_bytes / 1e9),
            "seconds": tn,
            "single_thread_value": n1 * ev_bytes / t1 / 1e9,
            "single_thread_sample": "first %d events" % n1,
            "traces_per_s": n / tn, "single_thread_traces_per_s": n1 * cfg.n_pixels / t1,
            "verified_events": verified, "n_events": cfg.n_events,
            "gpu_matches_oracle_on_every_event": {"ints_bit_exact": ints_equal,
                                                  "floats_bit_exact": floats_equal}}


def compact_summary(out):
    """Every leg as [ms per launch, fraction of the measured HBM copy peak] (host-fed legs:
    [GB/s, fraction of the measured host link]; latency: p50 microseconds per call), short
    enough to survive in the tail of the line. `cap` lists the legs during which the driver
    reported sw_power_cap."""
    r3 = lambda v: None if v is None else round(float(v), 3)
    pair = lambda d: [round(d["ms_avg"], 4), r3(d.get("frac_of_measured_hbm"))]
    sm = {"main": [round(out["roofline"]["avg_launch_ms"], 4), r3(out["roofline"]["frac"]),
                   r3(out["roofline"].get("frac_of_read_stream_peak"))]}
    for name, d in out.get("configs", {}).items():
        if name == "C1":
            sm["C1"] = {k.replace("_flushed", "_fl").replace("_resident", "_l2"): pair(v)
                        for k, v in d.items() if isinstance(v, dict)}
        else:
            sm[name] = pair(d)
    for leg in ("family", "packed12"):
        for name, d in out.get(leg, {}).items():
            if leg == "family":
                sm["fam." + name] = {k: pair(v) for k, v in d.items()}
            else:
                sm["p12." + name] = pair(d)
    for name, d in out.get("image", {}).items():
        peak = out["roofline"]["peak"]
        sm["img." + name] = {k: [round(d[k]["ms_avg"], 4), r3(d[k].get("frac_of_measured_hbm"))]
                             for k in ("fused", "moments", "two_calls") if k in d}
    if "ragged" in out:
        sm["ragged"] = pair(out["ragged"])
        if "unspecialised" in out["ragged"]:
            sm["ragged.unspec"] = pair(out["ragged"]["unspecialised"])
    for name, d in out.get("any_shape", {}).items():
        if isinstance(d, dict) and "staged_any" in d:
            sm["any." + name] = pair(d["staged_any"])
    e = out.get("e2e", {})
    if e.get("value") is not None:
        sm["e2e"] = [r3(e["value"]), r3(e.get("frac_of_host_link"))]
    su = out.get("sustained", {})
    if su:
        sm["sus"] = [r3(su["value"]), r3(su.get("frac_of_host_link"))]
        for k in ("pageable", "image", "packed12"):
            if k in su:
                sm["sus." + k] = [r3(su[k]["value"]), r3(su[k].get("frac_of_host_link"))]
    lat = out.get("latency", {})
    for k, d in lat.items():
        if k.startswith("n") and isinstance(d, dict):
            sm["lat." + k] = [round(d[m]["p50_us"], 1) for m in
                              ("extract_eager", "extract_graph_replay", "extract_host", "extract_image_host")]
    sm["cap"] = sorted(k for k, c in out.get("leg_clocks", {}).items() if c.get("sw_power_cap"))
    return sm


def multi_rank_command(n_gpus, argv):
    """The command `python bench.py --gpus N` re-executes itself as when no
    torchrun environment is present (rendezvous on 127.0.0.1: the container's
    hostname may not resolve)."""
    return [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1",
            "--nproc-per-node", str(int(n_gpus)), "--local-addr", "127.0.0.1",
            os.path.join(ROOT, "bench.py")] + list(argv)


def main():
    args = parse_args()
    if args.impl == "reference":
        return reference_arm(args)

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: one rank per GPU under torchrun, same arguments
        return subprocess.call(multi_rank_command(args.gpus, sys.argv[1:]))

    import torch
    import dl0gen
    import paper_1307_6489_b200 as rta

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    numa = None
    if world > 1:
        import torch.distributed as dist
        numa = bind_to_gpu_numa_node(torch, local)      # before any pinned allocation
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    rta.lib()
    cfg = workload(args.workload, dl0gen)
    peak, peak_src = hbm_peak()

    try:
        uuid = str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid)
    sampler.start()
    # Weak scaling: every rank extracts its own batch of the named workload
    # (independent events; no data-path collective).
    fmt = args.input_format
    if (fmt == "p12" or args.path != "extract" or args.workload.startswith("X")
            or args.extractor != "sliding"):
        args.no_extra = True     # the packed / image / family main legs are profiling/diagnostic runs
    if args.extractor != "sliding" and (fmt != "u16" or args.path != "extract"):
        raise SystemExit("--extractor goes with --path extract --input-format u16")
    main_run = kernel_only(cfg, args.steps, args.warmup, torch, dl0gen, rta, barrier, sampler, fmt,
                           args.path, args.extractor)
    clocks = sampler.stop(*main_run["marks"])
    t_local = sum(main_run["per_launch_ms"])
    t_max = t_local
    if dist is not None:
        t = torch.tensor([t_local], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_max = float(t.item())
    ms_per_step = t_max / args.steps
    value = world * cfg.input_bytes / ms_per_step / 1e6
    summ = summarise(cfg, main_run["per_launch_ms"], peak)
    algo_bytes = cfg.input_bytes + cfg.output_bytes
    kname = rta.rta_kernel_name(cfg.n_samples, cfg.W, True)
    bytes_per_trace = 2 * cfg.n_samples + ALGO_BYTES_PER_TRACE_OUT
    if fmt == "p12":
        # same value definition (2 bytes per sample extracted); the roofline counts the packed bytes
        algo_bytes = dl0gen.packed12_nbytes(cfg.n_traces * cfg.n_samples) + cfg.output_bytes
        kname = rta.rta_kernel_name_packed12(cfg.n_samples, cfg.W, True)
        bytes_per_trace = 1.5 * cfg.n_samples + ALGO_BYTES_PER_TRACE_OUT
        avg = summ["ms_avg"]
        summ["algorithmic_GBps"] = algo_bytes / avg / 1e6
        summ["frac_of_measured_hbm"] = algo_bytes / avg / 1e6 / peak
        summ["frac_of_nominal_8TBps"] = algo_bytes / avg / 1e6 / 8000.0
    if args.extractor != "sliding":
        kname = "%s:%s" % (args.extractor, kname)
        per_trace, _ = (fixed_gather_bytes_per_trace(cfg, main_run["fixed_start"])
                        if args.extractor == "fixed" else (None, None))
        if per_trace is not None:     # the gathering route: sectors touched, not whole traces
            kname = "fixed:gather(generic)"
            bytes_per_trace = per_trace
            algo_bytes = per_trace * cfg.n_traces
            avg = summ["ms_avg"]
            summ["algorithmic_GBps"] = algo_bytes / avg / 1e6
            summ["frac_of_measured_hbm"] = algo_bytes / avg / 1e6 / peak
            summ["frac_of_nominal_8TBps"] = algo_bytes / avg / 1e6 / 8000.0
    if args.path != "extract":
        ev_bytes = EVENT_OUT_BYTES * cfg.n_events
        if args.path == "image":
            algo_bytes = cfg.input_bytes + ev_bytes
            kname = rta.rta_image_kernel_name(cfg.n_pixels, cfg.n_samples, cfg.W, True)
            bytes_per_trace = 2 * cfg.n_samples + EVENT_OUT_BYTES / cfg.n_pixels
        else:
            # the charge row is read once; peak times are gathered for the mask pixels only
            algo_bytes = 4 * cfg.n_traces + ev_bytes
            kname = "image_moments:%s" % cfg.name      # its DRAM traffic depends on the camera
            bytes_per_trace = 4 + EVENT_OUT_BYTES / cfg.n_pixels
        avg = summ["ms_avg"]
        summ["algorithmic_GBps"] = algo_bytes / avg / 1e6
        summ["frac_of_measured_hbm"] = algo_bytes / avg / 1e6 / peak
        summ["frac_of_nominal_8TBps"] = algo_bytes / avg / 1e6 / 8000.0
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {
            "workload": "%s: %s" % (cfg.name, cfg.label) + (" as a P12 stream" if fmt == "p12" else "")
                        + ("" if args.extractor == "sliding" else " through rta_extract_" + args.extractor)
                        + {"extract": "", "image": " through rta_extract_image",
                           "moments": " charges through rta_image_moments"}[args.path],
            "per_gpu": "%d events x %d pixels x %d samples uint16, W=%d" % (
                cfg.n_events, cfg.n_pixels, cfg.n_samples, cfg.W),
            "l2": "input %.2f GB per step exceeds the 126 MB L2 (no flush needed)" % (cfg.input_bytes / 1e9),
            "parallelism": "independent events per GPU, no collective",
            "seed": cfg.seed, "input_checksum": main_run["checksum_first_64Mi_samples"],
        },
        "traces_per_s": world * cfg.n_traces / ms_per_step * 1e3,
        "pct_of_measured_hbm": 100.0 * summ["frac_of_measured_hbm"],
        "gpu_launches": main_run["launches"],
        "clocks": clocks,
        "roofline": {
            "bound": "hbm", "kernel": kname,
            "achieved": summ["algorithmic_GBps"], "peak": peak, "unit": "GB/s",
            "frac": summ["frac_of_measured_hbm"], "peak_source": peak_src,
            "algorithmic_bytes_per_launch": algo_bytes,
            "bytes_per_trace": bytes_per_trace,
            "avg_launch_ms": summ["ms_avg"],
            "frac_of_nominal_8TBps": summ["frac_of_nominal_8TBps"],
        },
    }
    traffic, t_commit, t_stale = ncu_traffic(kname)
    out["roofline"]["traffic"] = traffic
    out["roofline"]["traffic_commit"] = t_commit
    out["roofline"]["traffic_source"] = (
        "no capture" if t_commit is None else
        "null: csrc changed since the ncu capture of that commit" if t_stale else
        "ncu --set full dram__bytes_read.sum + dram__bytes_write.sum per launch, captured at that "
        "commit with the same kernel sources (profiles/)")
    if numa is not None:
        out["config"]["host_affinity"] = numa

    if not args.no_extra:
        # host-fed leg on every rank (each GPU has its own host link); max over ranks
        keep = main_run["keep"]
        barrier()
        e2e = e2e_leg(cfg, keep, args.steps, args.e2e_chunk_mb, torch, rta)
        if dist is not None:
            t = torch.tensor([e2e["ms_per_step"]], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e["ms_per_step"] = float(t.item())
            e2e["value"] = world * cfg.input_bytes / e2e["ms_per_step"] / 1e6
            e2e["h2d_bytes_per_step"] *= world
            e2e["d2h_bytes_per_step"] *= world
        out["e2e"] = e2e
        if world > 1 and not args.no_sustained:
            # the host-fed number is the one that scales with the GPU count (one host link
            # per GPU) until host memory bandwidth saturates: every rank feeds its own GPU
            main_run["keep"] = keep = None
            torch.cuda.empty_cache()
            link = host_link_bandwidth(torch)
            t = torch.tensor([link], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MIN)
            out["sustained"] = sustained_leg(torch, dl0gen, rta, float(t.item()), world, rank, dist)
        if rank == 0 and world == 1:
            if not args.no_cpu:
                out["cpu_baseline"] = cpu_baseline_leg(cfg, keep, dl0gen, torch)
            main_run["keep"] = keep = None
            torch.cuda.empty_cache()
            legs = set(SECONDARY_LEGS if args.legs == "all" else
                       [x for x in args.legs.split(",") if x])
            leg_sampler = ClockSampler(local, uuid)
            leg_sampler.start()
            leg_clocks = {}

            def timed_leg(name, fn):
                lo = leg_sampler.mark()
                r = fn()
                c = leg_sampler.window(lo, leg_sampler.mark())
                if c:
                    leg_clocks[name] = c
                return r
            if legs - set(SECONDARY_LEGS):
                raise SystemExit("--legs: unknown leg(s) %s" % sorted(legs - set(SECONDARY_LEGS)))
            others = {}
            for name in ("C3", "C4"):
                if name == cfg.name or "configs" not in legs:
                    continue
                c = dl0gen.CONFIGS[name]
                r = kernel_only(c, max(10, args.steps // 2), 3, torch, dl0gen, rta)
                others[name] = summarise(c, r["per_launch_ms"], peak)
                r = None
                torch.cuda.empty_cache()
            if "configs" in legs:
                # C1 is configs[0]: the small case, bound by launch latency, not by HBM
                others["C1"] = small_batch_leg(dl0gen.CONFIGS["C1"], max(20, args.steps), peak,
                                               torch, dl0gen, rta)
                out["configs"] = others
            if "latency" in legs:
                out["latency"] = latency_leg(dl0gen.CONFIGS["C2"], torch, dl0gen, rta)
                torch.cuda.empty_cache()
            fam = {}
            for name in ("C2", "C3", "C4") if "family" in legs else ():
                fam[name] = family_leg(dl0gen.CONFIGS[name], max(10, args.steps // 4), peak,
                                       torch, dl0gen, rta)
                torch.cuda.empty_cache()
            if fam:
                out["family"] = fam
            pk = {}
            for name in ("C2", "C3", "C4") if "packed12" in legs else ():
                pk[name] = timed_leg("packed12." + name, lambda: packed_leg(
                    dl0gen.CONFIGS[name], max(10, args.steps // 4), peak, torch, dl0gen, rta))
                torch.cuda.empty_cache()
            if pk:
                out["packed12"] = pk
            if "any_shape" in legs:
                out["any_shape"] = any_shape_leg(max(10, args.steps // 4), peak, torch, dl0gen, rta)
                torch.cuda.empty_cache()
            if "ragged" in legs:
                out["ragged"] = ragged_leg(max(10, args.steps // 4), peak, torch, dl0gen, rta)
                torch.cuda.empty_cache()
                xs = extra_shapes(dl0gen)      # cameras without a specialised kernel: extract_ragged_dyn_kernel
                out["ragged"]["unspecialised"] = ragged_leg(
                    max(10, args.steps // 4), peak, torch, dl0gen, rta, n_events=1000,
                    slots=((xs["X60"], 6), (xs["X96"], 6)), label="6 x 1855x60 W7 + 6 x 2048x96 W8")
                torch.cuda.empty_cache()
            img = {}
            for name in ("C2", "C3", "C4") if "image" in legs else ():
                img[name] = timed_leg("image." + name, lambda: image_leg(
                    dl0gen.CONFIGS[name], max(10, args.steps // 4), peak, torch, dl0gen, rta))
                torch.cuda.empty_cache()
            if img:
                out["image"] = img
            rs_peak, rs_how = read_stream_peak(torch)
            r = out["roofline"]
            r["read_stream_peak"] = rs_peak
            r["read_stream_peak_source"] = rs_how
            r["frac_of_read_stream_peak"] = r["achieved"] / rs_peak
            r["note"] = ("`peak` is the driver's copy figure (1:1 reads and writes); this kernel is 5:1 "
                         "reads, which HBM serves faster, so `frac` can pass 1; frac_of_read_stream_peak "
                         "divides by a read-only stream measured in this run")
            leg_sampler.stop()
            if leg_clocks:
                out["leg_clocks"] = leg_clocks   # whole leg (set-up included): sm clock, peak power
            link = host_link_bandwidth(torch)
            out["e2e"]["host_link_GBps_measured"] = link
            out["e2e"]["frac_of_host_link"] = out["e2e"]["value"] / link
            if not args.no_sustained:
                out["sustained"] = sustained_leg(torch, dl0gen, rta, link)
    else:
        out["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0,
                      "d2h_bytes_per_step": 0, "note": "skipped by --no-extra"}
    if rank == 0:
        if world == 1 and not args.no_extra:
            out["summary"] = compact_summary(out)   # last key: the tail of the line carries every leg
        print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
