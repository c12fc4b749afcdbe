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
  configs       kernel-only numbers for the other single-GPU configs (C3, C4)
  family        the other extractors (NEXT-1) on the same batches
  packed12      NEXT-2: the same batches as P12 streams (12 bits per sample),
                decoded inside the extraction kernel; sustained.packed12 is C5
                fed as 22.26 GB of P12 through rta_extract_stream_packed12
  ragged        NEXT-3: a mixed-camera array through rta_extract_ragged
  image         NEXT-4: rta_extract_image (extraction + cleaning + moments in one
                kernel) next to rta_extract followed by rta_image_moments;
                sustained.image is C5 through rta_extract_image_stream
  any_shape     shapes without a specialised kernel (not BASELINE configs) through
                the staged kernel with runtime (n_samples, W), next to the generic one
Secondary legs are single-GPU diagnostics (N = 1 only) and run ten untimed launches first.
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
                    choices=["C1", "C2", "C3", "C4", "X60", "X40w5", "X96", "X128w10"],
                    help="C1..C4: BASELINE.json configs; X*: shapes without a specialised kernel "
                         "(diagnostic runs of the runtime-shape kernel, imply --no-extra)")
    ap.add_argument("--input-format", default="u16", choices=["u16", "p12"],
                    help="u16: BASELINE.json's uint16 waveforms (the headline); p12: the same batch as "
                         "a packed 12-bit stream through rta_extract_packed12 (NEXT-2)")
    ap.add_argument("--path", default="extract", choices=["extract", "image", "moments"],
                    help="main leg: rta_extract (default, the BASELINE metric); 'image' = "
                         "rta_extract_image, 'moments' = rta_image_moments (diagnostic runs "
                         "for profiling, imply --no-extra)")
    ap.add_argument("--no-extra", action="store_true", help="skip configs/e2e/sustained/cpu legs")
    ap.add_argument("--no-sustained", action="store_true", help="skip the 29.68 GB C5 leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--e2e-chunk-mb", type=int, default=64)
    return ap.parse_args()


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(name):
    """DRAM bytes per launch from the committed ncu --set full capture, if any."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(name)
    except Exception:
        return None


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
                self.samples.append((mhz, mask))
            except Exception:
                pass
            time.sleep(0.001)

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def mark(self):
        """Number of samples so far: bracket the timed region with two marks."""
        return len(self.samples) if self.nvml else len(self.lines)

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
            reasons = sorted(k for k, b in bits.items() if any(m & b for _, m in sel))
            sm = [x for x, _ in sel]
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
    # ~0.3 GB/s per core: size the per-step sample for about 1 s of all-cores work
    n_ev = max(cores, min(cfg.n_events, 200 * cores))
    wf = dl0gen.events_cpu(cfg, 0, n_ev, threads=cores)
    for _ in range(max(1, min(args.warmup, 2))):
        oracle.extract_threads(wf, ped, gain, cfg.W, cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.extract_threads(wf, ped, gain, cfg.W, cores)
    dt = (time.perf_counter() - t0) / args.steps
    val = wf.nbytes / dt / 1e9
    sample = "first %d of %d events of %s per step, %d threads" % (n_ev, cfg.n_events, cfg.name, cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
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


def kernel_only(cfg, steps, warmup, torch, dl0gen, rta, barrier=None, sampler=None, fmt="u16",
                path="extract"):
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
            "marks": (m0, m1),
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
    start = torch.from_numpy(np.random.default_rng(cfg.seed).integers(
        0, cfg.n_samples - cfg.W + 1, cfg.n_pixels).astype(np.int32)).cuda()
    taps = [1, 2, 3, 4, 3, 2, 1, 1][:cfg.W]
    base = (d_wf, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain)
    runs = {
        "fixed": lambda: rta.rta_extract_fixed(*base, cfg.W, start, *outs, stream=stream),
        "local_peak": lambda: rta.rta_extract_local_peak(*base, cfg.W, cfg.W // 2, *outs, stream=stream),
        "fir": lambda: rta.rta_extract_fir(*base, taps, *outs, stream=stream),
    }
    res = {}
    for name, run in runs.items():
        for _ in range(LEG_WARMUP):
            run()
        torch.cuda.synchronize()
        res[name] = summarise(cfg, time_steps(run, steps, stream), peak)
    res["fir"]["taps"] = taps
    res["fixed"]["note"] = ("reads W samples per trace; traces longer than 96 bytes are gathered from global "
                            "memory instead of streamed, so GB/s figures (which count the whole waveform) can "
                            "exceed the HBM peak")
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


def ragged_leg(steps, peak, torch, dl0gen, rta, n_events=1000):
    """NEXT-3: a mixed-camera array (4 LST-, 10 MST-, 6 SST-like telescopes, the
    cameras of C2/C3/C4), every event holding one block per telescope, through
    one rta_extract_ragged call (one launch per camera shape)."""
    m = dl0gen.MixedArray(n_events=n_events)
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
    res = {"workload": "mixed array: %d events x (4 x 1855x40 W7 + 10 x 1764x25 W4 + 6 x 2048x128 W8), "
                       "%d blocks on 16-byte boundaries" % (m.n_events, len(m.blk_tel)),
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
                                  n_events=10_000, W=10)]
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


def sustained_leg(torch, dl0gen, rta, link_gbs):
    """BASELINE.json:configs[4]: C5 in pinned host memory, 1 GiB chunks."""
    cfg = dl0gen.CONFIGS["C5"]
    try:
        avail_kb = int([l for l in open("/proc/meminfo") if l.startswith("MemAvailable")][0].split()[1])
    except Exception:
        avail_kb = 0
    if avail_kb < 44 * 1024 * 1024:
        return {"skipped": "needs 29.68 GB of pinned host memory; MemAvailable=%d MB" % (avail_kb // 1024)}
    t0 = time.perf_counter()
    host = torch.empty((cfg.n_events, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, pin_memory=True)
    t_alloc = time.perf_counter() - t0
    gen_ev = 10_000
    stage = torch.empty((gen_ev, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    for e0 in range(0, cfg.n_events, gen_ev):
        dl0gen.events_cuda(cfg, stage.data_ptr(), e0, gen_ev, st)
        host[e0:e0 + gen_ev].copy_(stage)
    torch.cuda.synchronize()
    del stage
    ped, gain = dl0gen.calib(cfg)
    d_ped, d_gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()
    outs = [torch.empty(cfg.n_traces, dtype=dt, device="cuda")
            for dt in (torch.int32, torch.int32, torch.float32, torch.float32)]
    stream = torch.cuda.current_stream()

    def run():
        rta.rta_extract_stream(host, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped, d_gain,
                               cfg.W, *outs, chunk_bytes=1 << 30, stream=stream)
    run()                                        # warm-up: allocates the workspace
    torch.cuda.synchronize()
    times = []
    before = rta.rta_launch_count()
    for _ in range(2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()                 # first cudaMemcpyAsync issue ...
        run()
        torch.cuda.synchronize()                 # ... to completion of the last kernel
        times.append(time.perf_counter() - t0)
    launches = (rta.rta_launch_count() - before) // 2
    dt = min(times)
    val = cfg.input_bytes / dt / 1e9
    res = {"workload": "%s: %s" % (cfg.name, cfg.label), "value": val, "unit": UNIT,
           "seconds": dt, "traces_per_s": cfg.n_traces / dt, "chunk_bytes": 1 << 30,
           "chunks": launches, "h2d_bytes": cfg.input_bytes,
           "host_link_GBps_measured": link_gbs, "frac_of_host_link": val / link_gbs,
           "paper_array_rate_GBps": list(PAPER_RATE_GBS),
           "x_paper_max_rate": val / PAPER_RATE_GBS[1],
           "pinned_alloc_s": t_alloc, "outputs": "stay on device (5.94 GB)"}
    # NEXT-4: the same pinned buffer through rta_extract_image_stream: waveforms in at
    # link speed, 36 bytes of event parameters per event out (they stay on the device)
    try:
        cam = camera_on_device(cfg, torch, dl0gen)
        n_pix = torch.empty(cfg.n_events, dtype=torch.int32, device="cuda")
        par = torch.empty((cfg.n_events, 8), dtype=torch.float32, device="cuda")

        def run_img():
            rta.rta_extract_image_stream(host, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped,
                                         d_gain, cfg.W, *cam, n_pix, par, None,
                                         chunk_bytes=1 << 30, stream=stream)
        run_img()
        torch.cuda.synchronize()
        # the first events again from the per-trace outputs of the uint16 leg above
        n64, p64 = image_outputs(dl0gen.CONFIGS["C1"], torch)            # 64 events
        rta.rta_image_moments(outs[2], outs[3], 64, cfg.n_pixels, *cam, n64, p64, None, stream=stream)
        torch.cuda.synchronize()
        same_img = bool((n_pix[:64] == n64).all()) and bool(
            (par[:64].view(torch.int32) == p64.view(torch.int32)).all())
        times = []
        for _ in range(2):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            run_img()
            torch.cuda.synchronize()
            times.append(time.perf_counter() - t0)
        dti = min(times)
        res["image"] = {
            "value": cfg.input_bytes / dti / 1e9, "unit": UNIT, "seconds": dti,
            "api": "rta_extract_image_stream (extraction + cleaning + moments in one kernel per chunk)",
            "events_per_s": cfg.n_events / dti, "frac_of_host_link": cfg.input_bytes / dti / 1e9 / link_gbs,
            "result_bytes": EVENT_OUT_BYTES * cfg.n_events,
            "mean_pixels_in_image": float(n_pix.float().mean()),
            "first_64_events_equal_extract_then_moments": same_img}
        del n_pix, par
    except Exception as ex:
        res["image"] = {"error": repr(ex)}
    # NEXT-2: the same 200 000 events as a P12 stream (22.26 GB) in the same pinned
    # buffer, through rta_extract_stream_packed12 (chunks of 9644 events = 1.07 GB)
    try:
        ev_samples = cfg.n_pixels * cfg.n_samples
        nb = dl0gen.packed12_nbytes(cfg.n_traces * cfg.n_samples)
        hp = host.view(-1).view(torch.uint8)[:nb]
        stage = torch.empty((gen_ev, cfg.n_pixels, cfg.n_samples), dtype=torch.int16, device="cuda")
        stage_pk = torch.empty(gen_ev * ev_samples * 3 // 2, dtype=torch.uint8, device="cuda")
        for e0 in range(0, cfg.n_events, gen_ev):
            dl0gen.events_cuda(cfg, stage.data_ptr(), e0, gen_ev, st)
            dl0gen.pack12_cuda(stage.data_ptr(), gen_ev * ev_samples, stage_pk.data_ptr(), st)
            b0 = e0 * ev_samples * 3 // 2
            hp[b0:b0 + stage_pk.numel()].copy_(stage_pk)
        torch.cuda.synchronize()
        del stage, stage_pk
        want = [o[:64 * cfg.n_pixels].clone() for o in outs]     # uint16-path result, first events
        for o in outs:
            o.zero_()

        def run12():
            rta.rta_extract_stream_packed12(hp, cfg.n_events, cfg.n_pixels, cfg.n_samples, d_ped,
                                            d_gain, cfg.W, *outs, chunk_bytes=1 << 30, stream=stream)
        run12()
        torch.cuda.synchronize()
        same = all(bool((o[:64 * cfg.n_pixels] == w).all()) for o, w in zip(outs, want))
        times = []
        before = rta.rta_launch_count()
        for _ in range(2):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            run12()
            torch.cuda.synchronize()
            times.append(time.perf_counter() - t0)
        dt12 = min(times)
        res["packed12"] = {
            "value": cfg.input_bytes / dt12 / 1e9, "unit": UNIT,
            "meaning": "raw-waveform-equivalent GB/s (2 bytes per sample) of the same 200000 events",
            "seconds": dt12, "h2d_bytes": nb, "link_GBps": nb / dt12 / 1e9,
            "frac_of_host_link": nb / dt12 / 1e9 / link_gbs,
            "chunks": (rta.rta_launch_count() - before) // 2,
            "chunk_events": rta.rta_chunk_events(cfg.n_events, cfg.n_pixels, cfg.n_samples, 1 << 30, 12),
            "traces_per_s": cfg.n_traces / dt12, "x_paper_max_rate": cfg.input_bytes / dt12 / 1e9 / PAPER_RATE_GBS[1],
            "speedup_vs_uint16_feed": dt / dt12,
            "first_64_events_equal_uint16_path": same}
    except Exception as ex:  # the uint16 leg above stands on its own
        res["packed12"] = {"error": repr(ex)}
    del host, outs
    rta.rta_shutdown()
    return res


def cpu_baseline_leg(cfg, keep, dl0gen):
    """The oracle, as it stands, on this box's host cores, on the same bytes."""
    import numpy as np
    import oracle
    d_wf, _, _, outs, ped, gain = keep
    cores = os.cpu_count() or 1
    # bounded sample: ~0.28 GB/s per thread -> about 5 s single-threaded
    n_ev = min(cfg.n_events, max(64, int(1.4e9 // (cfg.n_pixels * cfg.n_samples * 2))))
    wf = d_wf[:n_ev].cpu().numpy().view(np.uint16)
    t0 = time.perf_counter()
    r1 = oracle.extract(wf, ped, gain, cfg.W)
    t1 = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.extract_threads(wf, ped, gain, cfg.W, cores)
    tn = time.perf_counter() - t0
    n = n_ev * cfg.n_pixels
    ints_equal = bool((outs[0][:n].cpu().numpy() == r1[0]).all()
                      and (outs[1][:n].cpu().numpy() == r1[1]).all())
    floats_equal = bool((outs[2][:n].cpu().numpy() == r1[2]).all()
                        and (outs[3][:n].cpu().numpy() == r1[3]).all())
    return {"value": wf.nbytes / tn / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "first %d of %d events of %s (%.2f GB), same bytes as the GPU run"
                      % (n_ev, cfg.n_events, cfg.name, wf.nbytes / 1e9),
            "single_thread_value": wf.nbytes / t1 / 1e9,
            "traces_per_s": n / tn, "single_thread_traces_per_s": n / t1,
            "gpu_matches_oracle_on_sample": {"ints_bit_exact": ints_equal,
                                             "floats_bit_exact": floats_equal}}


def main():
    args = parse_args()
    if args.impl == "reference":
        return reference_arm(args)

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
    if world > 1:
        import torch.distributed as dist
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
    if fmt == "p12" or args.path != "extract" or args.workload.startswith("X"):
        args.no_extra = True     # the packed / image main legs are profiling/diagnostic runs
    main_run = kernel_only(cfg, args.steps, args.warmup, torch, dl0gen, rta, barrier, sampler, fmt,
                           args.path)
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
    if args.path != "extract":
        ev_bytes = EVENT_OUT_BYTES * cfg.n_events
        if args.path == "image":
            algo_bytes = cfg.input_bytes + ev_bytes
            kname = rta.rta_image_kernel_name(cfg.n_pixels, cfg.n_samples, cfg.W, True)
            bytes_per_trace = 2 * cfg.n_samples + EVENT_OUT_BYTES / cfg.n_pixels
        else:
            # the charge row is read once; peak times are gathered for the mask pixels only
            algo_bytes = 4 * cfg.n_traces + ev_bytes
            kname = "image_moments"
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
            "traffic": ncu_traffic(kname),
            "frac_of_nominal_8TBps": summ["frac_of_nominal_8TBps"],
        },
    }

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
        if rank == 0 and world == 1:
            if not args.no_cpu:
                out["cpu_baseline"] = cpu_baseline_leg(cfg, keep, dl0gen)
            main_run["keep"] = keep = None
            torch.cuda.empty_cache()
            others = {}
            for name in ("C3", "C4"):
                if name == cfg.name:
                    continue
                c = dl0gen.CONFIGS[name]
                r = kernel_only(c, max(10, args.steps // 2), 3, torch, dl0gen, rta)
                others[name] = summarise(c, r["per_launch_ms"], peak)
                r = None
                torch.cuda.empty_cache()
            out["configs"] = others
            fam = {}
            for name in ("C2", "C3", "C4"):
                fam[name] = family_leg(dl0gen.CONFIGS[name], max(10, args.steps // 4), peak,
                                       torch, dl0gen, rta)
                torch.cuda.empty_cache()
            out["family"] = fam
            pk = {}
            for name in ("C2", "C3", "C4"):
                pk[name] = packed_leg(dl0gen.CONFIGS[name], max(10, args.steps // 4), peak,
                                      torch, dl0gen, rta)
                torch.cuda.empty_cache()
            out["packed12"] = pk
            out["any_shape"] = any_shape_leg(max(10, args.steps // 4), peak, torch, dl0gen, rta)
            torch.cuda.empty_cache()
            out["ragged"] = ragged_leg(max(10, args.steps // 4), peak, torch, dl0gen, rta)
            torch.cuda.empty_cache()
            img = {}
            for name in ("C2", "C3", "C4"):
                img[name] = image_leg(dl0gen.CONFIGS[name], max(10, args.steps // 4), peak,
                                      torch, dl0gen, rta)
                torch.cuda.empty_cache()
            out["image"] = img
            link = host_link_bandwidth(torch)
            out["e2e"]["host_link_GBps_measured"] = link
            out["e2e"]["frac_of_host_link"] = out["e2e"]["value"] / link
            if not args.no_sustained:
                out["sustained"] = sustained_leg(torch, dl0gen, rta, link)
    else:
        out["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0,
                      "d2h_bytes_per_step": 0, "note": "skipped by --no-extra"}
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
