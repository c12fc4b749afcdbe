"""Host-side logic of bench.py that needs no GPU: the oracle sampling rule, the slab walk of
the full-size verification, the byte accounting of the gathering fixed-window route, the
tie between profiles/traffic.json and the kernel sources, the per-leg clock window."""
import json
import os

import numpy as np
import pytest

import bench
import dl0gen


def test_one_sampling_rule_for_the_oracle_timing():
    """Whole workload up to 2 GB of input, else the first 2 GB of events (both bench arms)."""
    c = dl0gen.CONFIGS
    assert bench.oracle_sample_events(c["C2"]) == c["C2"].n_events           # 1.48 GB: all of it
    assert bench.oracle_sample_events(c["C3"]) == c["C3"].n_events           # 1.76 GB
    n4 = bench.oracle_sample_events(c["C4"])                                # 10.5 GB: the first 2 GB
    ev = c["C4"].n_pixels * c["C4"].n_samples * 2
    assert n4 * ev <= 2e9 < (n4 + 1) * ev
    assert bench.oracle_sample_events(c["C1"]) == c["C1"].n_events


@pytest.mark.parametrize("n_events,event_bytes,slab", [(10, 100, 250), (7, 3, 1), (200000, 148400, 1 << 30),
                                                       (1, 10, 5), (5, 100, 100)])
def test_event_slabs_cover_every_event_once(n_events, event_bytes, slab):
    seen = []
    for first, count in bench.event_slabs(n_events, event_bytes, slab):
        assert count >= 1 and count * event_bytes <= max(slab, event_bytes)
        seen.extend(range(first, first + count))
    assert seen == list(range(n_events))


def test_fixed_window_gather_counts_sectors():
    """Traces longer than 96 bytes: 32-byte sectors the W-sample window overlaps + 16 bytes out;
    shorter traces stream (None)."""
    import torch
    c4, c2 = dl0gen.CONFIGS["C4"], dl0gen.CONFIGS["C2"]
    assert bench.fixed_gather_bytes_per_trace(c2, torch.zeros(c2.n_pixels, dtype=torch.int32)) == (None, None)
    # window at sample 0 of a 256-byte trace: bytes [0, 16) of a 32-byte-aligned trace: one sector
    per, sectors = bench.fixed_gather_bytes_per_trace(c4, torch.zeros(c4.n_pixels, dtype=torch.int32))
    assert sectors == 1.0 and per == 32.0 + 16.0
    # window at sample 12: bytes [24, 40): always two sectors
    per, sectors = bench.fixed_gather_bytes_per_trace(c4, torch.full((c4.n_pixels,), 12, dtype=torch.int32))
    assert sectors == 2.0 and per == 64.0 + 16.0


def test_traffic_is_tied_to_the_kernel_sources(tmp_path, monkeypatch):
    """bench reports the committed ncu traffic only when profiles/traffic.json was captured on
    the kernel sources that are being run (content hash of csrc/)."""
    t = json.load(open(os.path.join(bench.ROOT, "profiles", "traffic.json")))
    assert set(t) >= {"commit", "csrc_sha256", "kernels"} and "tile<S=40,W=7>" in t["kernels"]
    sha = bench.csrc_sha256()
    assert len(sha) == 16 and sha == bench.csrc_sha256()
    root = tmp_path / "repo"
    (root / "profiles").mkdir(parents=True)
    monkeypatch.setattr(bench, "ROOT", str(root))
    monkeypatch.setattr(bench, "csrc_sha256", lambda: "0123456789abcdef")
    json.dump({"commit": "abc1234", "csrc_sha256": "0123456789abcdef", "kernels": {"k": 42}},
              open(root / "profiles" / "traffic.json", "w"))
    assert bench.ncu_traffic("k") == (42, "abc1234", False)
    assert bench.ncu_traffic("other") == (None, "abc1234", False)
    monkeypatch.setattr(bench, "csrc_sha256", lambda: "ffffffffffffffff")        # sources changed since
    assert bench.ncu_traffic("k") == (None, "abc1234", True)
    os.remove(root / "profiles" / "traffic.json")
    assert bench.ncu_traffic("k") == (None, None, None)


def test_clock_window_of_a_leg():
    class Nvml:
        nvmlClocksThrottleReasonSwPowerCap = 4
    s = bench.ClockSampler(0)
    s.nvml = Nvml()
    s.samples = [(1965.0, 0, 300.0), (1965.0, 0, 310.0), (1700.0, 4, 800.0), (1650.0, 4, 790.0), (1965.0, 0, None)]
    w = s.window(2, 4)
    assert w == {"sm_mhz": 1675.0, "sm_min_mhz": 1650.0, "watts_max": 800.0, "sw_power_cap": True, "samples": 2}
    assert s.window(0, 2)["sw_power_cap"] is False and s.window(3, 3) is None


def test_extra_shapes_are_not_baseline_configs():
    xs = bench.extra_shapes(dl0gen)
    assert set(xs) == {"X60", "X40w5", "X96", "X128w10", "X2048"}
    for name, c in xs.items():
        assert name not in dl0gen.CONFIGS and c.n_samples * c.W * 65535 < 2 ** 31
        assert bench.workload(name, dl0gen) is not None
    assert bench.workload("C2", dl0gen) is dl0gen.CONFIGS["C2"]


def test_compact_summary_is_short_and_carries_every_leg():
    """The driver keeps the tail of the bench line: the last key must hold every leg as
    [ms, fraction] in well under 2 KB ("only C2 is in the record")."""
    import json
    import bench
    leg = lambda ms, f: {"ms_avg": ms, "frac_of_measured_hbm": f}
    lat = {m: {"p50_us": 12.345, "p99_us": 20.0, "min_us": 10.0} for m in
           ("extract_eager", "extract_graph_replay", "extract_host", "extract_image_host")}
    out = {
        "roofline": {"avg_launch_ms": 0.26, "frac": 1.046, "peak": 6546.6, "frac_of_read_stream_peak": 0.93},
        "configs": {"C3": leg(0.336, 1.057), "C4": leg(1.734, 0.98),
                    "C1": {"workload": "C1", "l2": "x", "eager_flushed": leg(0.01, 0.1),
                           "eager_resident": leg(0.008, 0.2), "graph_replay_flushed": leg(0.009, 0.1),
                           "graph_replay_resident": leg(0.007, 0.2)}},
        "family": {c: {k: leg(0.3, 0.9) for k in ("fixed", "local_peak", "fir")} for c in ("C2", "C3", "C4")},
        "packed12": {c: leg(0.3, 0.9) for c in ("C2", "C3", "C4")},
        "image": {c: {k: leg(0.3, 0.9) for k in ("fused", "moments", "two_calls")} for c in ("C2", "C3", "C4")},
        "ragged": dict(leg(0.83, 0.95), unspecialised=leg(0.66, 0.93)),
        "any_shape": {n: {"kernel": "staged<jit>", "staged_any": leg(0.36, 1.0), "generic": leg(2.0, 0.2)}
                      for n in ("X60", "X40w5", "X96", "X128w10", "X2048")},
        "e2e": {"value": 53.8, "frac_of_host_link": 0.97},
        "sustained": {"value": 55.2, "frac_of_host_link": 0.99,
                      "pageable": {"value": 44.0, "frac_of_host_link": 0.8},
                      "image": {"value": 55.0, "frac_of_host_link": 0.99},
                      "packed12": {"value": 73.0, "frac_of_host_link": 0.99}},
        "latency": dict({"calls": 1000, "abi_call_us": 0.4}, **{"n%d" % n: lat for n in (1, 8, 64, 512, 4096)}),
        "leg_clocks": {"packed12.C4": {"sw_power_cap": True}, "image.C2": {"sw_power_cap": False}},
    }
    sm = bench.compact_summary(out)
    text = json.dumps(sm)
    assert len(text) < 2000, len(text)
    assert sm["C3"] == [0.336, 1.057] and sm["C4"] == [1.734, 0.98]
    assert sm["main"] == [0.26, 1.046, 0.93]
    assert sm["C1"]["graph_replay_l2"] == [0.007, 0.2]
    assert sm["fam.C4"]["fixed"] == [0.3, 0.9] and sm["p12.C2"] == [0.3, 0.9]
    assert sm["img.C3"]["moments"] == [0.3, 0.9] and sm["ragged.unspec"] == [0.66, 0.93]
    assert sm["sus.packed12"] == [73.0, 0.99] and sm["lat.n64"] == [12.3, 12.3, 12.3, 12.3]
    assert sm["cap"] == ["packed12.C4"]
