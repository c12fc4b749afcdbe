"""The seeded input generator: reproducible, chunk-independent, and shaped as
BASELINE.json:configs describes. The gpu test checks
that the CUDA build writes the same bytes as the host build, which is what
lets full-size parity tests regenerate any event range for the oracle."""
import dataclasses

import numpy as np
import pytest

import dl0gen


def test_configs_match_baseline_shapes():
    c = dl0gen.CONFIGS
    assert (c["C1"].n_events, c["C1"].n_pixels, c["C1"].n_samples, c["C1"].W) == (64, 1855, 30, 7)
    assert (c["C2"].n_events, c["C2"].n_pixels, c["C2"].n_samples, c["C2"].W) == (10000, 1855, 40, 7)
    assert (c["C3"].n_events, c["C3"].n_pixels, c["C3"].n_samples, c["C3"].W) == (20000, 1764, 25, 4)
    assert (c["C4"].n_events, c["C4"].n_pixels, c["C4"].n_samples, c["C4"].W) == (20000, 2048, 128, 8)
    assert (c["C5"].n_events, c["C5"].n_pixels, c["C5"].n_samples, c["C5"].W) == (200000, 1855, 40, 7)
    assert c["C1"].seed == 0
    assert c["C2"].input_bytes == 1_484_000_000 and c["C5"].input_bytes == 29_680_000_000


def test_reproducible_and_chunk_independent():
    c = dl0gen.CONFIGS["C1"]
    a = dl0gen.events_cpu(c, 0, 12)
    b = dl0gen.events_cpu(c, 0, 12)
    assert (a == b).all()
    mid = dl0gen.events_cpu(c, 5, 4, threads=3)
    assert (mid == a[5:9]).all()
    other = dl0gen.events_cpu(dataclasses.replace(c, seed=7), 0, 2)
    assert (other != a[:2]).any()


@pytest.mark.parametrize("name,n_ev", [("C1", 64), ("C2", 40), ("C3", 40), ("C4", 20)])
def test_statistics_follow_the_recipe(name, n_ev):
    c = dl0gen.CONFIGS[name]
    ped, gain = dl0gen.calib(c)
    assert ped.min() >= c.ped_lo and ped.max() <= c.ped_hi
    assert len(np.unique(ped)) > (c.ped_hi - c.ped_lo) * 0.8
    assert gain.min() >= 0.9 and gain.max() <= 1.1 and 0.98 < gain.mean() < 1.02
    wf = dl0gen.events_cpu(c, 0, n_ev, threads=4)
    assert wf.dtype == np.uint16 and wf.max() <= 4095
    x = wf.astype(np.int64) - ped[None, :, None]
    head = x[:, :, :3]                      # before any pulse can reach
    assert abs(head.mean()) < 0.05
    # rounding to integers adds 1/12 to the variance
    assert abs(head.std() - np.sqrt(c.noise_sigma ** 2 + 1 / 12)) < 0.05
    # pulsed fraction: traces whose maximum stands far above the noise
    amp_med = np.exp(c.amp_mu)
    thr = 5 * c.noise_sigma
    bright = (x.max(-1) > thr).mean()
    # P(A > thr) for the log-normal, times the Bernoulli fraction
    from math import erf, log, sqrt
    p_amp = 0.5 * (1 - erf((log(thr) - c.amp_mu) / (c.amp_sigma * sqrt(2))))
    assert 0.5 * c.pulse_frac * p_amp < bright < 1.5 * c.pulse_frac * p_amp + 1e-3
    assert amp_med > 0
    # pulse positions fall in the configured range
    t_peak = x.argmax(-1)[x.max(-1) > 4 * thr]
    if len(t_peak) > 20:
        assert t_peak.min() >= c.peak_lo - 2 and t_peak.max() <= c.peak_hi + 2


@pytest.mark.gpu
@pytest.mark.parametrize("name,first,n_ev", [("C1", 0, 64), ("C2", 9990, 10),
                                             ("C3", 12345, 7), ("C4", 19995, 5),
                                             ("C5", 199_990, 10)])
def test_cuda_generator_is_byte_identical_to_host(name, first, n_ev):
    import torch
    c = dl0gen.CONFIGS[name]
    dev = torch.empty((n_ev, c.n_pixels, c.n_samples), dtype=torch.int16, device="cuda")
    dl0gen.events_cuda(c, dev.data_ptr(), first, n_ev,
                       torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    got = dev.cpu().numpy().view(np.uint16)
    want = dl0gen.events_cpu(c, first, n_ev, threads=4)
    assert (got == want).all()
