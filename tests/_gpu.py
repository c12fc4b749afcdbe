"""Helpers for the -m gpu tests: move numpy inputs to the device with torch,
call the C ABI through the binding, bring the four outputs back."""
from __future__ import annotations

import numpy as np


def to_dev_u16(wf: np.ndarray):
    import torch
    return torch.from_numpy(np.ascontiguousarray(wf).view(np.int16)).cuda()


def alloc_outputs(n: int):
    import torch
    return (torch.empty(n, dtype=torch.int32, device="cuda"),
            torch.empty(n, dtype=torch.int32, device="cuda"),
            torch.empty(n, dtype=torch.float32, device="cuda"),
            torch.empty(n, dtype=torch.float32, device="cuda"))


def run_gpu(wf: np.ndarray, pedestal, gain, W: int, generic: bool = False):
    """wf uint16 [E][P][S] on the host -> outputs as numpy arrays."""
    import torch
    import paper_1307_6489_b200 as rta
    E, P, S = wf.shape
    d_wf = to_dev_u16(wf)
    d_ped = torch.from_numpy(np.ascontiguousarray(pedestal, np.int32)).cuda()
    d_gain = torch.from_numpy(np.ascontiguousarray(gain, np.float32)).cuda()
    outs = alloc_outputs(E * P)
    rta.rta_extract(d_wf, E, P, S, d_ped, d_gain, W, *outs, generic=generic)
    torch.cuda.synchronize()
    return tuple(o.cpu().numpy() for o in outs)


def assert_parity(got, want, what=""):
    """north_star's bar: ints bit-exact, charge rel 1e-6, time abs 1e-4 (R12:
    bit-equal to RN32 where |t| > 1024). The kernels are built to be
    bit-identical on floats as well, which is checked first and reported."""
    gs, gt, gq, gtm = got
    ws, wt, wq, wtm = want
    assert (gs == ws).all(), what + ": out_sum differs"
    assert (gt == wt).all(), what + ": out_start differs"
    q_ok = (gq == wq) | (np.isnan(gq) & np.isnan(wq)) | np.isclose(gq, wq, rtol=1e-6, atol=0.0)
    assert q_ok.all(), what + ": charge outside rel 1e-6"
    big = np.abs(wtm) > 1024.0
    assert (np.abs(gtm[~big].astype(np.float64) - wtm[~big].astype(np.float64)) <= 1e-4).all(), \
        what + ": time outside abs 1e-4"
    assert (gtm[big] == wtm[big]).all(), what + ": time != RN32 beyond 1024"


def bit_identical(got, want) -> bool:
    return all(np.array_equal(g.view(np.int32), w.view(np.int32)) for g, w in zip(got, want))
