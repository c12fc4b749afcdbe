"""rta_extract_image_noalloc against rta_extract_image (include/rta.h).

The no-allocation entry point exists for callers that may not touch the device
allocator: an analysis thread during data taking (cudaMalloc / cudaFree synchronise
the whole device and would stall the event feed) and processes whose device memory
is already owned in full by something else. It keeps its scratch in a fixed static
device array, shared by every call and never cleared between calls, so the thing
to check is that a second call is not disturbed by what the first one left there.

Each test therefore makes two calls in a row, on different events and different
shapes, and compares both with the ordinary entry point on the same inputs:
n_pix, mask and q_max bit for bit, the fp32 parameters within the tolerances of
tests/_image.py (the two routes run the same integer extraction and the same
moments code, so on shapes where the ordinary call also takes two kernels they have
to agree bit for bit; that is asserted too. On the BASELINE shapes the ordinary call
is one fused kernel that sums in another order: tolerances only).

This file sorts after every other test file on purpose: `pytest -x` stops at the
first failure and a failure here must not hide the rest of the suite. It passes on
its own in a fresh process (first use of the library on the device) and after all
the other GPU tests (scheduler pools, JIT cache and memory pools already warm)."""
import numpy as np
import pytest

import dl0gen
from tests._image import F32, assert_image_parity

TP, TB = 40.0, 20.0   # picture / boundary thresholds, ADC counts after gain


def dev(a, dtype=None):
    import torch
    a = np.ascontiguousarray(a, dtype)
    if a.dtype == np.uint16:
        a = a.view(np.int16)
    return torch.from_numpy(a).cuda()


def image_outputs(E, P, mask=True):
    """Sentinel-filled outputs: an element the call does not write shows up."""
    import torch
    return (torch.full((E,), -7, dtype=torch.int32, device="cuda"),
            torch.full((E, 8), -7.0, dtype=torch.float32, device="cuda"),
            torch.full((E, P), 9, dtype=torch.uint8, device="cuda") if mask else None)


def host(outs):
    import torch
    torch.cuda.synchronize()
    return tuple(None if o is None else o.cpu().numpy() for o in outs)


def _inputs(E, P, S, W, seed):
    """Noise + pulses of the BASELINE signal model on a hex camera (inputs only)."""
    rng = np.random.default_rng(seed)
    x, y, nbr = dl0gen.hex_camera(P, 0.05)
    ped = rng.integers(380, 421, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(F32)
    wf = rng.normal(0.0, 4.0, (E, P, S)) + ped[None, :, None]
    s = np.arange(S)[None, None, :]
    for e in range(E):  # a blob of pulsed pixels around a random centre, so that images are not empty
        c = rng.integers(0, P)
        near = np.hypot(x - x[c], y - y[c]) < 0.05 * rng.uniform(2.0, 5.0)
        amp = rng.lognormal(3.5, 1.0, P) * near
        peak = rng.uniform(0.3 * S, 0.7 * S, P)
        wf[e] += amp[:, None] * np.exp(-0.5 * ((s[0] - peak[:, None]) / 1.5) ** 2)
    wf = np.clip(np.rint(wf), 0, 4095).astype(np.uint16)
    return wf, ped, gain, x, y, nbr


def _both(wf, ped, gain, W, x, y, nbr, mask=True):
    """(existing path, no-allocation path) on the same device buffers."""
    import paper_1307_6489_b200 as rta
    E, P, S = wf.shape
    args = (dev(wf), E, P, S, dev(ped, np.int32), dev(gain, F32), W, dev(x, F32), dev(y, F32),
            dev(nbr, np.int32), TP, TB)
    ref, got = image_outputs(E, P, mask), image_outputs(E, P, mask)
    rta.rta_extract_image(*args, *ref)
    rta.rta_extract_image_noalloc(*args, *got)
    return host(ref), host(got)


def _assert_same(ref, got, x, y, what, bits):
    assert_image_parity(got, ref, x, y, what)
    assert ref[0].sum() > 0, what + ": every image is empty, the comparison says nothing"
    if bits:
        assert np.array_equal(got[1].view(np.uint32), ref[1].view(np.uint32)), what + ": parameter bits"


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    # first call: a shape with no ahead-of-time kernel, ragged tail (E*P not a tile multiple)
    a = _inputs(37, 1855, 36, 5, seed=11)
    ref, got = _both(*a[:3], 5, *a[3:])
    _assert_same(ref, got, a[3], a[4], "call 1 (S=36, W=5)", bits=True)
    # second call: other events, other camera, odd n_samples, fewer traces than the first call
    # left in the scratch (stale results sit behind this call's arrays)
    b = _inputs(9, 1039, 27, 4, seed=12)
    ref, got = _both(*b[:3], 4, *b[3:], mask=False)
    _assert_same(ref, got, b[3], b[4], "call 2 (S=27, W=4)", bits=True)
    # and a third, larger than both, on a BASELINE shape (the existing path fuses this one)
    c = _inputs(64, 1855, 40, 7, seed=13)
    ref, got = _both(*c[:3], 7, *c[3:])
    _assert_same(ref, got, c[3], c[4], "call 3 (S=40, W=7)", bits=False)
    # and one that fills the scratch to its last byte: exactly RTA_NOALLOC_MAX_TRACES traces
    import paper_1307_6489_b200 as rta
    assert 512 * 2048 == rta.RTA_NOALLOC_MAX_TRACES
    d = _inputs(512, 2048, 34, 6, seed=14)
    ref, got = _both(*d[:3], 6, *d[3:])
    _assert_same(ref, got, d[3], d[4], "call 4 (the maximum size)", bits=True)


@pytest.mark.gpu
def test_back_to_back_on_one_stream_without_a_sync_between():
    """Two calls queued on one stream share the scratch safely (stream order); the
    second must not see the first one's scheduler words or results."""
    import torch
    import paper_1307_6489_b200 as rta
    a = _inputs(40, 1855, 32, 6, seed=21)
    b = _inputs(40, 1855, 32, 6, seed=22)
    outs, refs = [], []
    st = torch.cuda.Stream()
    bufs = []
    for wf, ped, gain, x, y, nbr in (a, b):
        E, P, S = wf.shape
        bufs.append((dev(wf), E, P, S, dev(ped, np.int32), dev(gain, F32), 6, dev(x, F32),
                     dev(y, F32), dev(nbr, np.int32), TP, TB))
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        for args in bufs:
            o = image_outputs(args[1], args[2])
            rta.rta_extract_image_noalloc(*args, *o, stream=st)
            outs.append(o)
    st.synchronize()
    for args in bufs:
        r = image_outputs(args[1], args[2])
        rta.rta_extract_image(*args, *r)
        refs.append(r)
    for i, (o, r, inp) in enumerate(zip(outs, refs, (a, b))):
        _assert_same(host(r), host(o), inp[3], inp[4], "queued call %d" % (i + 1), bits=True)


def test_limits_are_reported_not_silently_truncated():
    """Argument checks come before the first CUDA call, so this one runs without a GPU."""
    import paper_1307_6489_b200 as rta
    L = rta.lib()
    P = 1855
    too_many = rta.RTA_NOALLOC_MAX_TRACES // P + 1
    call = lambda E=1, S=40, W=7, wf=0x1000: L.rta_extract_image_noalloc(
        wf, E, P, S, 0x2000, 0x3000, W, 0x4000, 0x5000, 0x6000, 1.0, 0.5, 0x7000, 0x8000, None, 0)
    assert call(E=too_many) == rta.RTA_ERR_TOO_LARGE
    assert "RTA_NOALLOC_MAX_TRACES" in rta.rta_strerror(rta.RTA_ERR_TOO_LARGE)
    assert call(wf=0x1002) == rta.RTA_ERR_ALIGN           # staged loads need 16 bytes
    assert call(S=2048, W=8) == rta.RTA_ERR_UNSUPPORTED   # trace longer than the staged kernel takes
    assert call(E=0) == rta.RTA_OK
    assert call(W=41) == rta.RTA_ERR_SHAPE
