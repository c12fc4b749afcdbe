"""Whole-batch comparisons with the oracle: EVERY event of a bench-sized batch,
not sampled blocks. The device-resident input is copied back in slabs of about
1 GB, the unmodified oracle functions run on disjoint event ranges of a slab on
all host cores (ctypes releases the GIL), and the device results of the slab
are compared bit for bit. Holds none of the method's arithmetic."""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

SENTINEL = (-7, -7, -7.0, -7.0)


def host_threads() -> int:
    return os.cpu_count() or 1


def split_events(n_events: int, work, n_threads: int | None = None):
    """work(a, b) -> tuple of arrays for events [a, b); results concatenated in order."""
    n = max(1, min(n_threads or host_threads(), n_events))
    b = [n_events * i // n for i in range(n + 1)]
    with ThreadPoolExecutor(n) as ex:
        parts = list(ex.map(lambda i: work(b[i], b[i + 1]), range(n)))
    return tuple(np.concatenate([p[k] for p in parts]) for k in range(len(parts[0])))


def slabs(n_events: int, event_bytes: int, slab_bytes: int = 1 << 30, multiple: int = 1):
    """(first event, count) of consecutive slabs of at most slab_bytes; counts are
    multiples of `multiple` except the last."""
    step = max(multiple, (slab_bytes // event_bytes) // multiple * multiple)
    e0 = 0
    while e0 < n_events:
        yield e0, min(step, n_events - e0)
        e0 += step


def fill_sentinel(outs):
    """Pre-fill device outputs so that a trace nobody wrote cannot pass by holding
    a stale correct value (the caching allocator hands freed blocks out again)."""
    for o, v in zip(outs, SENTINEL):
        o.fill_(v)


def alloc_filled_outputs(n: int):
    import torch
    outs = (torch.empty(n, dtype=torch.int32, device="cuda"),
            torch.empty(n, dtype=torch.int32, device="cuda"),
            torch.empty(n, dtype=torch.float32, device="cuda"),
            torch.empty(n, dtype=torch.float32, device="cuda"))
    fill_sentinel(outs)
    return outs


def bits_equal(got, want) -> bool:
    return all(np.array_equal(g.view(np.int32), w.view(np.int32)) for g, w in zip(got, want))


def first_mismatch(got, want):
    for k, (g, w) in enumerate(zip(got, want)):
        bad = np.flatnonzero(g.view(np.int32) != w.view(np.int32))
        if bad.size:
            return "output %d: %d traces differ, first at %d (got %r, want %r)" % (
                k, bad.size, int(bad[0]), g[bad[0]], w[bad[0]])
    return "equal"


def compare_every_event(n_events, n_pixels, slab_iter, fetch_input, oracle_fn, outs):
    """For each slab (e0, n): `fetch_input(e0, n)` -> host input of those events,
    `oracle_fn(input, a, b)` -> oracle outputs of events [a, b) of the slab; the
    device outputs `outs` (flat [n_events * n_pixels]) must equal them bit for bit.
    Returns the number of events compared."""
    done = 0
    for e0, n in slab_iter:
        src = fetch_input(e0, n)
        want = split_events(n, lambda a, b: oracle_fn(src, a, b))
        lo, hi = e0 * n_pixels, (e0 + n) * n_pixels
        got = tuple(o[lo:hi].cpu().numpy() for o in outs)
        assert bits_equal(got, want), "events %d..%d: %s" % (e0, e0 + n, first_mismatch(got, want))
        done += n
    assert done == n_events
    return done
