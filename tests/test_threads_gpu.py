"""The boundary's threading promises (SURVEY.md §8(b) "Re-entrancy"; include/rta.h:
rta_extract is thread-safe across streams, the host-fed calls serialise on the
library's workspace mutex, rta_prepare and first-use compiles of one shape do not
hold up other shapes). Eight host threads, each with its own stream, issue a mix of
calls at the same time; ctypes drops the GIL for the duration of a foreign call,
so the library really is entered concurrently. Every result is compared with the
oracle's, computed once up front: integers bit-exact, floats bit-identical.

Between rounds, with every thread parked at a barrier and its stream drained, one
thread calls rta_shutdown: the next round meets a library with no workspace, no
scheduler pool, no compiled specialisations, and all threads race to rebuild them."""
import threading

import numpy as np
import pytest

import dl0gen
import oracle
from tests._gpu import bit_identical
from tests._image import F32, assert_image_parity
from tests._ragged import make_batch

pytestmark = pytest.mark.gpu

N_THREADS, ROUNDS, REPEATS = 8, 3, 6
FILL = (-7, -7, -7.0, -7.0)


def _noise(E, P, S, seed):
    rng = np.random.default_rng(seed)
    ped = rng.integers(380, 421, P).astype(np.int32)
    gain = rng.uniform(0.9, 1.1, P).astype(F32)
    wf = np.clip(np.rint(rng.normal(0, 4, (E, P, S)) + ped[None, :, None]), 0, 4095).astype(np.uint16)
    hot = rng.random((E, P)) < 0.08
    wf[hot, S // 2] += rng.integers(20, 400, int(hot.sum())).astype(np.uint16)
    return wf, ped, gain


class Uniform:
    """rta_extract on one shape (ahead-of-time, run-time compiled, or a P12 stream)."""

    def __init__(self, E, P, S, W, seed, host_fed=False):
        import torch
        self.shape, self.W, self.host_fed = (E, P, S), W, host_fed
        wf, ped, gain = _noise(E, P, S, seed)
        self.want = oracle.extract(wf, ped, gain, W)
        self.wf_host = torch.from_numpy(wf.view(np.int16)).pin_memory()
        self.wf = self.wf_host.cuda()
        self.ped, self.gain = torch.from_numpy(ped).cuda(), torch.from_numpy(gain).cuda()

    def run(self, rta, stream):
        import torch
        E, P, S = self.shape
        outs = [torch.full((E * P,), f, dtype=dt, device="cuda")
                for f, dt in zip(FILL, (torch.int32, torch.int32, torch.float32, torch.float32))]
        if self.host_fed:   # two chunks per call: the double buffer is exercised
            rta.rta_extract_stream(self.wf_host, E, P, S, self.ped, self.gain, self.W, *outs,
                                   chunk_bytes=E * P * S, stream=stream)
        else:
            rta.rta_extract(self.wf, E, P, S, self.ped, self.gain, self.W, *outs, stream=stream)
        stream.synchronize()
        got = tuple(o.cpu().numpy() for o in outs)
        assert bit_identical(got, self.want), "rta_extract%s %r" % ("_stream" if self.host_fed else "", self.shape)


class Image:
    """rta_extract_image on a shape with no fused kernel (scratch from the library's pool)."""

    def __init__(self, E, P, S, W, seed):
        import torch
        self.shape, self.W = (E, P, S), W
        wf, ped, gain = _noise(E, P, S, seed)
        x, y, nbr = dl0gen.hex_camera(P, 0.05)
        self.xy = (x, y)
        _, _, q, t = oracle.extract(wf, ped, gain, W)
        self.want = oracle.image_moments(q.reshape(E, P), t.reshape(E, P), x, y, nbr, 40.0, 20.0)
        d = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt)).cuda()
        self.args = (torch.from_numpy(wf.view(np.int16)).cuda(), E, P, S, d(ped, np.int32), d(gain, F32), W,
                     d(x, F32), d(y, F32), d(nbr, np.int32), 40.0, 20.0)

    def run(self, rta, stream):
        import torch
        E, P, _ = self.shape
        outs = (torch.full((E,), -7, dtype=torch.int32, device="cuda"),
                torch.full((E, 8), -7.0, dtype=torch.float32, device="cuda"),
                torch.full((E, P), 9, dtype=torch.uint8, device="cuda"))
        rta.rta_extract_image(*self.args, *outs, stream=stream)
        stream.synchronize()
        assert_image_parity(tuple(o.cpu().numpy() for o in outs), self.want, *self.xy, "image %r" % (self.shape,))


class Ragged:
    """rta_extract_ragged on a mixed-camera batch (library-owned side streams)."""

    def __init__(self, seed):
        import torch
        b = make_batch([("C1", 1), ((300, 44, 6), 1), ((120, 25, 4), 1)], 24, seed=seed, align=8)
        self.b = b
        self.want = oracle.extract_ragged(b.wf, *b.tables(), b.pedestal, b.gain, b.n_out, fill=FILL)
        self.wf = torch.from_numpy(b.wf.view(np.int16)).cuda()
        self.ped, self.gain = torch.from_numpy(b.pedestal).cuda(), torch.from_numpy(b.gain).cuda()

    def run(self, rta, stream):
        import torch
        plan = rta.rta_ragged_plan_create(*self.b.tables())
        try:
            outs = [torch.full((self.b.n_out,), f, dtype=dt, device="cuda")
                    for f, dt in zip(FILL, (torch.int32, torch.int32, torch.float32, torch.float32))]
            rta.rta_extract_ragged(plan, self.wf, self.ped, self.gain, *outs, stream=stream)
            stream.synchronize()
            got = tuple(o.cpu().numpy() for o in outs)
        finally:
            rta.rta_ragged_plan_destroy(plan)
        assert bit_identical(got, self.want), "rta_extract_ragged"


def test_eight_threads_mixed_calls_and_shutdown_between_rounds():
    import torch
    import paper_1307_6489_b200 as rta
    jobs = [
        Uniform(48, 1855, 40, 7, 1),                   # ahead-of-time kernel
        Uniform(40, 1000, 46, 6, 2),                   # compiled at first use: all threads race on it
        Uniform(40, 1000, 52, 9, 3),                   # a second new shape compiling at the same time
        Uniform(32, 1855, 40, 7, 4, host_fed=True),    # workspace + mutex
        Image(24, 1039, 36, 5, 5),                     # scratch pool
        Ragged(6),                                     # side streams
    ]
    torch.cuda.synchronize()
    barrier = threading.Barrier(N_THREADS)
    errors = []

    def worker(tid):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            for rnd in range(ROUNDS):
                barrier.wait()
                for rep in range(REPEATS):
                    for k in range(len(jobs)):   # every thread starts on another job
                        jobs[(k + tid + rep) % len(jobs)].run(rta, stream)
                stream.synchronize()
                barrier.wait()
                if tid == rnd % N_THREADS:       # everyone else is parked at the next barrier
                    torch.cuda.synchronize()
                    rta.rta_shutdown()
        except BaseException as exc:  # noqa: BLE001 - reported by the main thread
            errors.append((tid, repr(exc)))
            barrier.abort()

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(N_THREADS)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(600)
    assert not any(t.is_alive() for t in threads), "a worker is stuck"
    assert not errors, errors


def test_prepare_takes_the_compile_off_the_first_call():
    """After rta_prepare the first call of a never-seen shape compiles nothing: it costs
    a small fraction of what the preparation did."""
    import time
    import torch
    import paper_1307_6489_b200 as rta
    S, W = 58, 11   # no other test uses this shape
    if not rta.rta_kernel_name(S, W).startswith("staged<jit>"):
        pytest.skip("no libnvrtc on this box")
    rta.rta_shutdown()
    t0 = time.perf_counter()
    assert rta.rta_prepare(S, W) is True
    t_prepare = time.perf_counter() - t0
    assert rta.rta_prepare(S, W, rta.RTA_EXTRACTOR_LOCAL_PEAK) is True
    assert rta.rta_prepare(40, 7) is True                    # built ahead of time
    assert rta.rta_prepare(2048, 8) is False                 # too long for a specialisation
    job = Uniform(64, 1855, S, W, 9)
    torch.cuda.synchronize()
    stream = torch.cuda.Stream()
    t0 = time.perf_counter()
    job.run(rta, stream)
    t_first = time.perf_counter() - t0
    assert t_first < max(0.1, 0.5 * t_prepare), (t_prepare, t_first)
