"""N > 1 host logic on CPU (gloo, world sizes 2, 4 and 8): the path shards by contiguous
event ranges with replicated calibration and NO data-path collective
(SURVEY.md §8(e)); torch.distributed is used only for the barrier and the MAX
over ranks of the timed region, exactly as bench.py does with NCCL.

What is checked without a GPU: the event ranges of `shard_events` tile the
batch exactly, every rank generates exactly its own events (counter-based
generator, no communication), the per-rank results concatenated in rank order
equal the single-rank result, and the MAX-over-ranks reduction bench.py relies
on. The per-rank extraction itself is stood in for by the oracle here (tests may
call it); on the GPU box the same ranges go through rta_extract."""
import os
import socket

import numpy as np
import pytest

import dl0gen
import oracle
from paper_1307_6489_b200 import shard_events


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n_events, tmpdir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = dl0gen.CONFIGS["C1"]
        ped, gain = dl0gen.calib(c)                       # replicated calibration
        first, count = shard_events(n_events, world, rank)
        wf = dl0gen.events_cpu(c, first, count, threads=1)
        res = oracle.extract(wf, ped, gain, c.W)
        np.savez(os.path.join(tmpdir, "rank%d.npz" % rank), first=first, count=count,
                 s=res[0], t=res[1], q=res[2], tm=res[3])
        # every rank plans the chunks of its own event range (rta_extract_stream's rule):
        # whole events, at least one per chunk, and the chunks tile the range exactly
        import paper_1307_6489_b200 as rta
        ev_bytes = c.n_pixels * c.n_samples * 2
        for chunk_bytes in (0, ev_bytes, 3 * ev_bytes + 5, 10 ** 9):
            ce = rta.rta_chunk_events(count, c.n_pixels, c.n_samples, chunk_bytes, 16)
            want = max(1, min(count, ((chunk_bytes or 1 << 30) // ev_bytes) or 1))
            assert ce == want, (rank, count, chunk_bytes, ce, want)
            assert sum(min(ce, count - e0) for e0 in range(0, count, ce)) == count
        dist.barrier()
        # bench.py's reduction: the step time is the MAX over ranks
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert float(t) == 10.0 + world - 1
        # whole-job units = sum over ranks of the units each processed
        n = torch.tensor([count], dtype=torch.int64)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
        assert int(n) == n_events
        # the sustained leg sizes every rank's pinned buffer by the MIN over ranks
        m = torch.tensor([1000 * (rank + 3)], dtype=torch.int64)
        dist.all_reduce(m, op=dist.ReduceOp.MIN)
        assert int(m) == 3000
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_events,world", [(64, 2), (7, 2), (64, 4), (61, 8)])
def test_ranks_shard_events_without_a_collective(tmp_path, n_events, world):
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(world, _free_port(), n_events, str(tmp_path)), nprocs=world, join=True)
    c = dl0gen.CONFIGS["C1"]
    ped, gain = dl0gen.calib(c)
    whole = oracle.extract(dl0gen.events_cpu(c, 0, n_events, threads=2), ped, gain, c.W)
    parts = [np.load(os.path.join(str(tmp_path), "rank%d.npz" % r)) for r in range(world)]
    assert int(parts[0]["first"]) == 0
    assert sum(int(p["count"]) for p in parts) == n_events
    for r in range(1, world):
        assert int(parts[r]["first"]) == int(parts[r - 1]["first"]) + int(parts[r - 1]["count"])
    for k, key in enumerate(("s", "t", "q", "tm")):
        cat = np.concatenate([p[key] for p in parts])
        assert np.array_equal(cat.view(np.int32), whole[k].view(np.int32))


@pytest.mark.parametrize("n_events,world", [(0, 1), (1, 4), (10, 3), (10_000, 8), (200_000, 7)])
def test_shard_events_tiles_the_batch(n_events, world):
    ranges = [shard_events(n_events, world, r) for r in range(world)]
    pos = 0
    for first, count in ranges:
        assert first == pos and count >= 0
        pos += count
    assert pos == n_events
    counts = [c for _, c in ranges]
    assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        shard_events(n_events, world, world)


def test_bench_spawns_one_rank_per_gpu_when_asked_for_several():
    """`python bench.py --gpus N` outside torchrun re-executes itself under
    torch.distributed.run with N ranks on 127.0.0.1 and the same arguments."""
    import importlib.util
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    cmd = bench.multi_rank_command(8, ["--gpus", "8", "--steps", "5"])
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert cmd[cmd.index("--nproc-per-node") + 1] == "8"
    assert "--standalone" in cmd and cmd[cmd.index("--local-addr") + 1] == "127.0.0.1"
    assert cmd[-5:] == [os.path.join(root, "bench.py"), "--gpus", "8", "--steps", "5"]
    # one sampling rule for the oracle timing of both arms
    import dl0gen
    assert bench.oracle_sample_events(dl0gen.CONFIGS["C2"]) == 10_000
    assert bench.oracle_sample_events(dl0gen.CONFIGS["C4"]) == int(2e9 // (2048 * 128 * 2))
