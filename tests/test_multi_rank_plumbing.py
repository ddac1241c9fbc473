"""world_size-2 gloo test (CPU) of the only multi-rank logic the path has: replicas only, no data-path collective
(SURVEY 8(e)); bench.py's value is all ranks' units over the slowest rank's device time."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local = [10.0 + 5.0 * rank, 100.0 - rank, 7.0, 0.5 * (rank + 1)]            # per-rank device times (ms)
    dist.barrier()
    got = bench.max_over_ranks(local, world, torch.device("cpu"))
    q.put((rank, got, bench.whole_job_value(32768, world, 5, got[0])))
    dist.destroy_process_group()


def test_replicas_max_reduce_and_value():
    world, port = 2, 29533
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, value in res:
        assert got == [15.0, 100.0, 7.0, 1.0]                                    # max over the two ranks, on every rank
        assert abs(value - 2 * 32768 * 5 / 15e-3) < 1e-6 * value                 # all ranks' tokens / slowest rank


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], 1, torch.device("cpu")) == [1.5, 2.5]
    assert bench.whole_job_value(100, 1, 2, 1000.0) == 200.0
