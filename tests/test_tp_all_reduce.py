"""world_size-2 gloo test (CPU) of the tensor-parallel exchange step (paper_2606_09916_b200/tp.py): every
rank scores its own KV-head shard with the oracle, the partial score vectors are all-reduced, and the sum equals the
oracle's score over all heads -- fillers included."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import ikv_oracle as o
    from paper_2606_09916_b200 import tp, workloads as wl
    shape = wl.ModelShape(2, 8, 4, 64, "bf16")
    w = wl.small(seed=5, shape=shape, n_tokens=400, budget=100, prefix_len=11, span_len=9, kv_dtype="bf16")
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy().copy()
    S[::13] = w.dead_slot
    M = np.zeros((shape.L, shape.Hq, shape.D))
    for rows in s.updates():
        o.memory_update(M, rows.numpy(), 0.5)
    # this rank's shard: KV heads [rank*2, rank*2+2), query heads [rank*4, rank*4+4)
    hk, hq = shape.Hkv // world, shape.Hq // world
    k_shard = w.k_pool[:, :, rank * hk:(rank + 1) * hk].contiguous()
    g = o.Geometry(shape.L, hq, hk, shape.D, w.n_slots, o.BF16, w.dead_slot)
    part = o.score(g, wl.to_numpy_bits(k_shard), np.ascontiguousarray(M[:, rank * hq:(rank + 1) * hq]), S, s.pi, s.qs, s.qe)
    t = torch.from_numpy(part.astype(np.float32))
    tp.all_reduce_scores(t)
    full = o.score(o.Geometry(shape.L, shape.Hq, shape.Hkv, shape.D, w.n_slots, o.BF16, w.dead_slot),
                   wl.to_numpy_bits(w.k_pool), M, S, s.pi, s.qs, s.qe)
    q.put((rank, t.numpy(), full))
    dist.destroy_process_group()


def test_head_sharded_scores_all_reduce_to_the_full_score():
    world, port = 2, 29541
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, full in res:
        fin = np.isfinite(full)
        assert np.array_equal(np.isposinf(got), np.isposinf(full)) and np.array_equal(np.isneginf(got), np.isneginf(full))
        assert np.allclose(got[fin], full[fin], rtol=1e-6, atol=1e-7)          # fp32 partial sums
        assert abs(got[fin].sum() - 2 * 8) < 1e-4                                # P1: sum_j rule_j = L * H_q
