"""Tensor-parallel scoring (App. H: "tensor-parallel ranks all-reduce the per-token score vector before
top-k").

Under tensor parallelism by KV head every rank holds the K/V pools of its own head shard and the matching slice of the
QueryMemory, `[L][H_q / tp][D]`.  Each (layer, head) row of Eq. 3 is a softmax over the TOKENS, so a rank computes its
heads' rows completely; rule_j = sum over (l, h) is then a plain sum of the ranks' partial score vectors: ONE all-reduce
(sum) of N fp32 values (128 KB at 32k tokens), after which every rank runs the same deterministic selection.  The
fillers of forced / dead positions (+INF / -INF) are identical on every rank and survive the sum.

This module is the exchange step only (torch.distributed: NCCL over NVLink on GPUs, gloo in the CPU test); the scoring
itself is `ikv_score` of the rank's own context.  One GPU per process.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def all_reduce_scores(scores: torch.Tensor, group=None) -> torch.Tensor:
    """In-place sum of the ranks' partial score vectors.  A single small collective: latency-bound (~10 us over NVLink)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(scores, op=dist.ReduceOp.SUM, group=group)
    return scores


def tp_score_memory(ctx, reqs, scores: torch.Tensor, group=None, stream=None) -> torch.Tensor:
    """Rule score (IKV_MODE_MEMORY / QUERY family) under tensor parallelism: this rank's heads, then the all-reduce.
    `ctx` is the rank's own ikv.Context over its head shard.  The learnable mode additionally needs the mean key over ALL
    heads (a second all-reduce of T x D partial sums before the residual head) and is not wired here."""
    from . import ikv
    ctx.score(reqs, ikv.MODE_MEMORY, scores, None, stream)
    if stream is not None:
        with torch.cuda.stream(stream):
            return all_reduce_scores(scores, group)
    return all_reduce_scores(scores, group)
