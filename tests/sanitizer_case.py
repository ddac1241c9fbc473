"""The case run under compute-sanitizer (memcheck / racecheck / synccheck; summaries in profiles/r2_sanitizer.md):
the tiny config and a small bf16 learnable case -- prune (memory update, score, select / evict) followed by three
decode calls, programmatic launches on, and a multi-row / baseline / prefill call each.  Not collected by pytest.

    compute-sanitizer --tool memcheck python tests/sanitizer_case.py
"""
import math
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import torch  # noqa: E402

from paper_2606_09916_b200 import ikv, workloads as wl  # noqa: E402


def run(w, learnable, layer_major):
    shape = w.shape
    w.k_pool, w.v_pool = w.k_pool.cuda(), w.v_pool.cuda()
    s = w.sessions[0]
    ctx = ikv.Context(shape.L, shape.Hq, shape.Hkv, shape.D, w.k_pool, w.v_pool, dead_slot=w.dead_slot)
    ctx.tune(ikv.TUNE_LAYER_MAJOR, layer_major)
    ctx.residual_load(wl.residual_weights(shape.D, 5))
    ctx.session_open(1)
    for rows in s.updates():
        ctx.memory_update(1, rows.cuda().contiguous())
    S_dev = s.slot_map.clone().cuda()
    scores = torch.empty(s.N, device="cuda")
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    req = ikv.make_request(1, S_dev, s.N, s.pi, s.qs, s.qe, s.spec.budget, s.pi)
    dt = w.k_pool.dtype
    for mode in ([ikv.MODE_LEARNABLE] if learnable else []) + [ikv.MODE_MEMORY]:
        S_dev.copy_(s.slot_map.cuda())
        ctx.score([req], mode, scores)
        ctx.select_evict([req], scores, freed, nf, nk)
        for layer in range(3):
            q = torch.randn((1, shape.Hq, shape.D), device="cuda").to(dt)
            out = torch.empty_like(q)
            r = ikv.make_request(1, S_dev, s.N + 1 + layer % 2, s.pi, s.qs, s.qe, s.spec.budget, s.pi)
            ctx.decode_attn(layer % shape.L, [r], q, out, 1.0 / math.sqrt(shape.D))
    if dt == torch.bfloat16:
        rows = torch.randn((3, shape.L, shape.Hq, shape.D), device="cuda")
        S_dev.copy_(s.slot_map.cuda())
        ctx.score_rows([req], rows, [1.0, 0.5, 2.0], scores)
        ctx.score_baseline([req], ikv.BASE_SNAPKV, scores, rows=rows, pool_kernel=7)
        ctx.score_baseline([req], ikv.BASE_STREAMING, scores)
        ctx.select_evict([req], scores, freed, nf, nk)
        q = torch.randn((5, shape.Hq, shape.D), device="cuda").to(dt)
        out = torch.empty_like(q)
        reads = torch.zeros(2, dtype=torch.int64, device="cuda")
        r = ikv.make_request(1, S_dev, s.N + 5, s.pi, s.qs, s.qe, s.spec.budget, s.pi)
        ctx.prefill_attn(0, r, s.N, q, out, 1.0 / math.sqrt(shape.D), reads)
    torch.cuda.synchronize()
    print("ok", shape, "n_kept", int(nk.item()))


if __name__ == "__main__":
    run(wl.tiny(), True, 0)
    run(wl.small(seed=7, shape=wl.ModelShape(3, 8, 2, 128, "bf16"), n_tokens=900, budget=250, decode_tokens=8, kv_dtype="bf16"), True, 2)
    run(wl.small(seed=9, shape=wl.ModelShape(2, 10, 2, 128, "bf16"), n_tokens=700, budget=200, decode_tokens=8, kv_dtype="bf16"), True, 0)
