"""-m gpu parity of the SURVEY 8(f) follow-ups against oracle/ikv_oracle_next.c: multi-row scorer (NEXT-1), prefill
attention through the slot map with KV-read counters (NEXT-2), baseline scorers on the dead-slot substrate (NEXT-3)."""
import math

import numpy as np
import pytest
import torch

from paper_2606_09916_b200 import workloads as wl
from tests import gpu_common as gc

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ikv():
    from paper_2606_09916_b200 import ikv as m
    return m


def _setup(oracle, shape, n_tokens=1500, budget=400, seed=61):
    w = wl.small(seed=seed, shape=shape, n_tokens=n_tokens, budget=budget, kv_dtype=shape.kv_dtype)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    M = gc.fold_memory_oracle(oracle, s)
    S = s.slot_map[:s.N].clone()
    rng = np.random.default_rng(seed)
    S[torch.from_numpy(rng.choice(s.N, size=s.N // 9, replace=False))] = w.dead_slot
    return w, kp, vp, ctx, s, M, S


SHAPES = [("d128g4", wl.ModelShape(3, 8, 2, 128, "bf16")), ("d64g2", wl.ModelShape(2, 4, 2, 64, "bf16")),
          ("d128g5", wl.ModelShape(2, 10, 2, 128, "bf16"))]


@pytest.mark.parametrize("name,shape", SHAPES, ids=[n for n, _ in SHAPES])
@pytest.mark.parametrize("R", [1, 4, 7, 32])
def test_multirow_scorer_matches_oracle(ikv, oracle, name, shape, R):
    """R = 1: one single-row pass; R = 7, 32: banks of 128 / G rows on tcgen05 (R = 32 at G = 5 needs two banks); R = 4
    is forced through the tcgen05 path (IKV_TUNE_ROWS_TC = 2)."""
    w, kp, vp, ctx, s, M, S = _setup(oracle, shape)
    if R == 4:
        ctx.tune(ikv.TUNE_ROWS_TC, 2)
    S_dev = S.cuda()
    req = gc.request(ikv, s, S_dev)
    g = gc.oracle_geom(oracle, w)
    rows = torch.randn((R, shape.L, shape.Hq, shape.D), generator=torch.Generator().manual_seed(R))
    wt = (0.25 + torch.rand(R, generator=torch.Generator().manual_seed(R + 1))).tolist()
    scores = torch.full((s.N,), 3.0, device="cuda")
    ctx.score_rows([req], rows.cuda().contiguous(), wt, scores)
    cls, _ = oracle.partition(S.numpy(), w.dead_slot, s.pi, s.qs, s.qe)
    want = oracle.multirow_score(g, kp, rows.double().numpy(), wt, S.numpy(), cls)
    want = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, want))
    mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, f"{name} R={R}")
    print(f"[{name} R={R}] multi-row score max abs err {mabs:.3e} rel {mrel:.3e}")
    if R >= 4:   # the cp.async gather warps (IKV_TUNE_ROWS_TC = 3) feed the tensor cores the same operands as TMA gather4
        ctx.tune(ikv.TUNE_ROWS_TC, 3)
        again = torch.full((s.N,), 3.0, device="cuda")
        ctx.score_rows([req], rows.cuda().contiguous(), wt, again)
        assert torch.equal(scores.view(torch.int32), again.view(torch.int32))


def test_multirow_tc_several_tile_pairs(ikv, oracle):
    """40,000 tokens: more than 2 x 148 tiles of 128, so the CTAs of the tcgen05 scorer walk two pairs of tiles (the
    gather runs ahead into the next pair); ragged last tile, dead positions, 5 rows at G = 2 (10 of 128 bank rows).
    Checked against the oracle and against the row-by-row path."""
    shape = wl.ModelShape(1, 2, 1, 64, "bf16")
    w, kp, vp, ctx, s, M, S = _setup(oracle, shape, n_tokens=40000, budget=1000)
    S_dev = S.cuda()
    req = gc.request(ikv, s, S_dev)
    g = gc.oracle_geom(oracle, w)
    R = 5
    rows = torch.randn((R, shape.L, shape.Hq, shape.D), generator=torch.Generator().manual_seed(3))
    wt = [0.5, 1.0, 0.0, 2.0, 0.25]
    ctx.tune(ikv.TUNE_ROWS_TC, 2)
    scores = torch.full((s.N,), 3.0, device="cuda")
    ctx.score_rows([req], rows.cuda().contiguous(), wt, scores)
    cls, _ = oracle.partition(S.numpy(), w.dead_slot, s.pi, s.qs, s.qe)
    want = oracle.multirow_score(g, kp, rows.double().numpy(), wt, S.numpy(), cls)
    want = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, want))
    mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, "several pairs")
    print(f"[several pairs] multi-row score max abs err {mabs:.3e} rel {mrel:.3e}")
    ctx.tune(ikv.TUNE_ROWS_TC, 3)   # cp.async gather warps: bit-identical
    again = torch.full((s.N,), 3.0, device="cuda")
    ctx.score_rows([req], rows.cuda().contiguous(), wt, again)
    assert torch.equal(scores.view(torch.int32), again.view(torch.int32))
    ctx.tune(ikv.TUNE_ROWS_TC, 0)
    ref = torch.empty_like(scores)
    ctx.score_rows([req], rows.cuda().contiguous(), wt, ref)
    fin = torch.isfinite(ref)
    assert torch.equal(torch.isfinite(scores), fin)
    assert torch.allclose(scores[fin], ref[fin], rtol=1e-4, atol=1e-6)


def test_multirow_single_row_is_the_memory_scorer_bit_for_bit(ikv, oracle):
    """R = 1 with the session's QueryMemory as the row reproduces ikv_score(IKV_MODE_MEMORY) exactly (Eq. 3)."""
    w, kp, vp, ctx, s, M, S = _setup(oracle, SHAPES[0][1])
    S_dev = S.cuda()
    req = gc.request(ikv, s, S_dev)
    base = torch.empty(s.N, device="cuda")
    ctx.score([req], ikv.MODE_MEMORY, base)
    rows = ctx.session_get_memory(s.spec.session_id)[None].cuda().contiguous()
    got = torch.empty(s.N, device="cuda")
    ctx.score_rows([req], rows, [1.0], got)
    assert torch.equal(base.view(torch.int32), got.view(torch.int32))


def _select_matches(ikv, oracle, ctx, w, s, S, got_scores, budget):
    """select / evict on the GPU's baseline scores is bit-exact with the oracle's selection on the same scores."""
    S_dev = S.cuda()
    req = gc.request(ikv, s, S_dev, budget=budget)
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    ctx.select_evict([req], got_scores, freed, nf, nk)
    cls, _ = oracle.partition(S.numpy(), w.dead_slot, s.pi, s.qs, s.qe)
    keep, n_kept = oracle.select(got_scores.cpu().numpy(), cls, budget)
    S2, _, freed_o = oracle.rewrite(S.numpy(), w.dead_slot, keep, s.pi, w.n_slots)
    assert nk.item() == n_kept and np.array_equal(S_dev.cpu().numpy(), S2)
    assert np.array_equal(freed.cpu().numpy()[:nf.item()], freed_o)
    return keep.astype(bool)


def test_streaming_baseline(ikv, oracle):
    w, kp, vp, ctx, s, M, S = _setup(oracle, SHAPES[1][1], n_tokens=2100, budget=500)
    S[:3] = s.slot_map[:3]                              # positions 0..2 live; they sit in the protected prefix anyway
    sn = S.numpy()
    S_dev = S.cuda()
    # no protected prefix, so that the sink rule is what keeps the first four positions
    req = ikv.make_request(s.spec.session_id, S_dev, s.N, 0, s.qs, s.qe, 500, 0)
    scores = torch.empty(s.N, device="cuda")
    ctx.score_baseline([req], ikv.BASE_STREAMING, scores, n_sink=4)
    cls, _ = oracle.partition(sn, w.dead_slot, 0, s.qs, s.qe)
    want = oracle.streaming_scores(cls, 4)
    want = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, want)).astype(np.float32)
    assert np.array_equal(scores.cpu().numpy(), want)                       # integer-valued: exact


@pytest.mark.parametrize("kind", ["snapkv", "h2o"])
def test_snapkv_and_h2o_baselines(ikv, oracle, kind):
    shape = SHAPES[0][1]
    w, kp, vp, ctx, s, M, S = _setup(oracle, shape, n_tokens=1800, budget=450)
    S_dev = S.cuda()
    req = gc.request(ikv, s, S_dev, budget=450)
    g = gc.oracle_geom(oracle, w)
    W = 32 if kind == "snapkv" else 12
    rows = torch.randn((W, shape.L, shape.Hq, shape.D), generator=torch.Generator().manual_seed(12))
    scores = torch.empty(s.N, device="cuda")
    cls, _ = oracle.partition(S.numpy(), w.dead_slot, s.pi, s.qs, s.qe)
    mass = oracle.multirow_score(g, kp, rows.double().numpy(), np.ones(W), S.numpy(), cls)
    if kind == "snapkv":
        ctx.score_baseline([req], ikv.BASE_SNAPKV, scores, rows=rows.cuda().contiguous(), pool_kernel=7)
        want = oracle.maxpool_candidates(mass, cls, 7)
    else:
        ctx.score_baseline([req], ikv.BASE_H2O, scores, rows=rows.cuda().contiguous(), recent_ratio=0.5, recent_floor=64)
        want = oracle.h2o_scores(mass, cls, 450, 0.5, 64)
    want = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, want))
    mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, kind)
    print(f"[{kind}] baseline score max abs err {mabs:.3e} rel {mrel:.3e}")
    keep = _select_matches(ikv, oracle, ctx, w, s, S, scores, 450)
    if kind == "h2o":                                   # the recent floor is kept whatever the masses are
        cand = np.nonzero(cls == oracle.CAND)[0]
        n_recent = max(64, int(math.floor(0.5 * (450 - (cls == oracle.FORCED).sum()) + 0.5)))
        assert keep[cand[-n_recent:]].all()


@pytest.mark.parametrize("name,shape", SHAPES, ids=[n for n, _ in SHAPES])
def test_prefill_attention_matches_oracle(ikv, oracle, name, shape):
    """A chunk of 70 query rows right after a prune (the survivor list is cached, the chunk's positions are read from the
    slot map), and a chunk that starts before the cached range (rescan), with dead positions inside the chunk; KV-read
    counters accumulate over both calls."""
    w = wl.small(seed=71, shape=shape, n_tokens=1300, budget=300, decode_tokens=80, kv_dtype="bf16")
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    g = gc.oracle_geom(oracle, w)
    full = s.slot_map.clone()
    full[s.N + 5] = w.dead_slot                           # a dead position inside the chunk
    S_dev = full.cuda()
    scores = torch.empty(s.N, device="cuda")
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    req = gc.request(ikv, s, S_dev)
    ctx.score([req], ikv.MODE_MEMORY, scores)
    ctx.select_evict([req], scores, freed, nf, nk)
    scale = 1.0 / math.sqrt(shape.D)
    reads = torch.zeros(2, dtype=torch.int64, device="cuda")
    want_raw = want_eff = 0
    for q_pos0, n_q, layer in ((s.N, 70, 0), (s.N - 40, 50, shape.L - 1)):
        q = torch.randn((n_q, shape.Hq, shape.D), generator=torch.Generator().manual_seed(q_pos0)).to(torch.bfloat16)
        out = torch.empty((n_q, shape.Hq, shape.D), dtype=torch.bfloat16, device="cuda")
        r = gc.request(ikv, s, S_dev, seq_len=q_pos0 + n_q)
        ctx.prefill_attn(layer, r, q_pos0, q.cuda(), out, scale, reads)
        torch.cuda.synchronize()
        S_host = S_dev.cpu().numpy()
        want, raw, eff = oracle.prefill(g, kp, vp, layer, S_host, q_pos0, q.float().numpy(), scale)
        want_raw += raw
        want_eff += eff
        err = gc.assert_decode_close(out.float().cpu().numpy(), want, True, f"{name} prefill at {q_pos0}")
        print(f"[{name}] prefill chunk at {q_pos0} x {n_q}: max abs err {err:.3e}")
    assert reads.cpu().tolist() == [want_raw, want_eff]      # integer counters: exact


def test_prefill_tiled_long_chunk_and_row_by_row_agree(ikv, oracle):
    """A 300-row chunk (ten 32-row blocks, the last one ragged) far behind a stale survivor list, dead positions inside
    the chunk and before it: the tcgen05 kernel, the mma.sync tiled kernel (IKV_TUNE_PREFILL_TILED = 2) and the
    row-by-row path (= 0) all agree with the oracle; a first chunk at position 0 (empty survivor list) works too."""
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    w = wl.small(seed=73, shape=shape, n_tokens=2600, budget=700, decode_tokens=320, kv_dtype="bf16")
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    g = gc.oracle_geom(oracle, w)
    full = s.slot_map.clone()
    rng = np.random.default_rng(5)
    full[torch.from_numpy(rng.choice(s.N + 300, size=500, replace=False))] = w.dead_slot
    S_dev = full.cuda()
    scale = 1.0 / math.sqrt(shape.D)
    for q_pos0, n_q, layer in ((s.N, 300, 1), (0, 45, 0)):
        q = torch.randn((n_q, shape.Hq, shape.D), generator=torch.Generator().manual_seed(q_pos0 + 1)).to(torch.bfloat16)
        r = gc.request(ikv, s, S_dev, seq_len=q_pos0 + n_q)
        outs = []
        for tiled in (1, 2, 0, 3, 4, 5):   # tcgen05 kernel (TMA gather4 producers), mma.sync tiled kernel, row by row,
                                           # tcgen05 kernel with the cp.async producers, with TMA producers and one M
                                           # tile per CTA, with TMA producers and two M tiles per CTA
            ctx.tune(ikv.TUNE_PREFILL_TILED, tiled)
            out = torch.full((n_q, shape.Hq, shape.D), float("nan"), dtype=torch.bfloat16, device="cuda")
            reads = torch.zeros(2, dtype=torch.int64, device="cuda")
            ctx.prefill_attn(layer, r, q_pos0, q.cuda(), out, scale, reads)
            torch.cuda.synchronize()
            outs.append((out.float().cpu().numpy(), reads.cpu().tolist()))
        want, raw, eff = oracle.prefill(g, kp, vp, layer, S_dev.cpu().numpy(), q_pos0, q.float().numpy(), scale)
        e1 = gc.assert_decode_close(outs[0][0], want, True, f"tcgen05 prefill at {q_pos0}")
        e2 = gc.assert_decode_close(outs[1][0], want, True, f"mma.sync prefill at {q_pos0}")
        e0 = gc.assert_decode_close(outs[2][0], want, True, f"row-by-row prefill at {q_pos0}")
        e3 = gc.assert_decode_close(outs[3][0], want, True, f"tcgen05 (cp.async producers) prefill at {q_pos0}")
        e4 = gc.assert_decode_close(outs[4][0], want, True, f"tcgen05 (one M tile per CTA) prefill at {q_pos0}")
        e5 = gc.assert_decode_close(outs[5][0], want, True, f"tcgen05 (two M tiles per CTA) prefill at {q_pos0}")
        assert all(o[1] == [raw, eff] for o in outs)
        # both producer kinds hand the tensor cores the same operands: bit-identical outputs for the same tiling
        assert np.array_equal(outs[4][0], outs[3][0]) and e4 == e3
        print(f"prefill at {q_pos0} x {n_q}: max abs err tcgen05 {e1:.3e} (cp.async producers {e3:.3e}, two M tiles {e5:.3e}), mma.sync {e2:.3e}, "
              f"row by row {e0:.3e}")


@pytest.mark.parametrize("name,shape", [("d128g1", wl.ModelShape(2, 2, 2, 128, "bf16")), ("d64g8", wl.ModelShape(2, 16, 2, 64, "bf16")),
                                        ("d128g8", wl.ModelShape(1, 8, 1, 128, "bf16")), ("d64g4", wl.ModelShape(2, 8, 2, 64, "bf16"))],
                         ids=["d128g1", "d64g8", "d128g8", "d64g4"])
def test_prefill_tcgen05_head_layouts(ikv, oracle, name, shape):
    """k_prefill_tc on the remaining tile shapes (128 rows x 1 head, 16 rows x 8 heads, D = 64): chunks of 1, 33 and 150
    rows over several splits and tiles (the 150-row chunk lags the survivor list and crosses row blocks), against the
    oracle and against the mma.sync kernel."""
    w = wl.small(seed=81, shape=shape, n_tokens=2100, budget=500, decode_tokens=200, kv_dtype="bf16")
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    g = gc.oracle_geom(oracle, w)
    full = s.slot_map.clone()
    rng = np.random.default_rng(9)
    full[torch.from_numpy(rng.choice(s.N + 200, size=400, replace=False))] = w.dead_slot
    S_dev = full.cuda()
    scale = 1.0 / math.sqrt(shape.D)
    for q_pos0, n_q in ((s.N, 1), (s.N + 1, 33), (s.N + 40, 150)):
        q = torch.randn((n_q, shape.Hq, shape.D), generator=torch.Generator().manual_seed(q_pos0)).to(torch.bfloat16)
        r = gc.request(ikv, s, S_dev, seq_len=q_pos0 + n_q)
        outs = []
        for tiled in (1, 2, 3, 4, 5):
            ctx.tune(ikv.TUNE_PREFILL_TILED, tiled)
            out = torch.full((n_q, shape.Hq, shape.D), float("nan"), dtype=torch.bfloat16, device="cuda")
            ctx.prefill_attn(shape.L - 1, r, q_pos0, q.cuda(), out, scale)
            torch.cuda.synchronize()
            outs.append(out.float().cpu().numpy())
        want, _, _ = oracle.prefill(g, kp, vp, shape.L - 1, S_dev.cpu().numpy(), q_pos0, q.float().numpy(), scale)
        e1 = gc.assert_decode_close(outs[0], want, True, f"{name} tcgen05 prefill at {q_pos0} x {n_q}")
        e2 = gc.assert_decode_close(outs[1], want, True, f"{name} mma.sync prefill at {q_pos0} x {n_q}")
        assert np.array_equal(outs[3], outs[2]), f"{name}: TMA gather4 and cp.async producers disagree"
        gc.assert_decode_close(outs[3], want, True, f"{name} tcgen05 (one M tile per CTA) prefill at {q_pos0} x {n_q}")
        gc.assert_decode_close(outs[4], want, True, f"{name} tcgen05 (two M tiles per CTA) prefill at {q_pos0} x {n_q}")
        print(f"[{name}] prefill at {q_pos0} x {n_q}: max abs err tcgen05 {e1:.3e}, mma.sync {e2:.3e}")


def test_prefill_single_split_writes_the_output_itself(ikv, oracle):
    """Enough (row block, KV head) pairs to fill the SMs with one split each: k_prefill_tc then normalises and writes the
    output itself (no partials, no merge launch).  700 rows at 8 KV heads, G = 4: one M tile per CTA (22 blocks), two
    M tiles per CTA (11 blocks) and the cp.async producers, all against the oracle; ragged last block, dead positions."""
    shape = wl.ModelShape(1, 32, 8, 128, "bf16")
    w = wl.small(seed=91, shape=shape, n_tokens=1500, budget=600, decode_tokens=720, kv_dtype="bf16")
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    g = gc.oracle_geom(oracle, w)
    full = s.slot_map.clone()
    rng = np.random.default_rng(17)
    full[torch.from_numpy(rng.choice(s.N + 700, size=450, replace=False))] = w.dead_slot
    S_dev = full.cuda()
    scale = 1.0 / math.sqrt(shape.D)
    q_pos0, n_q = s.N, 700
    q = torch.randn((n_q, shape.Hq, shape.D), generator=torch.Generator().manual_seed(5)).to(torch.bfloat16)
    r = gc.request(ikv, s, S_dev, seq_len=q_pos0 + n_q)
    want, _, _ = oracle.prefill(g, kp, vp, 0, S_dev.cpu().numpy(), q_pos0, q.float().numpy(), scale)
    outs = {}
    for tiled in (1, 4, 3):
        ctx.tune(ikv.TUNE_PREFILL_TILED, tiled)
        out = torch.full((n_q, shape.Hq, shape.D), float("nan"), dtype=torch.bfloat16, device="cuda")
        ctx.prefill_attn(0, r, q_pos0, q.cuda(), out, scale)
        torch.cuda.synchronize()
        outs[tiled] = out.float().cpu().numpy()
        err = gc.assert_decode_close(outs[tiled], want, True, f"single-split prefill, IKV_TUNE_PREFILL_TILED = {tiled}")
        print(f"single-split prefill (tiled = {tiled}): max abs err {err:.3e}")
    assert np.array_equal(outs[4], outs[3])


@pytest.mark.parametrize("n,pos_rate", [(1, 1.0), (700, 0.05), (33000, 0.004), (5000, 0.0), (40, 0.5)])
def test_train_loss_matches_oracle(ikv, oracle, n, pos_rate):
    """Eq. 8 and dL/ds (ikv_train_loss) against the fp64 oracle: terms within 1e-5 relative, gradient within
    1e-7 + 1e-4 |g|; quantised scores (ties among the hard negatives), excluded labels, fewer than 64 negatives, no
    positives; run twice: bit-identical."""
    rng = np.random.default_rng(n)
    s = (np.round(rng.standard_normal(n) * 8) / 4).astype(np.float32)
    y = (rng.random(n) < pos_rate).astype(np.int32)
    y[rng.random(n) < 0.1] = -100
    rows = rng.standard_normal((12, 64)).astype(np.float32) * 0.2
    want_t, want_g = oracle.train_loss(s.astype(np.float64), y, rows.astype(np.float64))
    w = wl.small(seed=3, shape=wl.ModelShape(1, 2, 1, 64, "bf16"), n_tokens=64, budget=16, kv_dtype="bf16")
    gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    outs = []
    for _ in range(2):
        terms = torch.full((5,), float("nan"), device="cuda")
        grad = torch.full((n,), float("nan"), device="cuda")
        ctx.train_loss(torch.from_numpy(s).cuda(), torch.from_numpy(y).cuda(), terms, grad, torch.from_numpy(rows).cuda())
        torch.cuda.synchronize()
        outs.append((terms.cpu().numpy().astype(np.float64), grad.cpu().numpy().astype(np.float64)))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    got_t, got_g = outs[0]
    assert np.all(np.abs(got_t - want_t) <= 1e-5 * np.maximum(1e-3, np.abs(want_t))), (got_t, want_t)
    assert np.all(np.abs(got_g - want_g) <= 1e-7 + 1e-4 * np.abs(want_g)), np.abs(got_g - want_g).max()
    assert np.all(got_g[(y != 0) & (y != 1)] == 0.0)
    print(f"[n={n}] Eq. 8 terms {got_t}, max |dL/ds err| {np.abs(got_g - want_g).max():.2e}")
