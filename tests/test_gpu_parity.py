"""-m gpu parity tests: libikv (through the C-ABI binding) vs the CPU oracle, element by element, on the same
seeded inputs.  Sizes span several tiles plus a ragged tail and finish in seconds on the oracle."""
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


SHAPES = [
    ("tiny", None),
    ("bf16_d128_g4", wl.ModelShape(3, 8, 2, 128, "bf16")),
    ("bf16_d64_g2", wl.ModelShape(2, 4, 2, 64, "bf16")),
    ("bf16_d128_g5", wl.ModelShape(2, 10, 2, 128, "bf16")),
    ("bf16_d128_g1", wl.ModelShape(2, 3, 3, 128, "bf16")),
    ("bf16_d128_g8", wl.ModelShape(2, 16, 2, 128, "bf16")),
    ("f32_d128_g4", wl.ModelShape(2, 8, 2, 128, "f32")),
    ("bf16_d128_h12", wl.ModelShape(2, 24, 12, 128, "bf16")),   # more KV heads than warps
    ("bf16_d128_g5_h8", wl.ModelShape(2, 40, 8, 128, "bf16")),  # configs[2] head layout: one KV head per logit warp
]


def build(name, shape, seed=123, n_tokens=1500, budget=400):
    if name == "tiny":
        return wl.tiny()
    return wl.small(seed=seed, shape=shape, n_tokens=n_tokens, budget=budget, kv_dtype=shape.kv_dtype)


def run_memory(ikv, oracle, w):
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    M = gc.fold_memory_oracle(oracle, s)
    return ctx, s, M, kp, vp


# ------------------------------------------------------------------------------------------- a0
def test_memory_update_matches_oracle(ikv, oracle):
    w = build("bf16_d128_g4", SHAPES[1][1])
    ctx, s, M, _, _ = run_memory(ikv, oracle, w)
    got = ctx.session_get_memory(s.spec.session_id).numpy()
    assert np.abs(got - M).max() < 2e-6
    assert np.allclose(np.linalg.norm(got, axis=-1), 1.0, atol=1e-5)
    # bf16 query rows take the same path
    ctx.session_open(99)
    rows = s.mem_rows[:4].to(torch.bfloat16)
    ctx.memory_update(99, rows.cuda().contiguous())
    M2 = np.zeros_like(M)
    oracle.memory_update(M2, rows.float().numpy(), 0.5)
    assert np.abs(ctx.session_get_memory(99).numpy() - M2).max() < 2e-6
    # fork copies the state
    ctx.session_fork(s.spec.session_id, 100)
    torch.cuda.synchronize()
    assert np.array_equal(ctx.session_get_memory(100).numpy(), got)


# ------------------------------------------------------------------------------------------- a1-a3
@pytest.mark.parametrize("name,shape", SHAPES, ids=[n for n, _ in SHAPES])
def test_rule_score_matches_oracle(ikv, oracle, name, shape):
    w = build(name, shape)
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    S = s.slot_map[:s.N].clone()
    rng = np.random.default_rng(4)
    dead_idx = rng.choice(s.N, size=s.N // 7, replace=False)
    S[torch.from_numpy(dead_idx)] = w.dead_slot          # dead positions from an earlier round (also in prefix/span)
    S_dev = S.cuda()
    scores = torch.full((s.N,), 7.0, device="cuda")
    rule = torch.full((s.N,), 7.0, device="cuda")
    req = gc.request(ikv, s, S_dev)
    ctx.score([req], ikv.MODE_MEMORY, scores, rule)
    torch.cuda.synchronize()
    want, want_rule = oracle.score(gc.oracle_geom(oracle, w), kp, M, S.numpy(), s.pi, s.qs, s.qe, want_rule=True)
    mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, name)
    assert np.allclose(rule.cpu().numpy(), want_rule, rtol=1e-3, atol=1e-4)
    fin = np.isfinite(want)
    assert abs(scores.cpu().numpy()[fin].sum() - w.shape.L * w.shape.Hq) < 1e-2     # P1 on the GPU side
    print(f"[{name}] rule score max abs err {mabs:.3e} max rel err {mrel:.3e}")


def test_query_mode_and_fresh_session(ikv, oracle):
    w = build("bf16_d128_g4", SHAPES[1][1])
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    S = s.slot_map[:s.N]
    S_dev = S.cuda()
    scores = torch.empty(s.N, device="cuda")
    req = gc.request(ikv, s, S_dev)
    ctx.score([req], ikv.MODE_QUERY, scores)
    Mq = oracle.query_encoding(s.updates()[-1].numpy())
    want = oracle.score(gc.oracle_geom(oracle, w), kp, Mq, S.numpy(), s.pi, s.qs, s.qe)
    gc.assert_scores_close(scores.cpu().numpy(), want, "query mode")
    # fresh session: M = 0 -> uniform L*Hq/|A| (P3)
    ctx.session_open(555)
    req2 = ikv.make_request(555, S_dev, s.N, s.pi, s.qs, s.qe, 100)
    ctx.score([req2], ikv.MODE_MEMORY, scores)
    got = scores.cpu().numpy()
    fin = np.isfinite(got)
    assert np.allclose(got[fin], w.shape.L * w.shape.Hq / fin.sum(), rtol=1e-5)


# ------------------------------------------------------------------------------------------- a4-a5
@pytest.mark.parametrize("name,shape", [SHAPES[0], SHAPES[1], SHAPES[2], SHAPES[3], SHAPES[8], SHAPES[5]],
                         ids=["tiny", "d128g4", "d64g2", "d128g5", "d128g5h8", "d128g8"])
def test_learnable_score_matches_oracle(ikv, oracle, name, shape):
    w = build(name, shape)
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    S = s.slot_map[:s.N].clone()
    S[s.qs + 1] = w.dead_slot                            # a dead query position: excluded from K^q
    S[s.pi + 5: s.pi + 50: 3] = w.dead_slot
    S_dev = S.cuda()
    g = gc.oracle_geom(oracle, w)
    wts = wl.residual_weights(w.shape.D, 31)
    ow = oracle.ResidualWeights(**wts)
    ctx.residual_load(wts)
    req = gc.request(ikv, s, S_dev)
    base = torch.empty(s.N, device="cuda")
    ctx.score([req], ikv.MODE_MEMORY, base)
    for flags, oflags in ((0, 0), (ikv.FLAG_NO_XATTN, oracle.FLAG_NO_XATTN), (ikv.FLAG_NO_RESIDUAL, oracle.FLAG_NO_RESIDUAL)):
        scores = torch.empty(s.N, device="cuda")
        ctx.score([req], ikv.MODE_LEARNABLE | flags, scores)
        want = oracle.score(g, kp, M, S.numpy(), s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, oflags, w=ow)
        mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, f"{name} flags={flags:#x}")
        print(f"[{name} flags={flags:#x}] learnable score max abs err {mabs:.3e} rel {mrel:.3e}")
        if flags == ikv.FLAG_NO_RESIDUAL:
            assert torch.equal(scores, base)             # alpha = 0 recovers the rule scorer exactly
    # explicit xattn_pos list (with a dead and an out-of-span entry)
    xp = torch.tensor([s.qs, s.qs + 1, s.pi + 5, s.pi + 6, s.qe - 1], dtype=torch.int32)
    xp_dev = xp.cuda()                                   # keep alive: the request only holds the raw pointer
    req_x = gc.request(ikv, s, S_dev, xattn=xp_dev)
    scores = torch.empty(s.N, device="cuda")
    ctx.score([req_x], ikv.MODE_LEARNABLE, scores)
    want = oracle.score(g, kp, M, S.numpy(), s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, 0, xattn_pos=xp.numpy(), w=ow)
    gc.assert_scores_close(scores.cpu().numpy(), want, "explicit xattn_pos")
    # zero-initialised head reproduces the rule score exactly
    ctx.residual_load(wl.residual_weights(w.shape.D, 31, zero_init=True))
    ctx.score([req], ikv.MODE_LEARNABLE, scores)
    assert torch.equal(scores, base)


# ------------------------------------------------------------------------------------------- a6-a7
def _select_case(ikv, oracle, ctx, w, s, S, scores_np, budget, radix, seq_len=None):
    N = len(S) if seq_len is None else seq_len
    S_dev = torch.from_numpy(S.copy()).cuda()
    valid = torch.full((max(N, 1),), 9, dtype=torch.uint8, device="cuda")
    freed = torch.full((max(N, 1),), -7, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    pi, qs, qe = min(s.pi, N), min(max(s.qs, min(s.pi, N)), N), min(s.qe, N)
    req = ikv.make_request(s.spec.session_id, S_dev, N, pi, qs, qe, budget, radix, valid_mask=valid)
    sc_dev = torch.from_numpy(scores_np[:max(N, 1)].copy()).cuda()
    k_sum = w.k_pool.view(torch.int16 if w.k_pool.dtype == torch.bfloat16 else torch.int32).long().sum().item()
    ctx.select_evict([req], sc_dev, freed, nf, nk)
    torch.cuda.synchronize()
    cls, _ = oracle.partition(S[:N], w.dead_slot, pi, qs, qe)
    keep, n_kept = oracle.select(scores_np[:N], cls, budget)
    S2, valid_o, freed_o = oracle.rewrite(S[:N], w.dead_slot, keep, radix, w.n_slots)
    assert nk.item() == n_kept
    assert np.array_equal(S_dev.cpu().numpy()[:N], S2)                       # slot map bit-exact
    assert np.array_equal(valid.cpu().numpy()[:N], valid_o)
    assert nf.item() == len(freed_o)
    assert np.array_equal(freed.cpu().numpy()[:len(freed_o)], freed_o)      # freed list bit-exact, in order
    k_sum2 = w.k_pool.view(torch.int16 if w.k_pool.dtype == torch.bfloat16 else torch.int32).long().sum().item()
    assert k_sum == k_sum2                                                   # no K byte moved
    return S2, n_kept


def test_select_evict_bit_exact_on_oracle_scores(ikv, oracle):
    w = build("bf16_d128_g4", SHAPES[1][1], n_tokens=5000, budget=1300)
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    rng = np.random.default_rng(8)
    S = s.slot_map[:s.N].numpy().copy()
    S[rng.choice(s.N, 600, replace=False)] = w.dead_slot
    S[3000] = S[1000]                                     # alias with a (to be) kept position
    S[3500] = S[3400]                                     # alias between two dropped positions
    sc = oracle.score(gc.oracle_geom(oracle, w), kp, M, S, s.pi, s.qs, s.qe)
    sc[1000] = 10.0
    sc[[3000, 3400, 3500]] = -10.0
    S2, nk = _select_case(ikv, oracle, ctx, w, s, S, sc, 1300, radix=777)
    assert nk == 1300
    # second round on the pruned map is a no-op (N > C but live == C)
    _select_case(ikv, oracle, ctx, w, s, S2, sc, 1300, radix=777)


@pytest.mark.parametrize("case", ["ties", "all_equal", "nan_inf", "skip_N_le_C", "forced_gt_C", "cstar_zero",
                                  "keep_all_live", "empty", "one_token", "budget_zero"])
def test_select_evict_edge_cases(ikv, oracle, case):
    w = build("bf16_d64_g2", SHAPES[2][1], n_tokens=2100, budget=500)
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    rng = np.random.default_rng(len(case))
    N = s.N
    S = s.slot_map[:N].numpy().copy()
    sc = rng.standard_normal(N).astype(np.float32)
    budget, radix, seq_len = 500, s.pi, None
    if case == "ties":
        sc = np.round(sc * 2).astype(np.float32) / 2          # heavy ties, incl. +-0
        sc[::17] = -0.0
    elif case == "all_equal":
        sc[:] = 0.03125
    elif case == "nan_inf":
        sc[rng.choice(N, 300, replace=False)] = np.nan
        sc[rng.choice(N, 50, replace=False)] = np.inf
        sc[rng.choice(N, 50, replace=False)] = -np.inf
        budget = 1900                                           # threshold lands inside the NaN block
    elif case == "skip_N_le_C":
        budget = N
        S[rng.choice(N, 100, replace=False)] = w.dead_slot
    elif case == "forced_gt_C":
        budget = 20                                             # |F| = pi + span > C  (R14)
    elif case == "cstar_zero":
        budget = s.pi + (s.qe - s.qs)
    elif case == "keep_all_live":
        S[rng.choice(N, 1800, replace=False)] = w.dead_slot     # live < C although N > C
    elif case == "empty":
        seq_len = 0
    elif case == "one_token":
        seq_len = 1
        budget = 0
    elif case == "budget_zero":
        budget = 0
    _select_case(ikv, oracle, ctx, w, s, S, sc, budget, radix, seq_len)


@pytest.mark.parametrize("n_tokens", [33000, 70001, 131072, 140003])
def test_score_select_large_maps(ikv, oracle, n_tokens):
    """Long slot maps: every register-blocking variant of the cluster kernels (4 / 8 / 16 positions per thread) and
    the single-CTA kernels beyond 131,072 positions; ragged tails; heavy ties; dead positions."""
    w = build("bf16_d64_g2", SHAPES[2][1], n_tokens=n_tokens, budget=8192)
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    rng = np.random.default_rng(n_tokens)
    S = s.slot_map[:s.N].numpy().copy()
    S[rng.choice(s.N, s.N // 5, replace=False)] = w.dead_slot
    S_dev = torch.from_numpy(S.copy()).cuda()
    scores = torch.empty(s.N, device="cuda")
    req = gc.request(ikv, s, S_dev, budget=8192)
    ctx.score([req], ikv.MODE_MEMORY, scores)
    want = oracle.score(gc.oracle_geom(oracle, w), kp, M, S, s.pi, s.qs, s.qe)
    gc.assert_scores_close(scores.cpu().numpy(), want, f"N={n_tokens}")
    sc = np.round(rng.standard_normal(s.N) * 8).astype(np.float32) / 8      # ties across CTA boundaries
    S[s.N - 3] = S[s.pi + 7]                                                # an alias far away in another CTA
    _select_case(ikv, oracle, ctx, w, s, S, sc, 8192, radix=s.pi + 1000)


def test_end_to_end_prune_kept_set(ikv, oracle):
    """GPU scores -> GPU select vs oracle scores -> oracle select: the kept sets may differ only at tokens whose
    oracle score lies within the score tolerance of the C*-th threshold (north_star)."""
    w = build("bf16_d128_g4", SHAPES[1][1], n_tokens=4000, budget=1000)
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    S = s.slot_map[:s.N].numpy().copy()
    S_dev = torch.from_numpy(S.copy()).cuda()
    scores = torch.empty(s.N, device="cuda")
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    req = gc.request(ikv, s, S_dev, budget=1000)
    ctx.score([req], ikv.MODE_MEMORY, scores)
    ctx.select_evict([req], scores, freed, nf, nk)
    torch.cuda.synchronize()
    ev = oracle.prune_event(gc.oracle_geom(oracle, w), kp, M, S, s.pi, s.qs, s.qe, 1000, s.pi)
    assert nk.item() == ev["n_kept"] == 1000
    got_keep = S_dev.cpu().numpy() != w.dead_slot
    want_keep = ev["keep"].astype(bool)
    diff = np.nonzero(got_keep != want_keep)[0]
    cand_scores = ev["scores"][np.isfinite(ev["scores"]) & want_keep]
    thr = cand_scores.min()
    tol = gc.SCORE_ATOL + gc.SCORE_RTOL * abs(thr)
    assert np.all(np.abs(ev["scores"][diff] - thr) <= 2 * tol)
    jacc = (got_keep & want_keep).sum() / (got_keep | want_keep).sum()
    planted = got_keep[s.planted_pos].mean()
    print(f"kept-set Jaccard {jacc:.4f}, {len(diff)} positions differ, planted kept {planted:.2f}")
    assert jacc > 0.9 and planted == 1.0                     # P15 (sanity)
    # positions: kept rows still point at their original slots
    assert np.array_equal(S_dev.cpu().numpy()[got_keep], S[got_keep])


# ------------------------------------------------------------------------------------------- a8
@pytest.mark.parametrize("name,shape", SHAPES, ids=[n for n, _ in SHAPES])
def test_decode_matches_oracle(ikv, oracle, name, shape):
    w = build(name, shape, n_tokens=1200, budget=300)
    ctx, s, M, kp, vp = run_memory(ikv, oracle, w)
    g = gc.oracle_geom(oracle, w)
    dt = w.k_pool.dtype
    full = s.slot_map.clone()                              # N + decode_tokens positions
    S_dev = full.cuda()
    scores = torch.empty(s.N, device="cuda")
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    req = gc.request(ikv, s, S_dev)
    scale = 1.0 / math.sqrt(w.shape.D)
    gen = torch.Generator().manual_seed(3)

    def check(seq_len, flags=0):
        S_host = S_dev.cpu().numpy()[:seq_len]
        for layer in range(w.shape.L):
            q = torch.randn((w.shape.Hq, w.shape.D), generator=gen).to(dt)
            out = torch.empty((1, w.shape.Hq, w.shape.D), dtype=dt, device="cuda")
            r = gc.request(ikv, s, S_dev, seq_len=seq_len, flags=flags)
            ctx.decode_attn(layer, [r], q.cuda()[None].contiguous(), out, scale)
            want = oracle.decode(g, kp, vp, layer, S_host, q.float().numpy(), scale)
            gc.assert_decode_close(out[0].float().cpu().numpy(), want, dt == torch.bfloat16,
                                   f"{name} layer {layer} seq_len {seq_len}")

    check(s.N)                                             # before any prune: list built from the slot map
    ctx.score([req], ikv.MODE_MEMORY, scores)
    ctx.select_evict([req], scores, freed, nf, nk)
    check(s.N)                                             # through the pruned map (cached survivor list)
    for extra in (1, 2, s.spec.decode_tokens):             # appended decode tokens are read from the slot map
        check(s.N + extra)
    S_dev[s.N + 1] = w.dead_slot                           # caller edits the map itself -> RESCAN
    S_dev[5] = w.dead_slot
    check(s.N + s.spec.decode_tokens, flags=ikv.REQ_RESCAN)


def test_decode_batched_and_empty(ikv, oracle):
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    specs = [wl.SessionSpec(10 + i, n, 8, 100, prefix_len=8, span_len=8) for i, n in enumerate([700, 64, 1, 333])]
    w = wl.make_workload(shape, specs, 17)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    g = gc.oracle_geom(oracle, w)
    maps, reqs = [], []
    for s in w.sessions:
        ctx.session_open(s.spec.session_id)
        m = s.slot_map[:s.N].clone()
        if s.N > 100:
            m[::3] = w.dead_slot
        maps.append(m.cuda())
        reqs.append(ikv.make_request(s.spec.session_id, maps[-1], s.N, 0, 0, 0, 100))
    # a request whose every position is dead -> zeros
    ctx.session_open(99)
    dead_map = torch.zeros(40, dtype=torch.int32, device="cuda")
    reqs.append(ikv.make_request(99, dead_map, 40, 0, 0, 0, 100))
    q = torch.randn((len(reqs), 8, 128), generator=torch.Generator().manual_seed(1)).to(torch.bfloat16)
    out = torch.empty((len(reqs), 8, 128), dtype=torch.bfloat16, device="cuda")
    ctx.decode_attn(1, reqs, q.cuda(), out, 0.0883883)
    torch.cuda.synchronize()
    for i, s in enumerate(w.sessions):
        want = oracle.decode(g, kp, vp, 1, maps[i].cpu().numpy(), q[i].float().numpy(), 0.0883883)
        gc.assert_decode_close(out[i].float().cpu().numpy(), want, True, f"request {i}")
    assert torch.count_nonzero(out[-1]) == 0


def test_prune_decode_chain_without_host_sync(ikv, oracle):
    """The kernels of the prune pass and of decode are all launched with programmatic stream serialization
    (R27).  Six turns of score -> select/evict -> three decode layers are enqueued back to back on one
    stream with no host synchronisation; the shared per-call scratch (candidate list, logits, fragment tables,
    split-K partials) is reused by every turn, so a kernel that ran ahead of its predecessor would corrupt a
    neighbouring turn.  Every turn is then checked against the oracle."""
    shape = wl.ModelShape(3, 8, 2, 128, "bf16")
    w = wl.small(seed=17, shape=shape, n_tokens=5000, budget=1200, kv_dtype="bf16")
    ctx, s, M, kp, vp = run_memory(ikv, oracle, w)
    g = gc.oracle_geom(oracle, w)
    wts = wl.residual_weights(w.shape.D, 31)
    ow = oracle.ResidualWeights(**wts)
    ctx.residual_load(wts)
    S0 = s.slot_map[:s.N].numpy().copy()
    n_turn = 6
    budgets = [1200, 900, 2000, 700, 1500, 1000]
    modes = [ikv.MODE_LEARNABLE, ikv.MODE_MEMORY] * 3
    S_dev = [torch.from_numpy(S0.copy()).cuda() for _ in range(n_turn)]
    scores = [torch.empty(s.N, device="cuda") for _ in range(n_turn)]
    freed = [torch.empty(s.N, dtype=torch.int32, device="cuda") for _ in range(n_turn)]
    nf = torch.zeros(n_turn, dtype=torch.int32, device="cuda")
    nk = torch.zeros(n_turn, dtype=torch.int32, device="cuda")
    q = torch.randn((n_turn, 3, 1, 8, 128), generator=torch.Generator().manual_seed(3)).to(torch.bfloat16)
    q_dev = q.cuda()
    out = torch.zeros((n_turn, 3, 1, 8, 128), dtype=torch.bfloat16, device="cuda")
    scale = 1 / math.sqrt(128)
    reqs = [gc.request(ikv, s, S_dev[t], budget=budgets[t]) for t in range(n_turn)]
    torch.cuda.synchronize()
    for t in range(n_turn):
        ctx.score([reqs[t]], modes[t], scores[t])
        ctx.select_evict([reqs[t]], scores[t], freed[t], nf[t:t + 1], nk[t:t + 1])
        for layer in range(3):
            ctx.decode_attn(layer, [reqs[t]], q_dev[t, layer], out[t, layer], scale)
    torch.cuda.synchronize()
    for t in range(n_turn):
        omode = oracle.MODE_LEARNABLE if modes[t] == ikv.MODE_LEARNABLE else oracle.MODE_MEMORY
        want = oracle.score(g, kp, M, S0, s.pi, s.qs, s.qe, omode, 0, w=ow)
        got = scores[t].cpu().numpy()
        gc.assert_scores_close(got, want, f"turn {t}")
        # select / rewrite are bit-exact on the scores the GPU produced
        cls, _ = oracle.partition(S0, w.dead_slot, s.pi, s.qs, s.qe)
        keep, n_kept = oracle.select(got, cls, budgets[t])
        S2, _, freed_o = oracle.rewrite(S0, w.dead_slot, keep, s.pi, w.n_slots)
        assert nk[t].item() == n_kept
        assert np.array_equal(S_dev[t].cpu().numpy(), S2), f"turn {t}: slot map"
        assert nf[t].item() == len(freed_o)
        assert np.array_equal(freed[t].cpu().numpy()[:len(freed_o)], freed_o)
        for layer in range(3):
            o = oracle.decode(g, kp, vp, layer, S2, q[t, layer, 0].float().numpy(), scale)
            gc.assert_decode_close(out[t, layer, 0].float().cpu().numpy(), o, True, f"turn {t} layer {layer}")


def test_decode_back_to_back_calls(ikv, oracle):
    """Programmatic dependent launch (R27): 48 layer calls enqueued back to back without any host
    synchronisation share the split-K scratch; each must still see only its own partials."""
    shape = wl.ModelShape(3, 8, 2, 128, "bf16")
    w = wl.small(seed=5, shape=shape, n_tokens=6000, budget=6000)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    g = gc.oracle_geom(oracle, w)
    s = w.sessions[0]
    ctx.session_open(s.spec.session_id)
    S = s.slot_map[:s.N].clone()
    S[::5] = w.dead_slot
    S_dev = S.cuda()
    n_calls = 48
    q = torch.randn((n_calls, 1, 8, 128), generator=torch.Generator().manual_seed(8)).to(torch.bfloat16)
    q_dev = q.cuda()
    out = torch.zeros((n_calls, 1, 8, 128), dtype=torch.bfloat16, device="cuda")
    scale = 1 / math.sqrt(128)
    # 32 calls of one length (an unbroken chain of programmatically launched kernels), then shrinking lengths (each of
    # those forces a rescan kernel in between)
    lens = [s.N] * 32 + [s.N - (i % 7) * 100 for i in range(n_calls - 32)]
    torch.cuda.synchronize()
    for i in range(n_calls):
        r = gc.request(ikv, s, S_dev, seq_len=lens[i], flags=ikv.REQ_RESCAN if i == 0 else 0)
        ctx.decode_attn(i % 3, [r], q_dev[i], out[i], scale)
    torch.cuda.synchronize()
    for i in range(n_calls):
        want = oracle.decode(g, kp, vp, i % 3, S.numpy()[:lens[i]], q[i, 0].float().numpy(), scale)
        gc.assert_decode_close(out[i, 0].float().cpu().numpy(), want, True, f"call {i}")


def test_decode_padded_list_and_long_append(ikv, oracle):
    """Survivor list shorter than its host-side bound (live < C < N: the padding entries must be masked), then more
    than 4096 positions appended after the select (the library rescans the map instead of walking the tail)."""
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    w = wl.make_workload(shape, [wl.SessionSpec(5, n_tokens=3000, n_mem_rows=4, budget=2000, prefix_len=16, span_len=16,
                                                decode_tokens=5000)], 23)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    g = gc.oracle_geom(oracle, w)
    s = w.sessions[0]
    ctx.session_open(5)
    S = s.slot_map.clone()
    rng = np.random.default_rng(2)
    S[torch.from_numpy(rng.choice(3000, 1800, replace=False))] = w.dead_slot      # live 1200 < C 2000 < N 3000
    S_dev = S.cuda()
    scores = torch.randn(3000, generator=torch.Generator().manual_seed(9)).cuda()
    freed = torch.empty(3000, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    req = ikv.make_request(5, S_dev, 3000, 16, 2984, 3000, 2000, 16)
    ctx.select_evict([req], scores, freed, nf, nk)
    assert nk.item() == 1200
    scale = 1 / math.sqrt(128)
    gen = torch.Generator().manual_seed(4)
    for seq_len in (3000, 3001, 3000 + 4096, 3000 + 4097, 8000):
        q = torch.randn((1, 8, 128), generator=gen).to(torch.bfloat16)
        out = torch.empty((1, 8, 128), dtype=torch.bfloat16, device="cuda")
        r = ikv.make_request(5, S_dev, seq_len, 16, 2984, 3000, 2000, 16)
        ctx.decode_attn(0, [r], q.cuda(), out, scale)
        want = oracle.decode(g, kp, vp, 0, S_dev.cpu().numpy()[:seq_len], q[0].float().numpy(), scale)
        gc.assert_decode_close(out[0].float().cpu().numpy(), want, True, f"seq_len {seq_len}")


def test_decode_many_unequal_requests(ikv, oracle):
    """40 requests (more than one launch holds) of very different lengths: splits are handed out in proportion."""
    shape = wl.ModelShape(1, 8, 2, 128, "bf16")
    lens = [17 + (i * 977) % 9000 for i in range(40)]
    specs = [wl.SessionSpec(200 + i, n, 4, 100, prefix_len=4, span_len=4) for i, n in enumerate(lens)]
    w = wl.make_workload(shape, specs, 29)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w, max_sessions=64)
    g = gc.oracle_geom(oracle, w)
    maps, reqs = [], []
    for i, s in enumerate(w.sessions):
        ctx.session_open(s.spec.session_id)
        m = s.slot_map[:s.N].clone()
        if i % 3 == 0:
            m[1::2] = w.dead_slot
        maps.append(m.cuda())
        reqs.append(ikv.make_request(s.spec.session_id, maps[-1], s.N, 0, 0, 0, 100))
    q = torch.randn((40, 8, 128), generator=torch.Generator().manual_seed(6)).to(torch.bfloat16)
    out = torch.empty((40, 8, 128), dtype=torch.bfloat16, device="cuda")
    scale = 1 / math.sqrt(128)
    ctx.decode_attn(0, reqs, q.cuda(), out, scale)
    torch.cuda.synchronize()
    for i in range(40):
        want = oracle.decode(g, kp, vp, 0, maps[i].cpu().numpy(), q[i].float().numpy(), scale)
        gc.assert_decode_close(out[i].float().cpu().numpy(), want, True, f"request {i} len {lens[i]}")


# ------------------------------------------------------------------------------------------- batches, host path, errors
def test_batched_score_select(ikv, oracle):
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    specs = [wl.SessionSpec(20 + i, n, 8, c, prefix_len=16, span_len=16, n_planted=5)
             for i, (n, c) in enumerate([(900, 300), (2000, 256), (130, 500)])]
    w = wl.make_workload(shape, specs, 19)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    g = gc.oracle_geom(oracle, w)
    tot = sum(s.N for s in w.sessions)
    maps = [s.slot_map[:s.N].clone().cuda() for s in w.sessions]
    reqs = []
    for s, m in zip(w.sessions, maps):
        gc.fold_memory_gpu(ctx, s)
        reqs.append(gc.request(ikv, s, m))
    scores = torch.empty(tot, device="cuda")
    freed = torch.empty(tot, dtype=torch.int32, device="cuda")
    nf = torch.zeros(3, dtype=torch.int32, device="cuda")
    nk = torch.zeros(3, dtype=torch.int32, device="cuda")
    ctx.score(reqs, ikv.MODE_MEMORY, scores)
    sc_host = scores.cpu().numpy()
    ctx.select_evict(reqs, scores, freed, nf, nk)
    torch.cuda.synchronize()
    off = 0
    for i, s in enumerate(w.sessions):
        M = gc.fold_memory_oracle(oracle, s)
        S = s.slot_map[:s.N].numpy()
        want = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe)
        gc.assert_scores_close(sc_host[off:off + s.N], want, f"request {i}")
        cls, _ = oracle.partition(S, 0, s.pi, s.qs, s.qe)
        keep, n_kept = oracle.select(sc_host[off:off + s.N], cls, s.spec.budget)
        S2, _, freed_o = oracle.rewrite(S, 0, keep, s.pi, w.n_slots)
        assert nk[i].item() == n_kept and nf[i].item() == len(freed_o)
        assert np.array_equal(maps[i].cpu().numpy(), S2)
        assert np.array_equal(freed.cpu().numpy()[off:off + len(freed_o)], freed_o)
        off += s.N


@pytest.mark.parametrize("mode_name", ["memory", "learnable"])
def test_batched_score_lanes(ikv, oracle, mode_name):
    """A batch on 1, 3 and 8 lanes (IKV_TUNE_BATCH_LANES: small kernels of different requests on internal streams, each
    lane with its own scratch) gives bit-identical scores, on a non-blocking stream with the default stream busy, and
    agrees with the oracle; an empty request sits in the middle of the batch."""
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    lens = [(700, 200), (4500, 256), (130, 64), (2300, 512), (1, 1), (5200, 300), (3100, 128)]
    specs = [wl.SessionSpec(60 + i, n, 8, c, prefix_len=min(16, n // 4), span_len=min(16, n // 4), n_planted=min(5, n // 8))
             for i, (n, c) in enumerate(lens)]
    w = wl.make_workload(shape, specs, 23)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w, max_sessions=16)
    rw = wl.residual_weights(shape.D, 77)
    ctx.residual_load(rw)
    g = gc.oracle_geom(oracle, w)
    maps = [s.slot_map[:s.N].clone().cuda() for s in w.sessions]
    reqs = []
    for s, m in zip(w.sessions, maps):
        gc.fold_memory_gpu(ctx, s)
        reqs.append(gc.request(ikv, s, m))
    ctx.session_open(999)
    empty = ikv.make_request(999, maps[0], 0, 0, 0, 0, 1, 0)
    reqs.insert(3, empty)
    tot = sum(s.N for s in w.sessions)
    mode = ikv.MODE_MEMORY if mode_name == "memory" else ikv.MODE_LEARNABLE
    stream = torch.cuda.Stream()
    busy = torch.empty(64 << 20, device="cuda")
    outs = []
    for lanes in (1, 3, 8):
        ctx.tune(ikv.TUNE_BATCH_LANES, lanes)
        sc = torch.full((tot,), float("nan"), device="cuda")
        torch.cuda.synchronize()
        for _ in range(4):
            busy.add_(1.0)
        ctx.score(reqs, mode, sc, None, stream)
        stream.synchronize()
        outs.append(sc.cpu().numpy())
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    off = 0
    for i, s in enumerate(w.sessions):
        M = gc.fold_memory_oracle(oracle, s)
        S = s.slot_map[:s.N].numpy()
        if mode_name == "memory":
            want = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe)
        else:
            want = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, 0, w=oracle.ResidualWeights(**rw))
        gc.assert_scores_close(outs[0][off:off + s.N], want, f"lanes request {i}")
        off += s.N


def test_batched_select_many_requests(ikv, oracle):
    """20 requests in one ikv_select_evict call (two launches of one cluster per request) on pages interleaved in one
    pool: mixed lengths (one beyond 32,768 positions), heavy ties, dead positions; every request bit-exact."""
    shape = wl.ModelShape(1, 2, 1, 64, "bf16")
    lens = [300 + (i * 1237) % 5000 for i in range(19)] + [40000]
    specs = [wl.SessionSpec(300 + i, n, 4, 128 + 64 * (i % 5), prefix_len=8, span_len=8) for i, n in enumerate(lens)]
    w = wl.make_workload(shape, specs, 41)
    gc.to_cuda(w)
    ctx = gc.make_ctx(w, max_sessions=64)
    rng = np.random.default_rng(12)
    tot = sum(lens)
    maps_h, maps, reqs, sc_parts = [], [], [], []
    for s in w.sessions:
        ctx.session_open(s.spec.session_id)
        S = s.slot_map[:s.N].numpy().copy()
        S[rng.choice(s.N, s.N // 6, replace=False)] = w.dead_slot
        maps_h.append(S)
        maps.append(torch.from_numpy(S.copy()).cuda())
        reqs.append(gc.request(ikv, s, maps[-1], radix=s.pi + 50))
        sc_parts.append((np.round(rng.standard_normal(s.N) * 4) / 4).astype(np.float32))
    scores = torch.from_numpy(np.concatenate(sc_parts)).cuda()
    freed = torch.empty(tot, dtype=torch.int32, device="cuda")
    nf = torch.zeros(20, dtype=torch.int32, device="cuda")
    nk = torch.zeros(20, dtype=torch.int32, device="cuda")
    ctx.select_evict(reqs, scores, freed, nf, nk)
    torch.cuda.synchronize()
    off = 0
    for i, s in enumerate(w.sessions):
        cls, _ = oracle.partition(maps_h[i], 0, s.pi, s.qs, s.qe)
        keep, n_kept = oracle.select(sc_parts[i], cls, s.spec.budget)
        S2, _, freed_o = oracle.rewrite(maps_h[i], 0, keep, s.pi + 50, w.n_slots)
        assert nk[i].item() == n_kept and nf[i].item() == len(freed_o), f"request {i}"
        assert np.array_equal(maps[i].cpu().numpy(), S2), f"request {i}"
        assert np.array_equal(freed.cpu().numpy()[off:off + len(freed_o)], freed_o), f"request {i}"
        off += s.N
    # the shared scratch is back to its invariant: a second call on the pruned maps changes nothing
    before = [m.clone() for m in maps]
    ctx.select_evict(reqs, scores, freed, nf, nk)
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(before, maps)) and int(nf.sum().item()) == 0


@pytest.mark.parametrize("row_dtype", ["f32", "bf16"])
def test_prune_host_path(ikv, oracle, row_dtype):
    w = build("bf16_d128_g4", SHAPES[1][1], n_tokens=2500, budget=700)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    ctx.session_open(s.spec.session_id)
    ups = s.updates()
    for rows in ups[:-1]:
        ctx.memory_update(s.spec.session_id, rows.cuda().contiguous())
    S = s.slot_map[:s.N].clone()
    S_host = S.clone().pin_memory()
    valid = torch.empty(s.N, dtype=torch.uint8).pin_memory()
    sc = torch.empty(s.N, dtype=torch.float32).pin_memory()
    freed = torch.empty(s.N, dtype=torch.int32).pin_memory()
    req = ikv.make_request(s.spec.session_id, None, s.N, s.pi, s.qs, s.qe, 700, s.pi)
    last = ups[-1].contiguous()
    if row_dtype == "bf16":                                  # query rows in the model's dtype: half the H2D bytes
        last = last.to(torch.bfloat16)
    n_freed, n_kept = ctx.prune_host(req, last, ikv.MODE_MEMORY, S_host, valid, sc, freed)
    M = np.zeros((w.shape.L, w.shape.Hq, w.shape.D))
    for rows in ups[:-1]:
        oracle.memory_update(M, rows.numpy(), 0.5)
    oracle.memory_update(M, last.float().numpy(), 0.5)
    g = gc.oracle_geom(oracle, w)
    want = oracle.score(g, kp, M, S.numpy(), s.pi, s.qs, s.qe)
    gc.assert_scores_close(sc.numpy(), want, "prune_host scores")
    cls, _ = oracle.partition(S.numpy(), 0, s.pi, s.qs, s.qe)
    keep, nk = oracle.select(sc.numpy(), cls, 700)
    S2, valid_o, freed_o = oracle.rewrite(S.numpy(), 0, keep, s.pi, w.n_slots)
    assert n_kept == nk == 700 and n_freed == len(freed_o)
    assert np.array_equal(S_host.numpy(), S2) and np.array_equal(valid.numpy(), valid_o)
    assert np.array_equal(freed.numpy()[:n_freed], freed_o)


def test_errors_are_reported_not_thrown(ikv):
    w = build("bf16_d64_g2", SHAPES[2][1], n_tokens=300, budget=100)
    gc.to_cuda(w)
    ctx = gc.make_ctx(w, max_sessions=2)
    s = w.sessions[0]
    S_dev = s.slot_map[:s.N].cuda()
    scores = torch.empty(s.N, device="cuda")
    req = gc.request(ikv, s, S_dev)
    with pytest.raises(ikv.IkvError) as e:
        ctx.score([req], ikv.MODE_MEMORY, scores)          # session never opened
    assert e.value.status == ikv.ERR_NO_SESSION
    ctx.session_open(s.spec.session_id)
    with pytest.raises(ikv.IkvError) as e:
        ctx.score([req], ikv.MODE_LEARNABLE, scores)       # no residual weights loaded
    assert e.value.status == ikv.ERR_INVALID_ARG
    bad = ikv.make_request(s.spec.session_id, S_dev, s.N, 50, 40, 60, 10)   # pi > q_s
    with pytest.raises(ikv.IkvError) as e:
        ctx.score([bad], ikv.MODE_MEMORY, scores)
    assert e.value.status == ikv.ERR_INVALID_ARG
    # LRU: a third session evicts the least recently used one
    ctx.session_open(1001)
    ctx.session_open(1002)
    with pytest.raises(ikv.IkvError) as e:
        ctx.score([req], ikv.MODE_MEMORY, scores)
    assert e.value.status == ikv.ERR_NO_SESSION
    # unsupported geometry is refused at create
    with pytest.raises(ikv.IkvError):
        ikv.Context(1, 3, 2, 64, w.k_pool[:1].contiguous(), w.v_pool[:1].contiguous())


# ------------------------------------------------------------------------------------------- stream ordering
def test_decode_after_a_producer_that_triggers_early(ikv, oracle):
    """ikv_decode_attn is launched with programmatic stream serialization.  With default request flags it must read q
    (and the slot-map tail) only after the preceding kernel of the stream has completed -- even when that kernel signals
    its dependents BEFORE it writes q (R27; ikv.h).  The producer here triggers first, idles 200 us, then
    writes the real q over a buffer of zeros."""
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    w = wl.small(seed=41, shape=shape, n_tokens=3000, budget=700, kv_dtype="bf16")
    ctx, s, M, kp, vp = run_memory(ikv, oracle, w)
    g = gc.oracle_geom(oracle, w)
    S_dev = s.slot_map.clone().cuda()
    scores = torch.empty(s.N, device="cuda")
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    req = gc.request(ikv, s, S_dev)
    ctx.score([req], ikv.MODE_MEMORY, scores)
    ctx.select_evict([req], scores, freed, nf, nk)
    scale = 1.0 / math.sqrt(shape.D)
    q_true = torch.randn((shape.L, 1, shape.Hq, shape.D), generator=torch.Generator().manual_seed(9)).to(torch.bfloat16).cuda()
    out = torch.zeros_like(q_true)
    seq = s.N + 2                                           # two appended positions: the slot-map tail is read as well
    r = gc.request(ikv, s, S_dev, seq_len=seq)
    ctx.decode_attn(0, [r], q_true[0], out[0], scale)       # first call after the select (not programmatic)
    torch.cuda.synchronize()
    for rep in range(3):
        q_buf = torch.zeros_like(q_true[1])
        out[1].zero_()
        torch.cuda.synchronize()
        ikv.Context.test_late_writer(q_buf, q_true[1], 200)
        ctx.decode_attn(1, [r], q_buf, out[1], scale)       # programmatic launch right behind the late writer
        torch.cuda.synchronize()
        want = oracle.decode(g, kp, vp, 1, S_dev.cpu().numpy()[:seq], q_true[1, 0].float().cpu().numpy(), scale)
        err = gc.assert_decode_close(out[1, 0].float().cpu().numpy(), want, True, f"late writer rep {rep}")
    print(f"decode behind an early-triggering producer: max abs err {err:.3e}")


def test_sessions_on_a_non_blocking_stream(ikv, oracle):
    """Session creation (auto-create in ikv_memory_update, ikv_session_fork) zero-fills the memory on the CALLER's stream:
    on a non-blocking stream, with the legacy default stream busy, the fill must not land after the first update."""
    shape = wl.ModelShape(2, 8, 2, 128, "bf16")
    w = wl.small(seed=43, shape=shape, n_tokens=600, budget=200, kv_dtype="bf16")
    gc.to_cuda(w)
    ctx = gc.make_ctx(w)
    s = w.sessions[0]
    side = torch.cuda.Stream()                               # torch side streams are cudaStreamNonBlocking
    busy = torch.empty(1 << 28, device="cuda")
    rows = s.mem_rows[:4].cuda().contiguous()
    torch.cuda.synchronize()
    for sid in range(300, 306):
        for _ in range(8):
            busy.add_(1.0)                                   # keeps the default stream busy
        with torch.cuda.stream(side):
            ctx.memory_update(sid, rows, side)               # auto-create + first update, both on `side`
            ctx.session_fork(sid, sid + 100, side)
    torch.cuda.synchronize()
    M = np.zeros((shape.L, shape.Hq, shape.D))
    oracle.memory_update(M, s.mem_rows[:4].numpy(), 0.5)
    for sid in range(300, 306):
        assert np.abs(ctx.session_get_memory(sid).numpy() - M).max() < 2e-6
        assert np.abs(ctx.session_get_memory(sid + 100).numpy() - M).max() < 2e-6


def test_scores_are_bit_identical_from_run_to_run(ikv, oracle):
    """Every sum of the scorer is taken in a fixed order (per-layer statistics in CTA order, deferred rule sums per
    thread, KV heads in order): repeated calls give the same bits, in both scorer modes."""
    w = wl.small(seed=47, shape=wl.ModelShape(4, 8, 2, 128, "bf16"), n_tokens=6000, budget=1500, kv_dtype="bf16")
    ctx, s, M, kp, _ = run_memory(ikv, oracle, w)
    ctx.residual_load(wl.residual_weights(w.shape.D, 31))
    S_dev = s.slot_map[:s.N].cuda()
    req = gc.request(ikv, s, S_dev)
    for mode in (ikv.MODE_MEMORY, ikv.MODE_LEARNABLE):
        ref = torch.empty(s.N, device="cuda")
        ctx.score([req], mode, ref)
        for _ in range(5):
            again = torch.empty(s.N, device="cuda")
            ctx.score([req], mode, again)
            assert torch.equal(ref.view(torch.int32), again.view(torch.int32))


@pytest.mark.parametrize("lm", [0, 1], ids=["logits_scratch", "auto"])
@pytest.mark.parametrize("name,shape", [SHAPES[1], SHAPES[2], SHAPES[5]], ids=["d128g4", "d64g2", "d128g8"])
def test_key_pass_variants_match_oracle(ikv, oracle, name, shape, lm):
    """The parity tests above run the layer-major key pass wherever it fits (gpu_common.LAYER_MAJOR = 2).  Here the same
    scores come from the logits-scratch key pass (0) and from the library's default choice (1), in both scorer modes."""
    w = build(name, shape)
    kp, vp = gc.to_cuda(w)
    ctx = gc.make_ctx(w, layer_major=lm)
    s = w.sessions[0]
    gc.fold_memory_gpu(ctx, s)
    M = gc.fold_memory_oracle(oracle, s)
    wts = wl.residual_weights(w.shape.D, 31)
    ctx.residual_load(wts)
    S = s.slot_map[:s.N].clone()
    S[s.pi + 3: s.pi + 90: 4] = w.dead_slot
    S_dev = S.cuda()
    req = gc.request(ikv, s, S_dev)
    g = gc.oracle_geom(oracle, w)
    for mode, omode in ((ikv.MODE_MEMORY, oracle.MODE_MEMORY), (ikv.MODE_LEARNABLE, oracle.MODE_LEARNABLE)):
        scores = torch.empty(s.N, device="cuda")
        ctx.score([req], mode, scores)
        want = oracle.score(g, kp, M, S.numpy(), s.pi, s.qs, s.qe, omode, 0, w=oracle.ResidualWeights(**wts))
        mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, f"{name} lm={lm} mode={mode}")
        print(f"[{name} lm={lm} mode={mode}] max abs err {mabs:.3e} rel {mrel:.3e}")
