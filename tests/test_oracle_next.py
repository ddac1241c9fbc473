"""Pins for the oracle functions of the SURVEY 8(f) follow-ups (oracle/ikv_oracle_next.c): N1 multi-row scorer, N2 prefill
attention with KV-read counters, N3 baseline scorers.  Every check compares the C oracle with something other than
itself: the already-pinned Eq. 3 routine, torch library routines in float64, closed forms, or brute force."""
import math

import numpy as np
import torch
import torch.nn.functional as F

from paper_2606_09916_b200 import workloads as wl
from tests.test_oracle_score import geom, fold_memory


def _case(oracle, shape=None, n_tokens=300, seed=5, n_dead=40):
    shape = shape or wl.ModelShape(2, 4, 2, 64, "bf16")
    w = wl.small(seed=seed, shape=shape, n_tokens=n_tokens, budget=80, prefix_len=9, span_len=7, kv_dtype=shape.kv_dtype)
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy().copy()
    rng = np.random.default_rng(seed)
    S[rng.choice(s.N, n_dead, replace=False)] = w.dead_slot
    cls, _ = oracle.partition(S, w.dead_slot, s.pi, s.qs, s.qe)
    return w, s, S, cls


# ------------------------------------------------------------------------------------------- N1
def test_multirow_single_row_is_eq3(oracle):
    """R = 1, w = 1, rows[0] = M_t reproduces Eq. 3 (oracle.rule_score) bit for bit."""
    w, s, S, cls = _case(oracle)
    M = fold_memory(oracle, s)
    want = oracle.rule_score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), M, S, cls)
    got = oracle.multirow_score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), M[None], [1.0], S, cls)
    assert np.array_equal(got, want)


def test_multirow_matches_torch_per_row_softmax(oracle):
    """Independent implementation: per (row, layer, head) torch.softmax over the candidates, GQA by repeat_interleave,
    weighted sum over rows; and the closed form sum_j s_j = L * H_q * sum_r w_r."""
    w, s, S, cls = _case(oracle, wl.ModelShape(2, 6, 2, 64, "bf16"))
    R = 5
    rows = torch.randn((R, w.shape.L, w.shape.Hq, w.shape.D), generator=torch.Generator().manual_seed(2), dtype=torch.float64)
    wt = np.array([0.5, 1.0, 0.25, 2.0, 1.5])
    got = oracle.multirow_score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), rows.numpy(), wt, S, cls)
    cand = np.nonzero(cls == oracle.CAND)[0]
    K = w.k_pool.to(torch.float64)[:, torch.from_numpy(S[cand]).long()]            # [L, nc, Hkv, D]
    Kx = K.repeat_interleave(w.shape.G, dim=2)                                      # [L, nc, Hq, D]
    x = torch.einsum("rlhd,ljhd->rlhj", rows, Kx) / math.sqrt(w.shape.D)
    a = torch.softmax(x, dim=-1)
    want = torch.einsum("r,rlhj->j", torch.from_numpy(wt), a).numpy()
    assert np.allclose(got[cand], want, rtol=1e-12, atol=1e-15)
    assert np.all(got[cls != oracle.CAND] == 0.0)
    assert abs(got.sum() - w.shape.L * w.shape.Hq * wt.sum()) < 1e-9


def test_multirow_is_linear_in_the_weights(oracle):
    w, s, S, cls = _case(oracle)
    rows = np.random.default_rng(1).standard_normal((3, w.shape.L, w.shape.Hq, w.shape.D))
    g, kp = geom(oracle, w), wl.to_numpy_bits(w.k_pool)
    parts = [oracle.multirow_score(g, kp, rows[r:r + 1], [1.0], S, cls) for r in range(3)]
    both = oracle.multirow_score(g, kp, rows, [2.0, -1.0, 0.5], S, cls)
    assert np.allclose(both, 2.0 * parts[0] - parts[1] + 0.5 * parts[2], rtol=1e-12, atol=1e-15)


# ------------------------------------------------------------------------------------------- N3
def test_maxpool_dense_is_max_pool1d(oracle):
    """All positions candidates: the smoothing is torch's max_pool1d (kernel 7, stride 1, padding 3)."""
    rng = np.random.default_rng(3)
    s = rng.standard_normal(257)
    cls = np.full(257, oracle.CAND, np.uint8)
    got = oracle.maxpool_candidates(s, cls, 7)
    want = F.max_pool1d(torch.from_numpy(s)[None, None], 7, 1, 3)[0, 0].numpy()
    assert np.array_equal(got, want)


def test_maxpool_skips_non_candidates(oracle):
    rng = np.random.default_rng(4)
    n = 120
    s = rng.standard_normal(n)
    cls = rng.choice([oracle.DEAD, oracle.FORCED, oracle.CAND], size=n, p=[0.2, 0.1, 0.7]).astype(np.uint8)
    s[cls == oracle.FORCED] = np.inf
    s[cls == oracle.DEAD] = -np.inf
    got = oracle.maxpool_candidates(s, cls, 7)
    for j in range(n):                                   # brute force
        if cls[j] != oracle.CAND:
            assert got[j] == s[j]
            continue
        win = [s[i] for i in range(max(0, j - 3), min(n, j + 4)) if cls[i] == oracle.CAND]
        assert got[j] == max(win)


def test_streaming_keeps_sinks_and_the_most_recent(oracle):
    """Through the (already pinned) selection: sink candidates first, then the most recent candidates."""
    n, C = 200, 60
    cls = np.full(n, oracle.CAND, np.uint8)
    cls[10:20] = oracle.FORCED
    cls[[2, 50, 51, 199]] = oracle.DEAD
    sc = oracle.streaming_scores(cls, 4).astype(np.float32)
    scores = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, sc)).astype(np.float32)
    keep, n_kept = oracle.select(scores, cls, C)
    cand = [j for j in range(n) if cls[j] == oracle.CAND]
    cstar = C - 10
    sinks = [j for j in cand if j < 4]
    recent = [j for j in cand if j >= 4][-(cstar - len(sinks)):]
    want = np.zeros(n, bool)
    want[10:20] = True
    want[sinks + recent] = True
    assert n_kept == C and np.array_equal(keep.astype(bool), want)


def test_h2o_recent_floor_and_heavy_hitters(oracle):
    rng = np.random.default_rng(6)
    n, C = 300, 100
    cls = np.full(n, oracle.CAND, np.uint8)
    cls[:16] = oracle.FORCED
    cls[rng.choice(np.arange(16, n), 30, replace=False)] = oracle.DEAD
    hh = np.where(cls == oracle.CAND, rng.random(n), 0.0)
    for ratio, floor_ in ((0.5, 8), (0.0, 20), (1.0, 0), (0.1, 1000)):
        out = oracle.h2o_scores(hh, cls, C, ratio, floor_)
        cand = [j for j in range(n) if cls[j] == oracle.CAND]
        cstar = C - 16
        n_recent = min(cstar, max(floor_, int(math.floor(ratio * cstar + 0.5))))
        recent = cand[len(cand) - n_recent:] if n_recent else []
        for j in cand:
            assert out[j] == (1.0e30 + j if j in recent else hh[j])
        scores = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, out)).astype(np.float32)
        keep, n_kept = oracle.select(scores, cls, C)
        assert n_kept == C and all(keep[j] for j in recent)
        rest = [j for j in cand if j not in recent]
        top = sorted(rest, key=lambda j: (-np.float32(hh[j]), j))[:cstar - n_recent]
        assert all(keep[j] for j in top)


# ------------------------------------------------------------------------------------------- N2
def test_prefill_is_masked_sdpa_and_counts_reads(oracle):
    shape = wl.ModelShape(2, 4, 2, 64, "bf16")
    w, s, S, cls = _case(oracle, shape, n_tokens=150, n_dead=30)
    g = geom(oracle, w)
    kp, vp = wl.to_numpy_bits(w.k_pool), wl.to_numpy_bits(w.v_pool)
    q_pos0, n_q, layer = 110, 40, 1
    S[q_pos0 + 3] = w.dead_slot                                  # a dead position inside the chunk as well
    q = torch.randn((n_q, shape.Hq, shape.D), generator=torch.Generator().manual_seed(8)).to(torch.bfloat16).float()
    scale = 1.0 / math.sqrt(shape.D)
    out, raw, eff = oracle.prefill(g, kp, vp, layer, S, q_pos0, q.numpy(), scale)
    n = q_pos0 + n_q
    K = w.k_pool[layer].to(torch.float64)[torch.from_numpy(S[:n]).long()].repeat_interleave(shape.G, dim=1)   # [n, Hq, D]
    V = w.v_pool[layer].to(torch.float64)[torch.from_numpy(S[:n]).long()].repeat_interleave(shape.G, dim=1)
    live = torch.from_numpy(S[:n] != w.dead_slot)
    pos = torch.arange(n)
    mask = (pos[None, :] <= (q_pos0 + torch.arange(n_q))[:, None]) & live[None, :]              # [n_q, n]
    want = F.scaled_dot_product_attention(q.double().permute(1, 0, 2)[None], K.permute(1, 0, 2)[None],
                                          V.permute(1, 0, 2)[None], attn_mask=mask[None, None], scale=scale)
    assert np.allclose(out, want[0].permute(1, 0, 2).numpy(), rtol=1e-10, atol=1e-12)
    assert raw == sum(q_pos0 + i + 1 for i in range(n_q))
    assert eff == sum(int((S[:q_pos0 + i + 1] != w.dead_slot).sum()) for i in range(n_q))


def test_prefill_single_row_is_decode(oracle):
    shape = wl.ModelShape(2, 4, 2, 64, "bf16")
    w, s, S, cls = _case(oracle, shape, n_tokens=150, n_dead=30)
    g = geom(oracle, w)
    kp, vp = wl.to_numpy_bits(w.k_pool), wl.to_numpy_bits(w.v_pool)
    q = torch.randn((1, shape.Hq, shape.D), generator=torch.Generator().manual_seed(9)).to(torch.bfloat16).float()
    out, raw, eff = oracle.prefill(g, kp, vp, 0, S, 149, q.numpy(), 0.125)
    want = oracle.decode(g, kp, vp, 0, S[:150], q[0].numpy(), 0.125)
    assert np.array_equal(out[0], want) and raw == 150 and eff == int((S[:150] != w.dead_slot).sum())


# ------------------------------------------------------------------------------------------- N4: Eq. 8 and dL/ds
def _loss_case(seed, n=400, pos_rate=0.03, excl=0.1):
    rng = np.random.default_rng(seed)
    s = rng.standard_normal(n) * 2.0
    y = (rng.random(n) < pos_rate).astype(np.int32)
    y[rng.random(n) < excl] = -100
    return s, y


def test_train_loss_bce_term_is_torch_bce_with_logits(oracle):
    """L_BCE against the library routine (pos_weight = (1 - p~) / p~, mean over the valid entries), for a
    positive rate below, inside and above the clip [0.02, 0.5]."""
    import torch.nn.functional as F
    for seed, rate in ((1, 0.005), (2, 0.1), (3, 0.8)):
        s, y = _loss_case(seed, pos_rate=rate)
        terms, _ = oracle.train_loss(s, y)
        v = y >= 0
        p = y[v].mean()
        pt = min(max(p, 0.02), 0.5)
        want = F.binary_cross_entropy_with_logits(torch.from_numpy(s[v]), torch.from_numpy(y[v].astype(np.float64)),
                                                  pos_weight=torch.tensor((1 - pt) / pt, dtype=torch.float64))
        assert abs(terms[1] - want.item()) < 1e-12 * max(1.0, abs(want.item()))
        assert abs(terms[3] - torch.sigmoid(torch.from_numpy(s[v])).mean().item()) < 1e-14


def test_train_loss_rank_term_brute_force(oracle):
    """L_rank by brute force in Python: every positive against the 64 highest negatives (ties: lower position first),
    pairwise softplus, mean over the pairs; fewer than 64 negatives and heavy ties included."""
    import math
    for seed, n, q in ((4, 300, None), (5, 50, None), (6, 500, 0.5)):
        s, y = _loss_case(seed, n=n, pos_rate=0.1)
        if q:
            s = np.round(s / q) * q
        terms, _ = oracle.train_loss(s, y)
        neg = sorted([i for i in range(n) if y[i] == 0], key=lambda i: (-s[i], i))[:64]
        pos = [i for i in range(n) if y[i] == 1]
        tot = sum(math.log1p(math.exp(s[j] - s[i])) for i in pos for j in neg)
        want = tot / (len(pos) * len(neg)) if pos and neg else 0.0
        assert abs(terms[2] - want) < 1e-12 * max(1.0, want)


def test_train_loss_total_gradient_and_special_cases(oracle):
    """L = L_BCE + rho L_rank + gamma keep + eta norm; dL/ds against central differences of L itself (away from ties the
    hard-negative set is locally constant); excluded entries get no gradient; no positives: rank term 0 and p~ = 0.02;
    nothing valid: only the norm term; rows of norm 2 give norm term 1."""
    s, y = _loss_case(7, n=200, pos_rate=0.08)
    rows = np.random.default_rng(8).standard_normal((6, 16))
    rho, gamma, eta = 0.05, 0.01, 0.001
    terms, grad = oracle.train_loss(s, y, rows, rho, gamma, eta)
    assert abs(terms[0] - (terms[1] + rho * terms[2] + gamma * terms[3] + eta * terms[4])) < 1e-15
    want_norm = np.mean((np.linalg.norm(rows, axis=1) - 1.0) ** 2)
    assert abs(terms[4] - want_norm) < 1e-14
    eps = 1e-6
    for i in range(0, 200, 7):
        sp, sm = s.copy(), s.copy()
        sp[i] += eps
        sm[i] -= eps
        fd = (oracle.train_loss(sp, y, rows, rho, gamma, eta)[0][0] - oracle.train_loss(sm, y, rows, rho, gamma, eta)[0][0]) / (2 * eps)
        assert abs(grad[i] - fd) < 1e-8, (i, grad[i], fd)
    assert np.all(grad[y < 0] == 0.0)
    y0 = np.where(y == 1, 0, y)
    t0, _ = oracle.train_loss(s, y0)
    v = y0 >= 0
    assert t0[2] == 0.0
    assert abs(t0[1] - np.mean(np.logaddexp(0.0, s[v]))) < 1e-13          # only negatives: plain softplus, w+ unused
    tn, gn = oracle.train_loss(s, np.full_like(y, -100), 2.0 * np.eye(4), rho, gamma, eta)
    assert tn[1] == tn[2] == tn[3] == 0.0 and abs(tn[4] - 1.0) < 1e-15 and abs(tn[0] - eta) < 1e-18 and not gn.any()
