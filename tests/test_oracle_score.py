"""Pins for the oracle's scoring steps O1-O6 (memory update, rule score, residual head).

Every check compares the C oracle with something other than itself: a value the paper prints,
a closed form, an invariant of the formula, or an independent implementation built from torch
CPU library routines (softmax, scaled_dot_product_attention, linear, gelu) in float64.
"""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

from paper_2606_09916_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def golden():
    out = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


def geom(o, w):
    return o.Geometry(w.shape.L, w.shape.Hq, w.shape.Hkv, w.shape.D, w.n_slots,
                      o.BF16 if w.shape.kv_dtype == "bf16" else o.F32, w.dead_slot)


def fold_memory(o, sess, lam=0.5):
    L, Hq, D = sess.mem_rows.shape[1:]
    M = np.zeros((L, Hq, D), np.float64)
    for rows in sess.updates():
        o.memory_update(M, rows.numpy(), lam)
    return M


def torch_rule(w, sess, M, cand):
    """Independent rule score: HF-style repeat_kv + torch.softmax over the candidate set."""
    K = w.k_pool.to(torch.float64)[:, sess.slot_map[:sess.N].long()]       # [L, N, Hkv, D]
    K = K[:, cand]                                                        # [L, nc, Hkv, D]
    Kx = K.repeat_interleave(w.shape.G, dim=2)                            # GQA expansion -> [L, nc, Hq, D]
    x = torch.einsum("lhd,ljhd->lhj", torch.from_numpy(M), Kx) / math.sqrt(w.shape.D)
    a = torch.softmax(x, dim=-1)
    return a.sum(dim=(0, 1)).numpy(), x.numpy()


# ------------------------------------------------------------------ bf16 up-conversion
def test_bf16_upconversion_exact(oracle):
    """pool_elem's bf16 -> double is exact: mean_key of one token with L=Hq=Hkv=1 returns the key itself."""
    shape = wl.ModelShape(1, 1, 1, 64, "bf16")
    t = torch.randn((1, 32, 1, 64), generator=torch.Generator().manual_seed(5)).to(torch.bfloat16)
    t[0, 3, 0, :4] = torch.tensor([1.0, -0.0, 3.3895e38, -1.0e-38]).to(torch.bfloat16)
    g = oracle.Geometry(1, 1, 1, 64, 32, oracle.BF16, 0)
    S = np.arange(32, dtype=np.int32)
    kb = oracle.mean_key(g, wl.to_numpy_bits(t), S, np.arange(32, dtype=np.int32))
    assert np.array_equal(kb, t[0, :, 0, :].to(torch.float64).numpy())


# ------------------------------------------------------------------ O1 memory update
def test_memory_unit_norm_and_closed_form(oracle):
    """P4: rows are unit norm after every update; M_1 = normalize(mean rows);
    M_2 = normalize(e^-lambda M_1 + mean rows_2) (Eq. 2)."""
    g = torch.Generator().manual_seed(3)
    r1 = torch.randn((4, 2, 3, 16), generator=g, dtype=torch.float64).float()
    r2 = torch.randn((3, 2, 3, 16), generator=g, dtype=torch.float64).float()
    M = np.zeros((2, 3, 16))
    oracle.memory_update(M, r1.numpy(), 0.5)
    assert np.allclose(np.linalg.norm(M, axis=-1), 1.0, atol=1e-14)
    m1 = F.normalize(r1.double().mean(0), dim=-1)
    assert np.allclose(M, m1.numpy(), atol=1e-14)
    oracle.memory_update(M, r2.numpy(), 0.5)
    m2 = F.normalize(math.exp(-0.5) * m1 + r2.double().mean(0), dim=-1)
    assert np.allclose(M, m2.numpy(), atol=1e-14)
    assert np.allclose(np.linalg.norm(M, axis=-1), 1.0, atol=1e-14)
    assert golden()["lambda"] == 0.5


def test_memory_zero_rows_stay_zero(oracle):
    """R3: a zero row divided by max(norm, 1e-12) stays zero (no NaN)."""
    M = np.zeros((1, 2, 8))
    oracle.memory_update(M, np.zeros((2, 1, 2, 8), np.float32), 0.5)
    assert np.array_equal(M, np.zeros((1, 2, 8)))


def test_query_mode_is_one_update_from_zero(oracle):
    r = torch.randn((5, 2, 4, 8), generator=torch.Generator().manual_seed(1))
    Mq = oracle.query_encoding(r.numpy())
    assert np.allclose(Mq, F.normalize(r.double().mean(0), dim=-1).numpy(), atol=1e-14)


def test_uncollapsed_bank_identity(oracle):
    """P5 (reading R1): Eq. 2 is linear up to a positive per-row renormalisation, so the collapsed M_t
    equals the un-collapsed bank sum_tau w_tau Enc_tau with w_tau = e^{-lambda (t-tau)} / prod_{s=tau..t} n_s
    (n_s = the row norm divided out at step s).  Scoring against the bank would be an M x T x D
    contraction; the method avoids it."""
    g = torch.Generator().manual_seed(11)
    ups = [torch.randn((4, 2, 2, 8), generator=g) for _ in range(5)]
    M = np.zeros((2, 2, 8))
    for u in ups:
        oracle.memory_update(M, u.numpy(), 0.5)
    encs = [u.double().mean(0) for u in ups]
    norms, m = [], torch.zeros(2, 2, 8, dtype=torch.float64)
    for e in encs:                                   # row norms n_s of the recurrence
        raw = math.exp(-0.5) * m + e
        norms.append(raw.norm(dim=-1, keepdim=True))
        m = raw / norms[-1]
    t_last = len(ups) - 1
    bank = torch.zeros_like(m)
    for tau, e in enumerate(encs):
        wt = math.exp(-0.5 * (t_last - tau)) / torch.stack(norms[tau:]).prod(dim=0)
        bank = bank + wt * e
    assert np.allclose(M, bank.numpy(), atol=1e-13)
    assert torch.all(torch.stack(norms) > 0)


# ------------------------------------------------------------------ O3-O5 rule score
@pytest.mark.parametrize("kv_dtype", ["f32", "bf16"])
def test_rule_single_head_is_softmax(oracle, kv_dtype):
    """P2: L=1, Hq=Hkv=1 => rule = softmax(K m / sqrt(D)) (Eq. 3 reduces to one attention row)."""
    shape = wl.ModelShape(1, 1, 1, 32, kv_dtype)
    spec = wl.SessionSpec(1, 200, 4, 50, prefix_len=0, span_len=0)
    w = wl.make_workload(shape, [spec], 21, outliers=False)
    s = w.sessions[0]
    M = fold_memory(oracle, s)
    cls, counts = oracle.partition(s.slot_map[:s.N].numpy(), 0, 0, 200, 200)
    assert counts.tolist() == [0, 0, 200]
    rule = oracle.rule_score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), M, s.slot_map[:s.N].numpy(), cls)
    K = w.k_pool.double()[0, s.slot_map[:s.N].long(), 0]
    ref = torch.softmax(K @ torch.from_numpy(M[0, 0]) / math.sqrt(32), dim=0).numpy()
    assert np.allclose(rule, ref, rtol=1e-12, atol=1e-15)


def test_rule_matches_torch_gqa_and_sums_to_LHq(oracle):
    """P1 + R4/R5: sum_j rule_j = L*Hq; candidates only; query head h reads KV head h // G
    (HF repeat_kv convention) -- checked against an independent torch implementation."""
    w = wl.small(seed=5, shape=wl.ModelShape(3, 8, 2, 64, "bf16"), n_tokens=700, budget=100)
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy().copy()
    S[[50, 51, 300, 699]] = w.dead_slot      # some dead positions, one inside the span
    M = fold_memory(oracle, s)
    cls, counts = oracle.partition(S, w.dead_slot, s.pi, s.qs, s.qe)
    cand = np.nonzero(cls == oracle.CAND)[0]
    assert counts[0] == 4 and counts[1] == s.pi + (s.qe - s.qs) - 1
    rule, logits = oracle.rule_score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), M, S, cls, want_logits=True)
    assert abs(rule.sum() - w.shape.L * w.shape.Hq) < 1e-9
    assert np.all(rule[cls != oracle.CAND] == 0)
    assert np.all(rule[cand] > 0) and np.all(rule[cand] <= w.shape.L * w.shape.Hq)
    sess = s
    ref, xref = torch_rule(w, sess, M, torch.from_numpy(cand))
    assert np.allclose(rule[cand], ref, rtol=1e-11)
    assert np.allclose(logits[:, :, cand], xref, rtol=1e-11, atol=1e-13)


def test_rule_zero_memory_is_uniform(oracle):
    """P3: fresh session (M = 0) => rule_j = L*Hq/|A| for every candidate."""
    w = wl.small(seed=6, shape=wl.ModelShape(2, 4, 2, 64, "bf16"), n_tokens=300, budget=100)
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy()
    cls, counts = oracle.partition(S, 0, s.pi, s.qs, s.qe)
    rule = oracle.rule_score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), np.zeros((2, 4, 64)), S, cls)
    assert np.allclose(rule[cls == oracle.CAND], 2 * 4 / counts[2], rtol=1e-13)


def test_rule_is_invariant_to_slot_placement(oracle):
    """The score depends on K only through the slot map: permuting physical slots (and the map with
    them) leaves rule unchanged -- catches a wrong pool index / stride."""
    w = wl.small(seed=8, shape=wl.ModelShape(2, 4, 2, 64, "f32"), n_tokens=200, budget=50, kv_dtype="f32")
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy()
    M = fold_memory(oracle, s)
    cls, _ = oracle.partition(S, 0, s.pi, s.qs, s.qe)
    g = geom(oracle, w)
    r1 = oracle.rule_score(g, wl.to_numpy_bits(w.k_pool), M, S, cls)
    perm = torch.randperm(w.n_slots - 1, generator=torch.Generator().manual_seed(2)) + 1
    perm = torch.cat([torch.zeros(1, dtype=torch.long), perm])
    k2 = torch.empty_like(w.k_pool)
    k2[:, perm] = w.k_pool
    S2 = perm[torch.from_numpy(S).long()].to(torch.int32).numpy()
    r2 = oracle.rule_score(g, wl.to_numpy_bits(k2), M, S2, cls)
    assert np.array_equal(r1, r2)


# ------------------------------------------------------------------ O6 residual head
def test_param_count_matches_paper(oracle):
    """P6: the topology (R9) reproduces the paper's printed 214,274 parameters at D=128."""
    assert oracle.residual_param_count(128) == int(golden()["residual_params_D128"])
    for D in (64, 128):
        wts = wl.residual_weights(D, 1)
        n = sum(v.size for k, v in wts.items() if k != "alpha") + 1
        assert n == oracle.residual_param_count(D)
    assert golden()["xattn_heads"] == 4 and golden()["xattn_width"] == 128 and golden()["mlp_hidden"] == 256


def torch_residual(rule_c, kbar, mbar, Kq, wts, alpha, no_xattn=False):
    """Independent residual head from torch library routines in float64 (P8)."""
    t = lambda a: torch.from_numpy(np.asarray(a, dtype=np.float64))
    rule_c, kbar, mbar, Kq = t(rule_c), t(kbar), t(mbar), t(Kq)
    nc, D = kbar.shape
    phi = torch.cat([kbar, mbar.expand(nc, D), kbar * mbar, rule_c[:, None]], dim=1)
    if no_xattn or Kq.shape[0] == 0:
        c = torch.zeros(nc, 128, dtype=torch.float64)
    else:
        Q = F.linear(phi, t(wts["wq"]), t(wts["bq"]))
        Kc = F.linear(Kq, t(wts["wk"]), t(wts["bk"]))
        Vc = F.linear(Kq, t(wts["wv"]), t(wts["bv"]))
        nq = Kq.shape[0]
        c = F.scaled_dot_product_attention(Q.view(nc, 4, 32).transpose(0, 1)[None],
                                           Kc.view(nq, 4, 32).transpose(0, 1)[None],
                                           Vc.view(nq, 4, 32).transpose(0, 1)[None])[0]
        c = c.transpose(0, 1).reshape(nc, 128)
    h = F.gelu(F.linear(torch.cat([phi, c], 1), t(wts["fc1_w"]), t(wts["fc1_b"])))
    z = F.linear(h, t(wts["fc2_w"])[None], t(wts["fc2_b"]))[:, 0]
    return (rule_c + max(-5.0, min(5.0, alpha)) * z).numpy(), z.numpy()


@pytest.mark.parametrize("D", [64, 128])
@pytest.mark.parametrize("nq", [0, 1, 7])
def test_residual_matches_torch_modules(oracle, D, nq):
    """P8: cross-attn == F.scaled_dot_product_attention with 4 heads of 32 on the projected inputs,
    MLP == Linear -> exact GELU -> Linear, phi order [kbar | mbar | kbar*mbar | rule | c] (Eq. 4-6)."""
    rng = np.random.default_rng(D + nq)
    nc = 23
    rule_c = rng.random(nc) * 0.1
    kbar = rng.standard_normal((nc, D)) * 0.3
    mbar = rng.standard_normal(D) * 0.1
    Kq = rng.standard_normal((nq, D)) * 0.3
    wts = wl.residual_weights(D, 9)
    w = oracle.ResidualWeights(**wts)
    s, z = oracle.residual(rule_c, kbar, mbar, Kq, w, want_z=True)
    ref_s, ref_z = torch_residual(rule_c, kbar, mbar, Kq, wts, wts["alpha"])
    assert np.abs(z).max() > 1e-3
    assert np.allclose(z, ref_z, rtol=1e-10, atol=1e-13)
    assert np.allclose(s, ref_s, rtol=1e-12, atol=1e-15)
    # ablation knob "- x-attn": c_j = 0
    s2 = oracle.residual(rule_c, kbar, mbar, Kq, w, flags=oracle.FLAG_NO_XATTN)
    assert np.allclose(s2, torch_residual(rule_c, kbar, mbar, Kq, wts, wts["alpha"], no_xattn=True)[0], rtol=1e-12)


def test_alpha_is_clipped(oracle):
    rng = np.random.default_rng(0)
    wts = wl.residual_weights(64, 2)
    args = (rng.random(5), rng.standard_normal((5, 64)), rng.standard_normal(64), rng.standard_normal((3, 64)))
    for a, clipped in ((9.0, 5.0), (-7.5, -5.0), (0.3, 0.3)):
        wts["alpha"] = a
        s, z = oracle.residual(*args, oracle.ResidualWeights(**wts), want_z=True)
        assert np.allclose(s, args[0] + clipped * z, rtol=1e-14)


def test_zero_init_recovers_rule_exactly(oracle):
    """P7: (alpha=1, fc2=0, b2=0) 'exactly recovers Equation (3)'; 'alpha = 0, exactly
    recovering the rule scorer' -- bit for bit, through the composite scoring call."""
    w = wl.small(seed=9, shape=wl.ModelShape(2, 4, 2, 64, "bf16"), n_tokens=400, budget=100)
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy()
    M = fold_memory(oracle, s)
    g = geom(oracle, w)
    kp = wl.to_numpy_bits(w.k_pool)
    base = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe, oracle.MODE_MEMORY)
    zi = oracle.ResidualWeights(**wl.residual_weights(64, 4, zero_init=True))
    got = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, w=zi)
    assert np.array_equal(base, got)
    rnd = oracle.ResidualWeights(**wl.residual_weights(64, 4))
    got = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, flags=oracle.FLAG_NO_RESIDUAL, w=rnd)
    assert np.array_equal(base, got)
    full = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, w=rnd)
    cand = np.isfinite(base)
    assert not np.array_equal(base[cand], full[cand])
    # fillers (R6): +inf at forced live positions, -inf at dead ones
    assert np.all(np.isposinf(base[:s.pi])) and np.all(np.isposinf(base[s.qs:s.qe]))


def test_composite_score_matches_stepwise_torch(oracle):
    """The composite call wires O2..O6 together as PAPER.md:489-491 orders them: k_bar over GQA-expanded
    heads and layers, Kq from the LIVE query positions only."""
    w = wl.small(seed=10, shape=wl.ModelShape(2, 4, 2, 64, "bf16"), n_tokens=300, budget=100)
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy().copy()
    S[s.qs + 2] = 0      # a dead query position: must be excluded from Kq
    S[100] = 0
    M = fold_memory(oracle, s)
    wts = wl.residual_weights(64, 12)
    sc, rule = oracle.score(geom(oracle, w), wl.to_numpy_bits(w.k_pool), M, S, s.pi, s.qs, s.qe,
                            oracle.MODE_LEARNABLE, w=oracle.ResidualWeights(**wts), want_rule=True)
    cls, _ = oracle.partition(S, 0, s.pi, s.qs, s.qe)
    cand = np.nonzero(cls == oracle.CAND)[0]
    Kall = w.k_pool.double()[:, torch.from_numpy(S).long()]                   # [L, N, Hkv, D]
    kbar_all = Kall.repeat_interleave(w.shape.G, dim=2).mean(dim=(0, 2))       # [N, D]
    qpos = [j for j in range(s.qs, s.qe) if S[j] != 0]
    ref, _ = torch_residual(rule[cand], kbar_all[cand].numpy(), M.mean(axis=(0, 1)), kbar_all[qpos].numpy(),
                            wts, wts["alpha"])
    assert np.allclose(sc[cand], ref.astype(np.float32), rtol=2e-7, atol=1e-9)
    assert np.all(np.isneginf(sc[cls == oracle.DEAD])) and np.all(np.isposinf(sc[cls == oracle.FORCED]))
