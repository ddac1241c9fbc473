"""Pins for the oracle's select (O7), slot-map rewrite (O8) and decode (O9) steps."""
import math

import numpy as np
import pytest
import torch
import torch.nn.functional as F
from hypothesis import given, settings, strategies as st

from paper_2606_09916_b200 import workloads as wl
from tests.test_oracle_score import fold_memory, geom


def brute_select(scores, cls, C):
    """Full-sort brute force in pure Python: (score desc, position asc), NaN last, -0 == +0."""
    N = len(scores)
    forced = [j for j in range(N) if cls[j] == 1]
    cand = [j for j in range(N) if cls[j] == 2]
    if N <= C:
        return set(forced) | set(cand)
    cstar = max(0, C - len(forced))

    def key(j):
        s = float(scores[j])
        if math.isnan(s):
            return (1, 0.0, j)
        return (0, -(s + 0.0), j)
    return set(forced) | set(sorted(cand, key=key)[:cstar])


finite = st.floats(width=32, allow_nan=False, allow_infinity=False)
tiey = st.sampled_from([0.0, -0.0, 1.0, 1.0, 2.5, -3.0, float("nan"), 1e-38, -1e-38, 3.0e38])


@settings(max_examples=300, deadline=None)
@given(st.lists(st.tuples(st.one_of(finite, tiey), st.integers(0, 2)), min_size=0, max_size=60),
       st.integers(0, 70))
def test_select_matches_brute_force(scores_cls, C):
    """P10: brute force on tiny inputs, with hypothesis-generated ties, duplicates, NaN, +-0."""
    from oracle import ikv_oracle as o
    scores = np.array([s for s, _ in scores_cls], np.float32)
    cls = np.array([c for _, c in scores_cls], np.uint8)
    keep, nk = o.select(scores, cls, C)
    want = brute_select(scores, cls, C)
    assert set(np.nonzero(keep)[0].tolist()) == want
    assert nk == len(want)


def test_select_invariants(oracle):
    """P9: |K*| = min(C, live) when |F| <= C; F subset of K*; every kept candidate beats every dropped
    one under the total order (Eq. 1)."""
    rng = np.random.default_rng(1)
    N, C = 5000, 1200
    scores = rng.standard_normal(N).astype(np.float32)
    scores[rng.integers(0, N, 800)] = 0.25          # many exact ties
    S = np.arange(1, N + 1, dtype=np.int32)
    S[rng.integers(0, N, 300)] = 0
    cls, counts = oracle.partition(S, 0, 100, N - 50, N)
    keep, nk = oracle.select(scores, cls, C)
    live = counts[1] + counts[2]
    assert nk == min(C, live) == keep.sum()
    assert np.all(keep[cls == oracle.FORCED] == 1) and np.all(keep[cls == oracle.DEAD] == 0)
    kc = np.nonzero((cls == oracle.CAND) & (keep == 1))[0]
    dc = np.nonzero((cls == oracle.CAND) & (keep == 0))[0]
    worst_kept = min(kc, key=lambda j: (scores[j], -j))
    best_drop = max(dc, key=lambda j: (scores[j], -j))
    assert (scores[worst_kept], -worst_kept) > (scores[best_drop], -best_drop)
    # skip rule: N <= C keeps every live position
    keep2, nk2 = oracle.select(scores, cls, N)
    assert nk2 == live and np.array_equal(keep2, (cls != oracle.DEAD).astype(np.uint8))
    # R14: |F| > C keeps all of F and nothing else
    keep3, nk3 = oracle.select(scores, cls, 10)
    assert nk3 == counts[1] and np.array_equal(keep3, (cls == oracle.FORCED).astype(np.uint8))


def test_uniform_scores_keep_lowest_positions(oracle):
    """P3 / R13: equal scores => the C* lowest candidate positions survive."""
    N, C = 400, 100
    S = np.arange(1, N + 1, dtype=np.int32)
    cls, _ = oracle.partition(S, 0, 10, 380, 400)
    keep, nk = oracle.select(np.full(N, 0.5, np.float32), cls, C)
    assert nk == C
    assert np.nonzero(keep)[0].tolist() == list(range(0, 10 + 70)) + list(range(380, 400))


def test_rewrite_invariants(oracle):
    """P11 + P12 (Eq. 7)."""
    rng = np.random.default_rng(3)
    N, n_slots = 3000, 4096
    S = (1 + rng.permutation(n_slots - 1)[:N]).astype(np.int32)
    S[rng.integers(0, N, 200)] = 0                   # dead from an earlier round
    S[2000] = S[100]                                 # alias: dropped position shares a slot with a kept one
    S[2500] = S[2400]                                # alias between two dropped positions
    cls, _ = oracle.partition(S, 0, 64, N - 32, N)
    scores = rng.standard_normal(N).astype(np.float32)
    scores[100] = 100.0
    scores[[2000, 2400, 2500]] = -100.0
    keep, nk = oracle.select(scores, cls, 1000)
    radix = 500
    S2, valid, freed = oracle.rewrite(S, 0, keep, radix, n_slots)
    kept = keep.astype(bool)
    assert len(S2) == N                                              # N untouched
    assert np.array_equal(S2[kept], S[kept])                         # kept slots stay in place
    assert np.all(S2[~kept] == 0)                                    # everything else -> s+
    assert np.array_equal(valid, (S2 != 0).astype(np.uint8))
    kept_slots = set(S2[kept].tolist())
    assert not (set(freed.tolist()) & kept_slots)                    # (c)
    assert 0 not in freed.tolist()                                   # (b)
    assert len(set(freed.tolist())) == len(freed)                    # reported once
    assert S[100] not in freed.tolist() and S[2400] in freed.tolist()
    newly = [j for j in range(N) if not kept[j] and S[j] != 0]
    want = []
    for j in newly:                                                  # brute-force statement of (a)(b)(c)
        u = int(S[j])
        if j >= radix and u != 0 and u not in kept_slots and u not in want:
            want.append(u)
    assert freed.tolist() == want
    assert all(j >= radix for j in newly if S[j] in freed.tolist() and list(S).count(S[j]) == 1)
    # second call is a no-op
    keep_b, nk_b = oracle.select(scores, oracle.partition(S2, 0, 64, N - 32, N)[0], 1000)
    S3, valid3, freed3 = oracle.rewrite(S2, 0, keep_b, radix, n_slots)
    assert nk_b == nk and np.array_equal(S3, S2) and len(freed3) == 0 and np.array_equal(valid3, valid)


def torch_decode(w, layer, S, q, scale, dead=0):
    live = torch.from_numpy(np.nonzero(S != dead)[0])
    slots = torch.from_numpy(S).long()[live]
    K = w.k_pool.double()[layer, slots].repeat_interleave(w.shape.G, dim=1).transpose(0, 1)  # [Hq, n, D]
    V = w.v_pool.double()[layer, slots].repeat_interleave(w.shape.G, dim=1).transpose(0, 1)
    return F.scaled_dot_product_attention(q.double()[:, None, :], K, V, scale=scale)[:, 0].numpy()


@pytest.mark.parametrize("kv_dtype", ["f32", "bf16"])
def test_decode_is_sdpa_over_survivors(oracle, kv_dtype):
    """P13: decode through the slot map == dense attention over the gathered survivor rows."""
    w = wl.small(seed=31, shape=wl.ModelShape(2, 8, 2, 64, kv_dtype), n_tokens=500, budget=100)
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy().copy()
    S[np.random.default_rng(0).integers(0, s.N, 350)] = 0
    q = torch.randn((8, 64), generator=torch.Generator().manual_seed(4)).to(torch.bfloat16).float()
    g = geom(oracle, w)
    for layer in (0, 1):
        out = oracle.decode(g, wl.to_numpy_bits(w.k_pool), wl.to_numpy_bits(w.v_pool), layer, S, q.numpy(), 0.125)
        assert np.allclose(out, torch_decode(w, layer, S, q, 0.125), rtol=1e-11, atol=1e-13)
    # no live position => zeros
    out = oracle.decode(g, wl.to_numpy_bits(w.k_pool), wl.to_numpy_bits(w.v_pool), 0, np.zeros(9, np.int32), q.numpy(), 0.125)
    assert np.array_equal(out, np.zeros((8, 64)))


def test_sentinel_attend_equals_skip(oracle):
    """P14 / R16: with K[s+] = -1e4, V[s+] = 0 attending to dead entries equals skipping them
    whenever sum_d q_d > 0 (the sentinel logit is -1e4 * sum(q) * scale)."""
    w = wl.small(seed=32, shape=wl.ModelShape(1, 4, 2, 64, "f32"), n_tokens=300, budget=100, kv_dtype="f32")
    w.k_pool[:, 0] = -1.0e4
    w.v_pool[:, 0] = 0.0
    s = w.sessions[0]
    S = s.slot_map[:s.N].numpy().copy()
    S[::3] = 0
    q = torch.randn((4, 64), generator=torch.Generator().manual_seed(4)).abs()     # sum(q) > 0
    g = geom(oracle, w)
    kp, vp = wl.to_numpy_bits(w.k_pool), wl.to_numpy_bits(w.v_pool)
    skip = oracle.decode(g, kp, vp, 0, S, q.numpy(), 0.125)
    att = oracle.decode(g, kp, vp, 0, S, q.numpy(), 0.125, attend_all=True)
    assert np.allclose(skip, att, rtol=1e-12, atol=1e-300)


def test_tiny_config_end_to_end(oracle):
    """configs[0] through the whole event: exactly min(C, live) survive, kept bytes / positions unchanged,
    dropped -> dead slot, planted evidence is over-represented in K* (P15, sanity), decode == dense."""
    w = wl.tiny()
    s = w.sessions[0]
    g = geom(oracle, w)
    kp, vp = wl.to_numpy_bits(w.k_pool), wl.to_numpy_bits(w.v_pool)
    k_before = kp.copy()
    M = fold_memory(oracle, s)
    S = s.slot_map[:s.N].numpy()
    ev = oracle.prune_event(g, kp, M, S, s.pi, s.qs, s.qe, s.spec.budget, radix_len=s.pi)
    assert ev["n_kept"] == 128 == int((ev["slot_map"] != 0).sum())
    kept = ev["keep"].astype(bool)
    assert np.array_equal(ev["slot_map"][kept], S[kept]) and np.all(ev["slot_map"][~kept] == 0)
    assert np.array_equal(kp, k_before)
    assert len(ev["freed"]) == 512 - 128
    planted_kept = kept[s.planted_pos].mean()
    assert planted_kept >= 0.75 > 96 / 480          # base rate of a candidate being kept is 0.2
    q = torch.randn((4, 64), generator=torch.Generator().manual_seed(6)).to(torch.bfloat16).float()
    out = oracle.decode(g, kp, vp, 0, ev["slot_map"], q.numpy(), 1 / 8)
    assert np.allclose(out, torch_decode(w, 0, ev["slot_map"], q, 1 / 8), rtol=1e-11, atol=1e-13)


def test_fork_keeps_shared_slots_identity_stable(oracle):
    """P12 / R19: a forked session shares a prefix; with radix_protected_len = shared length neither side
    frees a shared slot, and positions both keep hold the same slot id."""
    w = wl.small(seed=41, shape=wl.ModelShape(1, 4, 2, 64, "f32"), n_tokens=600, budget=200, kv_dtype="f32",
                 decode_tokens=256)
    s = w.sessions[0]
    g = geom(oracle, w)
    kp = wl.to_numpy_bits(w.k_pool)
    shared = 400
    S_parent = s.slot_map[:600].numpy().copy()
    S_child = S_parent.copy()
    spare = np.setdiff1d(np.arange(16, w.n_slots), S_parent)[:200].astype(np.int32)
    S_child[shared:] = spare                           # child continues with its own slots
    Mp = fold_memory(oracle, s)
    Mc = Mp.copy()
    oracle.memory_update(Mc, torch.randn((4, 1, 4, 64), generator=torch.Generator().manual_seed(1)).numpy(), 0.5)
    a = oracle.prune_event(g, kp, Mp, S_parent, s.pi, s.qs, s.qe, 200, radix_len=shared)
    b = oracle.prune_event(g, kp, Mc, S_child, s.pi, s.qs, s.qe, 200, radix_len=shared)
    shared_slots = set(S_parent[:shared].tolist())
    assert not (set(a["freed"].tolist()) & shared_slots) and not (set(b["freed"].tolist()) & shared_slots)
    both = (a["keep"][:shared] == 1) & (b["keep"][:shared] == 1)
    assert both.sum() > 0
    assert np.array_equal(a["slot_map"][:shared][both], b["slot_map"][:shared][both])
