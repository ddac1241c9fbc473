"""-m gpu parity at the FULL sizes of BASELINE.json configs[2], configs[3] and configs[4] (configs[1] is in
test_gpu_multiturn.py), in the launch configuration bench.py uses.  The oracle runs whole passes, so every score is
compared; select / evict are checked bit-exact on the oracle's scores; decode on sampled layers."""
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


def _host_bits(t):
    return wl.to_numpy_bits(t)


def _layer_geom(oracle, w):
    """Geometry of ONE layer of the pool (decode checks copy a single layer of V to the host)."""
    return oracle.Geometry(1, w.shape.Hq, w.shape.Hkv, w.shape.D, w.n_slots, oracle.BF16, w.dead_slot)


def test_cfg2_full_size(ikv, oracle):
    """configs[2]: 48 layers, 40 Q / 8 KV heads (G = 5), D 128, 92,160 live tokens, M = 256, C = 8,192, learnable."""
    w = wl.cfg2(device="cuda", decode_tokens=4)
    s, shape = w.sessions[0], w.shape
    ctx = ikv.Context(shape.L, shape.Hq, shape.Hkv, shape.D, w.k_pool, w.v_pool, dead_slot=w.dead_slot)
    kp = _host_bits(w.k_pool)                              # after ikv_create initialised the dead slot
    ctx.reserve(s.N + 4, 1)
    wts = wl.residual_weights(shape.D, w.seed + 5)
    ctx.residual_load(wts)
    gc.fold_memory_gpu(ctx, s)
    M = gc.fold_memory_oracle(oracle, s)
    S = s.slot_map[:s.N].numpy().copy()
    S_dev = s.slot_map.clone().cuda()
    g = gc.oracle_geom(oracle, w)
    scores = torch.empty(s.N, device="cuda")
    req = ikv.make_request(s.spec.session_id, S_dev, s.N, s.pi, s.qs, s.qe, s.spec.budget, s.pi)
    ctx.score([req], ikv.MODE_LEARNABLE, scores)
    want = oracle.score(g, kp, M, S, s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, 0, w=oracle.ResidualWeights(**wts))
    mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, "cfg2 full size")
    print(f"cfg2 full: learnable score max abs err {mabs:.3e} rel {mrel:.3e}")
    # select / evict bit-exact on the oracle's scores
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    ctx.select_evict([req], torch.from_numpy(want).cuda(), freed, nf, nk)
    cls, _ = oracle.partition(S, w.dead_slot, s.pi, s.qs, s.qe)
    keep, n_kept = oracle.select(want, cls, s.spec.budget)
    S2, _, freed_o = oracle.rewrite(S, w.dead_slot, keep, s.pi, w.n_slots)
    assert nk.item() == n_kept == s.spec.budget
    assert np.array_equal(S_dev.cpu().numpy()[:s.N], S2)
    assert np.array_equal(freed.cpu().numpy()[:nf.item()], freed_o)
    # decode through the pruned map, two appended tokens, first and last layer
    S_full = S_dev.cpu().numpy()
    for layer in (0, shape.L - 1):
        q = torch.randn((1, shape.Hq, shape.D), generator=torch.Generator().manual_seed(layer)).to(torch.bfloat16)
        out = torch.empty((1, shape.Hq, shape.D), dtype=torch.bfloat16, device="cuda")
        r2 = ikv.make_request(s.spec.session_id, S_dev, s.N + 2, s.pi, s.qs, s.qe, s.spec.budget, s.pi)
        ctx.decode_attn(layer, [r2], q.cuda(), out, 1 / math.sqrt(shape.D))
        want_o = oracle.decode(_layer_geom(oracle, w), _host_bits(w.k_pool[layer:layer + 1]), _host_bits(w.v_pool[layer:layer + 1]),
                               0, S_full[:s.N + 2], q[0].float().numpy(), 1 / math.sqrt(shape.D))
        err = gc.assert_decode_close(out[0].float().cpu().numpy(), want_o, True, f"cfg2 decode layer {layer}")
        print(f"cfg2 full: decode layer {layer} max abs err {err:.3e}")


def test_cfg3_twenty_turns_with_fork(ikv, oracle):
    """configs[3] at scale: Qwen3-8B shape, 20 turns of a 64-token query + U(2k, 6k) tool tokens, 4 new memory rows per
    turn, prune to C = 8,192 after every turn, fork after turn 12 (the child shares the prefix and continues on different
    data for 8 turns).  Per turn: GPU scores vs oracle scores (all 36 layers), select / evict bit-exact on the oracle's
    scores (slot map, valid mask, freed list in order), then decode WITHOUT rescan -- cached survivor list plus two
    appended tokens -- on one layer.  Freed slots go back to the allocator.  Across the fork: positions kept by both
    branches hold the same slot, and no branch frees a slot of the shared prefix."""
    shape = wl.QWEN3_8B
    C, pi, span = 8192, 256, 64
    w = wl.make_workload(shape, [wl.SessionSpec(1, n_tokens=70000, n_mem_rows=4, budget=C, prefix_len=pi, span_len=span)],
                         seed=3000, device="cuda")
    ctx = ikv.Context(shape.L, shape.Hq, shape.Hkv, shape.D, w.k_pool, w.v_pool, dead_slot=w.dead_slot)
    kp = _host_bits(w.k_pool)
    g = gc.oracle_geom(oracle, w)
    ctx.reserve(20000, 1)
    wts = wl.residual_weights(shape.D, 77)
    ow = oracle.ResidualWeights(**wts)
    ctx.residual_load(wts)
    rng = np.random.default_rng(33)
    free = [int(x) for x in rng.permutation(np.arange(wl.PAGE, w.n_slots))]      # page 0 is reserved (dead slot)
    gen = torch.Generator().manual_seed(5)
    scale = 1 / math.sqrt(shape.D)
    dec_layer_k = {}

    class Sess:
        def __init__(self, sid, S, M, radix):
            self.sid, self.S, self.M, self.radix = sid, S, M, radix

    def alloc(n):
        return np.array([free.pop() for _ in range(n)], np.int32)

    def do_turn(s, turn, learnable):
        n_new = int(rng.integers(2048, 6145)) + span
        s.S = np.concatenate([s.S, alloc(n_new)])
        N = len(s.S)
        rows = torch.randn((4, shape.L, shape.Hq, shape.D), generator=gen)
        ctx.memory_update(s.sid, rows.cuda().contiguous())
        oracle.memory_update(s.M, rows.numpy(), 0.5)
        extra = alloc(2)                                                          # two decode appends after the prune
        S_dev = torch.from_numpy(np.concatenate([s.S, extra])).cuda()
        valid = torch.empty(N, dtype=torch.uint8, device="cuda")
        req = ikv.make_request(s.sid, S_dev, N, pi, N - span, N, C, s.radix, valid_mask=valid)
        scores = torch.empty(N, device="cuda")
        mode, omode = (ikv.MODE_LEARNABLE, oracle.MODE_LEARNABLE) if learnable else (ikv.MODE_MEMORY, oracle.MODE_MEMORY)
        ctx.score([req], mode, scores)
        want = oracle.score(g, kp, s.M, s.S, pi, N - span, N, omode, 0, w=ow)
        mabs, _ = gc.assert_scores_close(scores.cpu().numpy(), want, f"session {s.sid} turn {turn} N={N}")
        freed = torch.empty(N, dtype=torch.int32, device="cuda")
        nf = torch.zeros(1, dtype=torch.int32, device="cuda")
        nk = torch.zeros(1, dtype=torch.int32, device="cuda")
        ctx.select_evict([req], torch.from_numpy(want).cuda(), freed, nf, nk)
        cls, _ = oracle.partition(s.S, w.dead_slot, pi, N - span, N)
        keep, n_kept = oracle.select(want, cls, C)
        S2, valid_o, freed_o = oracle.rewrite(s.S, w.dead_slot, keep, s.radix, w.n_slots)
        assert nk.item() == n_kept == min(C, int((s.S != w.dead_slot).sum()))
        assert np.array_equal(S_dev.cpu().numpy()[:N], S2), f"turn {turn}: slot map"
        assert np.array_equal(valid.cpu().numpy(), valid_o)
        assert np.array_equal(freed.cpu().numpy()[:nf.item()], freed_o)
        # decode on the cached survivor list (no rescan) plus the two appended positions
        layer = turn % shape.L
        q = torch.randn((1, shape.Hq, shape.D), generator=gen).to(torch.bfloat16)
        out = torch.empty((1, shape.Hq, shape.D), dtype=torch.bfloat16, device="cuda")
        r2 = ikv.make_request(s.sid, S_dev, N + 2, pi, N - span, N, C, s.radix)
        ctx.decode_attn(layer, [r2], q.cuda(), out, scale)
        want_o = oracle.decode(_layer_geom(oracle, w), _host_bits(w.k_pool[layer:layer + 1]),
                               _host_bits(w.v_pool[layer:layer + 1]), 0, np.concatenate([S2, extra]), q[0].float().numpy(), scale)
        gc.assert_decode_close(out[0].float().cpu().numpy(), want_o, True, f"session {s.sid} turn {turn} decode")
        free.extend(int(x) for x in extra)
        s.S = S2
        return [int(x) for x in freed_o], mabs

    root = Sess(1, alloc(pi), np.zeros((shape.L, shape.Hq, shape.D)), pi)
    ctx.session_open(1)
    worst = 0.0
    for turn in range(12):
        fr, e = do_turn(root, turn, learnable=(turn == 5))
        free.extend(fr)
        worst = max(worst, e)
    shared = len(root.S)
    at_fork = root.S.copy()
    child = Sess(2, root.S.copy(), root.M.copy(), shared)                         # forks protect the shared prefix (R19)
    root.radix = shared
    ctx.session_fork(1, 2)
    shared_live = set(int(x) for x in at_fork[at_fork != w.dead_slot])
    for turn in range(12, 20):
        for s in (root, child):
            fr, e = do_turn(s, turn, learnable=(turn == 15))
            assert not (set(fr) & shared_live), "a branch freed a slot of the shared prefix"
            free.extend(fr)
            worst = max(worst, e)
    both = (root.S[:shared] != w.dead_slot) & (child.S[:shared] != w.dead_slot)
    assert np.array_equal(root.S[:shared][both], child.S[:shared][both])         # identity-stable across the fork
    assert np.array_equal(root.S[:shared][both], at_fork[both])
    print(f"cfg3 full: 20 turns + 8 forked turns, worst score abs err {worst:.3e}, final N root {len(root.S)} child {len(child.S)}")


def test_cfg4_sixty_four_sessions(ikv, oracle):
    """configs[4] on L_res = 4 resident layers: 64 sessions with lognormal live lengths (4k-64k) interleaved in one pool,
    budgets {4096, 8192, 16384}: ONE batched ikv_score (memory mode; every 16th session also through the learnable
    scorer), ONE batched ikv_select_evict on the oracle's scores (bit-exact per session), ONE batched decode call."""
    shape = wl.ModelShape(4, 32, 8, 128)
    w = wl.batched(device="cuda", shape=shape, decode_tokens=1)
    ctx = ikv.Context(shape.L, shape.Hq, shape.Hkv, shape.D, w.k_pool, w.v_pool, dead_slot=w.dead_slot, max_sessions=128)
    kp = _host_bits(w.k_pool)
    g = gc.oracle_geom(oracle, w)
    wts = wl.residual_weights(shape.D, w.seed + 5)
    ow = oracle.ResidualWeights(**wts)
    ctx.residual_load(wts)
    ctx.reserve(max(s.N for s in w.sessions) + 1, len(w.sessions))
    maps, reqs, Ms = [], [], []
    for s in w.sessions:
        gc.fold_memory_gpu(ctx, s)
        Ms.append(gc.fold_memory_oracle(oracle, s))
        maps.append(s.slot_map.clone().cuda())
        reqs.append(ikv.make_request(s.spec.session_id, maps[-1], s.N, s.pi, s.qs, s.qe, s.spec.budget, s.pi))
    tot = sum(s.N for s in w.sessions)
    scores = torch.empty(tot, device="cuda")
    ctx.score(reqs, ikv.MODE_MEMORY, scores)
    got = scores.cpu().numpy()
    wants, off, worst = [], 0, 0.0
    for s, M in zip(w.sessions, Ms):
        want = oracle.score(g, kp, M, s.slot_map[:s.N].numpy(), s.pi, s.qs, s.qe)
        mabs, _ = gc.assert_scores_close(got[off:off + s.N], want, f"cfg4 session {s.spec.session_id}")
        worst = max(worst, mabs)
        wants.append(want)
        off += s.N
    for i in range(0, len(reqs), 16):                          # the learnable scorer on every 16th session
        s = w.sessions[i]
        sc = torch.empty(s.N, device="cuda")
        ctx.score([reqs[i]], ikv.MODE_LEARNABLE, sc)
        want = oracle.score(g, kp, Ms[i], s.slot_map[:s.N].numpy(), s.pi, s.qs, s.qe, oracle.MODE_LEARNABLE, 0, w=ow)
        gc.assert_scores_close(sc.cpu().numpy(), want, f"cfg4 learnable session {s.spec.session_id}")
    freed = torch.empty(tot, dtype=torch.int32, device="cuda")
    nf = torch.zeros(len(reqs), dtype=torch.int32, device="cuda")
    nk = torch.zeros(len(reqs), dtype=torch.int32, device="cuda")
    ctx.select_evict(reqs, torch.from_numpy(np.concatenate(wants)).cuda(), freed, nf, nk)
    freed_h, nf_h, nk_h = freed.cpu().numpy(), nf.cpu().numpy(), nk.cpu().numpy()
    off = 0
    finals = []
    for i, s in enumerate(w.sessions):
        S = s.slot_map[:s.N].numpy()
        cls, _ = oracle.partition(S, w.dead_slot, s.pi, s.qs, s.qe)
        keep, n_kept = oracle.select(wants[i], cls, s.spec.budget)
        S2, _, freed_o = oracle.rewrite(S, w.dead_slot, keep, s.pi, w.n_slots)
        assert nk_h[i] == n_kept == min(s.spec.budget, s.N)
        assert np.array_equal(maps[i].cpu().numpy()[:s.N], S2), f"session {i}: slot map"
        assert nf_h[i] == len(freed_o) and np.array_equal(freed_h[off:off + nf_h[i]], freed_o)
        finals.append(np.concatenate([S2, s.slot_map[s.N:s.N + 1].numpy()]))
        off += s.N
    # one batched decode call over all 64 sessions (one appended token each), checked on a sample of sessions
    layer = 2
    q = torch.randn((len(reqs), shape.Hq, shape.D), generator=torch.Generator().manual_seed(4)).to(torch.bfloat16)
    out = torch.empty((len(reqs), shape.Hq, shape.D), dtype=torch.bfloat16, device="cuda")
    dreqs = [ikv.make_request(s.spec.session_id, m, s.N + 1, s.pi, s.qs, s.qe, s.spec.budget, s.pi)
             for s, m in zip(w.sessions, maps)]
    ctx.decode_attn(layer, dreqs, q.cuda(), out, 1 / math.sqrt(shape.D))
    k1, v1 = _host_bits(w.k_pool[layer:layer + 1]), _host_bits(w.v_pool[layer:layer + 1])
    for i in range(0, len(reqs), 7):
        want_o = oracle.decode(_layer_geom(oracle, w), k1, v1, 0, finals[i], q[i].float().numpy(), 1 / math.sqrt(shape.D))
        gc.assert_decode_close(out[i].float().cpu().numpy(), want_o, True, f"cfg4 decode session {i}")
    print(f"cfg4 full: 64 sessions, {tot} tokens, worst score abs err {worst:.3e}")


def test_next_rows_and_prefill_at_full_width(ikv, oracle):
    """The widened rows at the width and length of configs[1] (32 Q / 8 KV heads, D 128, 32,768 live tokens), on 4
    layers so that the oracle finishes in seconds: the 32-row window scorer on tcgen05 (one bank of 128 rows, every CTA
    on its full pair of tiles) against the oracle, then prune to C = 8,192 and a 256-row prefill chunk through the pruned
    map (tcgen05 kernel, 8 row blocks x 8 KV heads x 2 splits) against the oracle, counters exact."""
    shape = wl.ModelShape(4, 32, 8, 128, "bf16")
    w = wl.cfg1(device="cuda", shape=shape, n_tokens=32768, decode_tokens=256)
    s = w.sessions[0]
    ctx = ikv.Context(shape.L, shape.Hq, shape.Hkv, shape.D, w.k_pool, w.v_pool, dead_slot=w.dead_slot)
    kp = _host_bits(w.k_pool)
    ctx.reserve(s.N + 256, 1)
    gc.fold_memory_gpu(ctx, s)
    g = gc.oracle_geom(oracle, w)
    S = s.slot_map[:s.N].numpy().copy()
    S_dev = s.slot_map.clone().cuda()
    req = ikv.make_request(s.spec.session_id, S_dev, s.N, s.pi, s.qs, s.qe, 8192, s.pi)
    R = 32
    rows = torch.randn((R, shape.L, shape.Hq, shape.D), generator=torch.Generator().manual_seed(77))
    wt = [1.0 / R] * R
    scores = torch.empty(s.N, device="cuda")
    ctx.score_rows([req], rows.cuda().contiguous(), wt, scores)
    cls, _ = oracle.partition(S, w.dead_slot, s.pi, s.qs, s.qe)
    want = oracle.multirow_score(g, kp, rows.double().numpy(), wt, S, cls)
    want = np.where(cls == oracle.FORCED, np.inf, np.where(cls == oracle.DEAD, -np.inf, want))
    mabs, mrel = gc.assert_scores_close(scores.cpu().numpy(), want, "32-row scorer at full width")
    print(f"full width: 32-row scorer max abs err {mabs:.3e} rel {mrel:.3e}")
    # prune on these scores, then a prefill chunk through the pruned map
    freed = torch.empty(s.N, dtype=torch.int32, device="cuda")
    nf = torch.zeros(1, dtype=torch.int32, device="cuda")
    nk = torch.zeros(1, dtype=torch.int32, device="cuda")
    ctx.select_evict([req], scores, freed, nf, nk)
    torch.cuda.synchronize()
    assert nk.item() == 8192
    n_q, layer = 256, 2
    q = torch.randn((n_q, shape.Hq, shape.D), generator=torch.Generator().manual_seed(78)).to(torch.bfloat16)
    out = torch.empty((n_q, shape.Hq, shape.D), dtype=torch.bfloat16, device="cuda")
    reads = torch.zeros(2, dtype=torch.int64, device="cuda")
    r = ikv.make_request(s.spec.session_id, S_dev, s.N + n_q, s.pi, s.qs, s.qe, 8192, s.pi)
    ctx.prefill_attn(layer, r, s.N, q.cuda(), out, 1.0 / math.sqrt(shape.D), reads)
    torch.cuda.synchronize()
    vp = _host_bits(w.v_pool)
    want_o, raw, eff = oracle.prefill(g, kp, vp, layer, S_dev.cpu().numpy(), s.N, q.float().numpy(), 1.0 / math.sqrt(shape.D))
    err = gc.assert_decode_close(out.float().cpu().numpy(), want_o, True, "prefill chunk at full width")
    assert reads.cpu().tolist() == [raw, eff]
    print(f"full width: 256-row prefill chunk over {nk.item()} survivors max abs err {err:.3e}, reads {raw} / {eff}")
