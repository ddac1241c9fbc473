"""ctypes/numpy front end of the CPU oracle (oracle/ikv_oracle.c).

TEST INFRASTRUCTURE ONLY: may be imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg, never by the product package.
It holds no arithmetic of its own: every function marshals numpy arrays into the C
oracle, which follows /root/reference/PAPER.md step by step in fp64 (see the header
of ikv_oracle.c for the citations, DESIGN.md section 3 for the readings R1..R22).

bf16 tensors are passed as numpy uint16 arrays holding the exact bf16 bits.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ikv_oracle.c")
_SRC_NEXT = os.path.join(_HERE, "ikv_oracle_next.c")      # SURVEY 8(f) follow-ups (N1-N3)
_LIB = os.path.join(_HERE, "libikv_oracle.so")

F32, BF16 = 0, 1
DEAD, FORCED, CAND = 0, 1, 2
FLAG_NO_XATTN, FLAG_NO_RESIDUAL = 1, 2
MODE_MEMORY, MODE_LEARNABLE = 0, 1


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (plain C11 + OpenMP). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC),
                                                                         os.path.getmtime(_SRC_NEXT)):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _LIB, _SRC, _SRC_NEXT, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_residual_param_count.restype = C.c_int64
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


@dataclass
class Geometry:
    """Model / pool geometry (K,V in R^{L x H_kv x N x D})."""
    L: int
    Hq: int
    Hkv: int
    D: int
    n_slots: int
    kv_dtype: int  # F32 or BF16
    dead_slot: int

    def pool_shape(self):
        return (self.L, self.n_slots, self.Hkv, self.D)


def _pool(g: Geometry, pool):
    want = np.uint16 if g.kv_dtype == BF16 else np.float32
    assert pool.dtype == want and pool.flags["C_CONTIGUOUS"], (pool.dtype, want)
    assert pool.shape == g.pool_shape(), (pool.shape, g.pool_shape())
    return pool


@dataclass
class ResidualWeights:
    """Residual-head parameters, row-major [out][in] fp32 (reading R9)."""
    wq: np.ndarray
    bq: np.ndarray
    wk: np.ndarray
    bk: np.ndarray
    wv: np.ndarray
    bv: np.ndarray
    fc1_w: np.ndarray
    fc1_b: np.ndarray
    fc2_w: np.ndarray
    fc2_b: np.ndarray
    alpha: float

    def arrays(self):
        return [_c(getattr(self, n), np.float32) for n in
                ("wq", "bq", "wk", "bk", "wv", "bv", "fc1_w", "fc1_b", "fc2_w", "fc2_b")]


def memory_update(M, q_rows, lam: float):
    """O1 (Eq. 2). M: [L,Hq,D] float64, updated in place. q_rows: [n,L,Hq,D] fp32."""
    assert M.dtype == np.float64 and M.flags["C_CONTIGUOUS"]
    q_rows = _c(q_rows, np.float32)
    n, L, Hq, D = q_rows.shape
    assert M.shape == (L, Hq, D)
    lib().oracle_memory_update(_p(M), _p(q_rows), n, L, Hq, D, C.c_double(lam))
    return M


def query_encoding(q_rows):
    q_rows = _c(q_rows, np.float32)
    n, L, Hq, D = q_rows.shape
    M = np.zeros((L, Hq, D), np.float64)
    lib().oracle_query_encoding(_p(M), _p(q_rows), n, L, Hq, D)
    return M


def partition(S, dead, pi, qs, qe):
    """O2. Returns (cls[N] uint8, counts[3] = dead, forced, cand)."""
    S = _c(S, np.int32)
    cls = np.empty(S.shape[0], np.uint8)
    counts = np.zeros(3, np.int32)
    lib().oracle_partition(_p(S), S.shape[0], int(dead), int(pi), int(qs), int(qe), _p(cls), _p(counts))
    return cls, counts


def rule_score(g: Geometry, k_pool, M, S, cls, want_logits=False):
    """O3-O5 (Eq. 3). Returns rule[N] float64 (and logits [L,Hq,N] if asked)."""
    S = _c(S, np.int32)
    N = S.shape[0]
    M = _c(M, np.float64)
    rule = np.zeros(N, np.float64)
    logits = np.zeros((g.L, g.Hq, N), np.float64) if want_logits else None
    lib().oracle_rule_score(_p(_pool(g, k_pool)), g.kv_dtype, C.c_int64(g.n_slots), g.L, g.Hq, g.Hkv,
                            g.D, _p(M), _p(S), _p(_c(cls, np.uint8)), N, _p(rule), _p(logits))
    return (rule, logits) if want_logits else rule


def mean_key(g: Geometry, k_pool, S, pos):
    """O6a: k_bar for the listed positions -> [len(pos), D] float64."""
    S = _c(S, np.int32)
    pos = _c(pos, np.int32)
    out = np.zeros((pos.shape[0], g.D), np.float64)
    lib().oracle_mean_key(_p(_pool(g, k_pool)), g.kv_dtype, C.c_int64(g.n_slots), g.L, g.Hq, g.Hkv, g.D,
                          _p(S), _p(pos), pos.shape[0], _p(out))
    return out


def mean_memory(M):
    M = _c(M, np.float64)
    L, Hq, D = M.shape
    out = np.zeros(D, np.float64)
    lib().oracle_mean_memory(_p(M), L, Hq, D, _p(out))
    return out


def residual(rule_c, kbar, mbar, Kq, w: ResidualWeights, flags=0, want_z=False):
    """O6c (Eq. 4-6) on a candidate list. Returns s[nc] float64 (and z if asked)."""
    rule_c = _c(rule_c, np.float64)
    kbar = _c(kbar, np.float64)
    nc, D = kbar.shape
    mbar = _c(mbar, np.float64)
    Kq = _c(Kq, np.float64).reshape(-1, D)
    s = np.zeros(nc, np.float64)
    z = np.zeros(nc, np.float64) if want_z else None
    arrs = w.arrays()
    lib().oracle_residual(_p(rule_c), _p(kbar), nc, _p(mbar), _p(Kq), Kq.shape[0], D,
                          *[_p(a) for a in arrs], C.c_double(w.alpha), int(flags), _p(s), _p(z))
    return (s, z) if want_z else s


def select(scores, cls, C_budget):
    """O7 (Eq. 1). scores fp32 [N]. Returns (keep[N] uint8, n_kept)."""
    scores = _c(scores, np.float32)
    N = scores.shape[0]
    keep = np.zeros(N, np.uint8)
    nk = np.zeros(1, np.int32)
    lib().oracle_select(_p(scores), _p(_c(cls, np.uint8)), N, int(C_budget), _p(keep), _p(nk))
    return keep, int(nk[0])


def rewrite(S, dead, keep, radix_len, n_slots):
    """O8 (Eq. 7 + prefix-safe free). Returns (S' int32, valid uint8, freed int32[n_freed])."""
    S = np.array(S, dtype=np.int32, copy=True)
    N = S.shape[0]
    valid = np.zeros(N, np.uint8)
    freed = np.zeros(max(N, 1), np.int32)
    nf = np.zeros(1, np.int32)
    lib().oracle_rewrite(_p(S), N, int(dead), _p(_c(keep, np.uint8)), int(radix_len), C.c_int64(n_slots),
                         _p(valid), _p(freed), _p(nf))
    return S, valid, freed[: int(nf[0])].copy()


def decode(g: Geometry, k_pool, v_pool, layer, S, q, sm_scale, attend_all=False):
    """O9: dense softmax attention over {j : S[j] != dead}. q: [Hq,D] fp32 -> [Hq,D] float64."""
    S = _c(S, np.int32)
    q = _c(q, np.float32)
    out = np.zeros((g.Hq, g.D), np.float64)
    common = (_p(_pool(g, k_pool)), _p(_pool(g, v_pool)), g.kv_dtype, C.c_int64(g.n_slots), g.L, g.Hq,
              g.Hkv, g.D, int(layer), _p(S), S.shape[0])
    if attend_all:
        lib().oracle_decode_attend_all(*common, _p(q), C.c_double(sm_scale), _p(out))
    else:
        lib().oracle_decode(*common, int(g.dead_slot), _p(q), C.c_double(sm_scale), _p(out))
    return out


def score(g: Geometry, k_pool, M, S, pi, qs, qe, mode=MODE_MEMORY, flags=0, xattn_pos=None,
          w: ResidualWeights | None = None, want_rule=False):
    """Composite scoring call. Returns scores[N] fp32."""
    S = _c(S, np.int32)
    N = S.shape[0]
    M = _c(M, np.float64)
    scores = np.zeros(N, np.float32)
    rule = np.zeros(N, np.float64) if want_rule else None
    if xattn_pos is None:
        xattn_pos = np.arange(qs, qe, dtype=np.int32)
    xattn_pos = _c(xattn_pos, np.int32)
    if mode == MODE_LEARNABLE:
        assert w is not None
        arrs = w.arrays()
        alpha = w.alpha
    else:
        arrs = [None] * 10
        alpha = 0.0
    lib().oracle_score(_p(_pool(g, k_pool)), g.kv_dtype, C.c_int64(g.n_slots), g.L, g.Hq, g.Hkv, g.D,
                       _p(M), _p(S), N, int(g.dead_slot), int(pi), int(qs), int(qe), int(mode), int(flags),
                       _p(xattn_pos), xattn_pos.shape[0], *[_p(a) for a in arrs], C.c_double(alpha),
                       _p(scores), _p(rule))
    return (scores, rule) if want_rule else scores


def residual_param_count(D: int) -> int:
    return int(lib().oracle_residual_param_count(int(D)))


def prune_event(g: Geometry, k_pool, M, S, pi, qs, qe, C_budget, radix_len, mode=MODE_MEMORY,
                flags=0, xattn_pos=None, w=None):
    """One whole compression event (score -> select -> rewrite)."""
    sc = score(g, k_pool, M, S, pi, qs, qe, mode, flags, xattn_pos, w)
    cls, _ = partition(S, g.dead_slot, pi, qs, qe)
    keep, n_kept = select(sc, cls, C_budget)
    S2, valid, freed = rewrite(S, g.dead_slot, keep, radix_len, g.n_slots)
    return dict(scores=sc, keep=keep, n_kept=n_kept, slot_map=S2, valid=valid, freed=freed)


# ---------------------------------------------------------------------------------------------
# SURVEY 8(f) follow-ups (ikv_oracle_next.c)
# ---------------------------------------------------------------------------------------------
def multirow_score(g: Geometry, k_pool, rows, weights, S, cls):
    """N1: rows [R][L][Hq][D], weights [R] -> scores [N] (0 outside the candidates)."""
    rows = _c(rows, np.float64)
    w = _c(weights, np.float64)
    S = _c(S, np.int32)
    cls = _c(cls, np.uint8)
    out = np.zeros(S.shape[0], np.float64)
    lib().oracle_multirow_score(_p(_pool(g, k_pool)), g.kv_dtype, C.c_int64(g.n_slots), g.L, g.Hq, g.Hkv, g.D,
                                _p(rows), rows.shape[0], _p(w), _p(S), _p(cls), S.shape[0], _p(out))
    return out


def maxpool_candidates(s, cls, kernel):
    s = _c(s, np.float64)
    cls = _c(cls, np.uint8)
    out = np.zeros_like(s)
    lib().oracle_maxpool_candidates(_p(s), _p(cls), s.shape[0], int(kernel), _p(out))
    return out


def streaming_scores(cls, n_sink):
    cls = _c(cls, np.uint8)
    out = np.zeros(cls.shape[0], np.float64)
    lib().oracle_streaming_scores(_p(cls), cls.shape[0], int(n_sink), _p(out))
    return out


def h2o_scores(hh, cls, C_budget, ratio, floor_):
    hh = _c(hh, np.float64)
    cls = _c(cls, np.uint8)
    out = np.zeros_like(hh)
    lib().oracle_h2o_scores(_p(hh), _p(cls), hh.shape[0], int(C_budget), C.c_double(ratio), int(floor_), _p(out))
    return out


def prefill(g: Geometry, k_pool, v_pool, layer, S, q_pos0, q, sm_scale):
    """N2: q [n_q][Hq][D] fp32 -> (out [n_q][Hq][D] float64, raw_reads, eff_reads)."""
    q = _c(q, np.float32)
    S = _c(S, np.int32)
    out = np.zeros(q.shape, np.float64)
    reads = np.zeros(2, np.int64)
    lib().oracle_prefill(_p(_pool(g, k_pool)), _p(_pool(g, v_pool)), g.kv_dtype, C.c_int64(g.n_slots), g.Hq, g.Hkv,
                         g.D, int(layer), _p(S), int(g.dead_slot), int(q_pos0), q.shape[0], _p(q),
                         C.c_double(sm_scale), _p(out), _p(reads))
    return out, int(reads[0]), int(reads[1])


def train_loss(s, y, mem_rows=None, rho=0.05, gamma=0.01, eta=0.001):
    """N4: Eq. 8 and dL/ds.  s [n] float64, y [n] int32 (1 / 0 / -100), mem_rows [R][D] or None.
    Returns (terms[5] = L, L_BCE, L_rank, keep, norm; grad [n])."""
    s = _c(s, np.float64)
    y = _c(y, np.int32)
    if mem_rows is None:
        mem_rows = np.zeros((0, 1), np.float64)
    mem_rows = _c(mem_rows, np.float64)
    terms = np.zeros(5, np.float64)
    grad = np.zeros(s.shape[0], np.float64)
    lib().oracle_train_loss(_p(s), _p(y), s.shape[0], _p(mem_rows), mem_rows.shape[0], mem_rows.shape[1],
                            C.c_double(rho), C.c_double(gamma), C.c_double(eta), _p(terms), _p(grad))
    return terms, grad
