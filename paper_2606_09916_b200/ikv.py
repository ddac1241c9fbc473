"""ctypes binding of libikv.so (include/ikv.h).  Argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; this module only turns torch tensors into
device pointers and request structs.  It fails loudly at import if the library is missing: there is no CPU
fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libikv.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2606_09916_b200.build` "
                      "(there is no CPU fallback)")
_lib = C.CDLL(_LIB_PATH)

OK = 0
ERR_INVALID_ARG, ERR_NO_SESSION, ERR_CAPACITY, ERR_OOM, ERR_CUDA, ERR_UNSUPPORTED = -1, -2, -3, -4, -5, -6
F32, BF16 = 0, 1
MODE_MEMORY, MODE_LEARNABLE, MODE_QUERY = 0, 1, 2
FLAG_NO_XATTN, FLAG_NO_RESIDUAL = 0x100, 0x200
REQ_RESCAN, REQ_INPUTS_COMPLETE = 1, 2
CFG_NO_PDL, CFG_NO_PDL_PRUNE = 1, 2
TUNE_L2_HINTS, TUNE_RESID_TC, TUNE_LAYER_MAJOR, TUNE_BATCH_LANES, TUNE_ROWS_TC, TUNE_PREFILL_TILED = 1, 2, 3, 4, 5, 6
PROF_SLOTS = 12
PROF_NAMES = ["key_pass", "decode_split", "memory_update", "partition", "mem_prep", "post_key", "rule_fold", "residual",
              "select_evict", "decode_merge"]

EXPORTS = ["ikv_create", "ikv_destroy", "ikv_last_error", "ikv_reserve", "ikv_session_open", "ikv_session_fork",
           "ikv_session_close", "ikv_session_get_memory", "ikv_session_set_memory", "ikv_residual_load",
           "ikv_memory_update", "ikv_score", "ikv_select_evict", "ikv_decode_attn", "ikv_prune_host",
           "ikv_score_rows", "ikv_score_baseline", "ikv_prefill_attn", "ikv_decode_attn_static", "ikv_train_loss", "ikv_profile_enable", "ikv_profile_read", "ikv_tune", "ikv_test_late_writer", "ikv_version"]


class Config(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("page_size", C.c_int32), ("kv_dtype", C.c_int32), ("n_slots", C.c_int64),
                ("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("dead_slot", C.c_int32), ("lambda_", C.c_float),
                ("max_sessions", C.c_int32), ("flags", C.c_int32)]


class Request(C.Structure):
    _fields_ = [("session_id", C.c_uint64), ("slot_map", C.c_void_p), ("valid_mask", C.c_void_p),
                ("seq_len", C.c_int32), ("prefix_len", C.c_int32), ("q_start", C.c_int32), ("q_end", C.c_int32),
                ("budget", C.c_int32), ("radix_protected_len", C.c_int32), ("xattn_pos", C.c_void_p),
                ("n_xattn_pos", C.c_int32), ("flags", C.c_int32), ("map_epoch", C.c_uint32)]


class ResidualWeights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("wq", "bq", "wk", "bk", "wv", "bv", "fc1_w", "fc1_b", "fc2_w", "fc2_b")] + \
               [("alpha", C.c_float)]


_lib.ikv_version.restype = C.c_char_p
_lib.ikv_last_error.restype = C.c_char_p
_lib.ikv_last_error.argtypes = [C.c_void_p]
for _n in EXPORTS:
    if _n not in ("ikv_version", "ikv_last_error"):
        getattr(_lib, _n).restype = C.c_int32
_lib.ikv_create.argtypes = [C.POINTER(Config), C.POINTER(C.c_void_p)]
_lib.ikv_destroy.argtypes = [C.c_void_p]
_lib.ikv_reserve.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
_lib.ikv_session_open.argtypes = [C.c_void_p, C.c_uint64]
_lib.ikv_session_fork.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p]
_lib.ikv_session_close.argtypes = [C.c_void_p, C.c_uint64]
_lib.ikv_session_get_memory.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p]
_lib.ikv_session_set_memory.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p]
_lib.ikv_residual_load.argtypes = [C.c_void_p, C.POINTER(ResidualWeights)]
_lib.ikv_memory_update.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
_lib.ikv_score.argtypes = [C.c_void_p, C.POINTER(Request), C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ikv_select_evict.argtypes = [C.c_void_p, C.POINTER(Request), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_void_p]
_lib.ikv_decode_attn.argtypes = [C.c_void_p, C.c_int32, C.POINTER(Request), C.c_int32, C.c_void_p, C.c_void_p,
                                 C.c_float, C.c_void_p]
_lib.ikv_decode_attn_static.argtypes = [C.c_void_p, C.c_int32, C.POINTER(Request), C.c_void_p, C.c_void_p, C.c_float,
                                        C.c_void_p]
class LossCfg(C.Structure):
    _fields_ = [("rho", C.c_float), ("gamma", C.c_float), ("eta", C.c_float)]


_lib.ikv_train_loss.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32,
                                C.POINTER(LossCfg), C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ikv_tune.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
_lib.ikv_test_late_writer.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p]
_lib.ikv_profile_enable.argtypes = [C.c_void_p, C.c_int32]
_lib.ikv_profile_read.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ikv_prune_host.argtypes = [C.c_void_p, C.POINTER(Request), C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p,
                                C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]


class Baseline(C.Structure):
    _fields_ = [("kind", C.c_int32), ("rows", C.c_void_p), ("n_rows", C.c_int32), ("n_sink", C.c_int32),
                ("pool_kernel", C.c_int32), ("recent_ratio", C.c_float), ("recent_floor", C.c_int32)]


BASE_STREAMING, BASE_SNAPKV, BASE_H2O = 1, 2, 3
STATIC_SCRATCH_BYTES = 3 * 1024 * 1024
_lib.ikv_score_rows.argtypes = [C.c_void_p, C.POINTER(Request), C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p,
                                C.c_void_p]
_lib.ikv_score_baseline.argtypes = [C.c_void_p, C.POINTER(Request), C.c_int32, C.POINTER(Baseline), C.c_void_p, C.c_void_p]
_lib.ikv_prefill_attn.argtypes = [C.c_void_p, C.c_int32, C.POINTER(Request), C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                  C.c_float, C.c_void_p, C.c_void_p]


class IkvError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"ikv status {status}: {msg}")
        self.status = status


def version() -> str:
    return _lib.ikv_version().decode()


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def make_request(session_id, slot_map, seq_len, prefix_len, q_start, q_end, budget, radix_protected_len=0,
                 valid_mask=None, xattn_pos=None, flags=0, map_epoch=0) -> Request:
    r = Request()
    r.session_id = session_id
    r.slot_map = slot_map.data_ptr() if slot_map is not None else None
    r.valid_mask = valid_mask.data_ptr() if valid_mask is not None else None
    r.seq_len, r.prefix_len, r.q_start, r.q_end = seq_len, prefix_len, q_start, q_end
    r.budget, r.radix_protected_len = budget, radix_protected_len
    r.xattn_pos = xattn_pos.data_ptr() if xattn_pos is not None else None
    r.n_xattn_pos = int(xattn_pos.numel()) if xattn_pos is not None else 0
    r.flags = flags
    r.map_epoch = map_epoch
    return r


def _req_array(reqs):
    arr = (Request * len(reqs))(*reqs)
    return arr


class Context:
    """Thin owner of an ikv_ctx*.  Methods have the names of the C entry points (without the prefix)."""

    def __init__(self, n_layers, n_q_heads, n_kv_heads, head_dim, k_pool, v_pool, dead_slot=0, page_size=16,
                 lam=0.5, max_sessions=1024, flags=0):
        assert k_pool.is_cuda and v_pool.is_cuda and k_pool.is_contiguous() and v_pool.is_contiguous()
        assert k_pool.dtype == v_pool.dtype and k_pool.dtype in (torch.bfloat16, torch.float32)
        assert tuple(k_pool.shape) == (n_layers, k_pool.shape[1], n_kv_heads, head_dim) == tuple(v_pool.shape)
        self.k_pool, self.v_pool = k_pool, v_pool  # keep alive
        cfg = Config(n_layers, n_q_heads, n_kv_heads, head_dim, page_size,
                     BF16 if k_pool.dtype == torch.bfloat16 else F32, k_pool.shape[1], k_pool.data_ptr(),
                     v_pool.data_ptr(), dead_slot, lam, max_sessions, flags)
        self.cfg = cfg
        self._h = C.c_void_p()
        st = _lib.ikv_create(C.byref(cfg), C.byref(self._h))
        if st != OK:
            raise IkvError(st, _lib.ikv_last_error(None).decode() or "ikv_create failed")

    def _chk(self, st):
        if st != OK:
            raise IkvError(st, _lib.ikv_last_error(self._h).decode())

    def close(self):
        if self._h:
            _lib.ikv_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reserve(self, max_tokens, max_requests=1):
        self._chk(_lib.ikv_reserve(self._h, max_tokens, max_requests))

    def session_open(self, sid):
        self._chk(_lib.ikv_session_open(self._h, sid))

    def session_fork(self, parent, child, stream=None):
        self._chk(_lib.ikv_session_fork(self._h, parent, child, _stream(stream)))

    def session_close(self, sid):
        self._chk(_lib.ikv_session_close(self._h, sid))

    def session_get_memory(self, sid):
        out = torch.empty((self.cfg.n_layers, self.cfg.n_q_heads, self.cfg.head_dim), dtype=torch.float32)
        self._chk(_lib.ikv_session_get_memory(self._h, sid, C.c_void_p(out.data_ptr())))
        return out

    def session_set_memory(self, sid, m):
        m = m.detach().to("cpu", torch.float32).contiguous()
        self._chk(_lib.ikv_session_set_memory(self._h, sid, C.c_void_p(m.data_ptr())))

    def residual_load(self, w: dict):
        import numpy as np
        keep = {k: np.ascontiguousarray(w[k], dtype=np.float32) for k in
                ("wq", "bq", "wk", "bk", "wv", "bv", "fc1_w", "fc1_b", "fc2_w", "fc2_b")}
        rw = ResidualWeights(*[keep[k].ctypes.data for k in
                               ("wq", "bq", "wk", "bk", "wv", "bv", "fc1_w", "fc1_b", "fc2_w", "fc2_b")],
                             float(w["alpha"]))
        self._chk(_lib.ikv_residual_load(self._h, C.byref(rw)))

    def memory_update(self, sid, q_rows, stream=None):
        assert q_rows.is_cuda and q_rows.is_contiguous() and q_rows.dtype in (torch.float32, torch.bfloat16)
        self._chk(_lib.ikv_memory_update(self._h, sid, _ptr(q_rows), q_rows.shape[0],
                                         F32 if q_rows.dtype == torch.float32 else BF16, _stream(stream)))

    def score(self, reqs, mode, scores, rule_out=None, stream=None):
        self._chk(_lib.ikv_score(self._h, _req_array(reqs), len(reqs), mode, _ptr(scores), _ptr(rule_out),
                                 _stream(stream)))

    def select_evict(self, reqs, scores, freed_slots, n_freed, n_kept, stream=None):
        self._chk(_lib.ikv_select_evict(self._h, _req_array(reqs), len(reqs), _ptr(scores), _ptr(freed_slots),
                                        _ptr(n_freed), _ptr(n_kept), _stream(stream)))

    def decode_attn(self, layer, reqs, q, out, sm_scale, stream=None):
        self._chk(_lib.ikv_decode_attn(self._h, layer, _req_array(reqs), len(reqs), _ptr(q), _ptr(out),
                                       C.c_float(sm_scale), _stream(stream)))

    def train_loss(self, scores, labels, terms, grad, mem_rows=None, rho=0.05, gamma=0.01, eta=0.001, stream=None):
        """Eq. 8 and dL/dscores for one row of scores (device tensors; terms [5], grad [n] are written)."""
        cfg = LossCfg(rho, gamma, eta)
        nr, rd = (0, 0) if mem_rows is None else (mem_rows.shape[0], mem_rows.shape[1])
        self._chk(_lib.ikv_train_loss(self._h, _ptr(scores), _ptr(labels), scores.numel(), _ptr(mem_rows), nr, rd,
                                      C.byref(cfg), _ptr(terms), _ptr(grad), _stream(stream)))

    def decode_attn_static(self, layer, req, q, out, sm_scale, stream=None):
        """One request, no session, no allocation: split partials in the library's static device array."""
        self._chk(_lib.ikv_decode_attn_static(self._h, layer, C.byref(req), _ptr(q), _ptr(out), C.c_float(sm_scale),
                                              _stream(stream)))

    @staticmethod
    def test_late_writer(dst, src, delay_us, stream=None):
        """Test support: dst <- src by a kernel that triggers its dependents first and writes delay_us later."""
        st = _lib.ikv_test_late_writer(_ptr(dst), _ptr(src), src.numel() * src.element_size(), delay_us, _stream(stream))
        if st != OK:
            raise IkvError(st, "ikv_test_late_writer failed")

    def tune(self, knob: int, value: int):
        self._chk(_lib.ikv_tune(self._h, knob, value))

    def score_rows(self, reqs, rows, weights, scores, stream=None):
        assert rows.is_cuda and rows.is_contiguous() and rows.dtype == torch.float32
        w = (C.c_float * len(weights))(*[float(x) for x in weights])
        assert rows.shape[0] == len(weights)
        self._chk(_lib.ikv_score_rows(self._h, _req_array(reqs), len(reqs), _ptr(rows), rows.shape[0], w, _ptr(scores),
                                      _stream(stream)))

    def score_baseline(self, reqs, kind, scores, rows=None, n_sink=4, pool_kernel=7, recent_ratio=0.5, recent_floor=0,
                       stream=None):
        b = Baseline(kind, _ptr(rows).value if rows is not None else None, 0 if rows is None else rows.shape[0], n_sink,
                     pool_kernel, recent_ratio, recent_floor)
        self._chk(_lib.ikv_score_baseline(self._h, _req_array(reqs), len(reqs), C.byref(b), _ptr(scores), _stream(stream)))

    def prefill_attn(self, layer, req, q_pos0, q, out, sm_scale, kv_reads=None, stream=None):
        self._chk(_lib.ikv_prefill_attn(self._h, layer, C.byref(req), q_pos0, q.shape[0], _ptr(q), _ptr(out),
                                        C.c_float(sm_scale), _ptr(kv_reads), _stream(stream)))

    def profile_enable(self, level):
        """0/False off, 1/True the two dominant kernels, 2 every kernel (diagnostic)."""
        self._chk(_lib.ikv_profile_enable(self._h, int(level)))

    def profile_read(self) -> dict:
        ms = (C.c_float * PROF_SLOTS)()
        n = (C.c_int32 * PROF_SLOTS)()
        self._chk(_lib.ikv_profile_read(self._h, ms, n))
        out = {"score_logits_ms": ms[0], "score_logits_n": n[0], "decode_split_ms": ms[1], "decode_split_n": n[1]}
        out["slots"] = {name: (ms[i], n[i]) for i, name in enumerate(PROF_NAMES) if n[i] > 0}
        return out

    def prune_host(self, req, q_rows_host, mode, slot_map_host, valid_host, scores_host, freed_host, stream=None):
        """HOST-buffer variant. Tensors are CPU tensors (pinned or not). Returns (n_freed, n_kept)."""
        nf, nk = C.c_int32(0), C.c_int32(0)
        n_rows = 0 if q_rows_host is None else q_rows_host.shape[0]
        q_dtype = BF16 if (q_rows_host is not None and q_rows_host.dtype == torch.bfloat16) else F32
        self._chk(_lib.ikv_prune_host(self._h, C.byref(req), _ptr(q_rows_host), n_rows, q_dtype, mode, _ptr(slot_map_host),
                                      _ptr(valid_host), _ptr(scores_host), _ptr(freed_host), C.byref(nf),
                                      C.byref(nk), _stream(stream)))
        return nf.value, nk.value
