"""Seeded synthetic workloads (DESIGN.md section 5 "Input recipe").

This module serves BOTH the CPU oracle (through tests / bench) and the CUDA path.  It holds
none of the method's arithmetic: it only draws random tensors with the shapes, value
distributions and paging structure of the paper's workloads (BASELINE.json `configs`) and
lays them out in a paged pool.  It imports neither `oracle/` nor the CUDA binding.

Stand-in note: the paper measures on BrowseComp-Plus / FRAMES agent trajectories with
Qwen3-8B / Qwen2.5-14B weights; none of that exists here, so i.i.d.
N(0,1) K/V with outlier channels, random page placement and planted memory-aligned
evidence tokens stand in for it (shapes: PAPER.md:183, 226-243, 251, 349).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

PAGE = 16


@dataclass
class ModelShape:
    L: int
    Hq: int
    Hkv: int
    D: int
    kv_dtype: str = "bf16"  # "bf16" | "f32"

    @property
    def G(self):
        return self.Hq // self.Hkv

    @property
    def torch_dtype(self):
        return torch.bfloat16 if self.kv_dtype == "bf16" else torch.float32

    @property
    def elem_bytes(self):
        return 2 if self.kv_dtype == "bf16" else 4


TINY = ModelShape(L=1, Hq=4, Hkv=2, D=64, kv_dtype="f32")
QWEN3_8B = ModelShape(L=36, Hq=32, Hkv=8, D=128)
QWEN25_14B = ModelShape(L=48, Hq=40, Hkv=8, D=128)


@dataclass
class SessionSpec:
    session_id: int
    n_tokens: int          # N at the time of the prune
    n_mem_rows: int        # BASELINE.json "QueryMemory of M vectors": source rows, 4 per update
    budget: int            # C
    prefix_len: int = 256  # pi
    span_len: int = 64     # actionable span = last span_len tokens
    n_planted: int = 0
    decode_tokens: int = 0  # slots pre-allocated after N for decode appends


@dataclass
class Session:
    spec: SessionSpec
    slot_map: torch.Tensor        # int32 [N + decode_tokens] (CPU); positions >= N are the decode appends
    mem_rows: torch.Tensor        # fp32 [n_mem_rows, L, Hq, D]  (CPU)
    planted_pos: np.ndarray       # int32 positions of planted evidence tokens
    planted_row: np.ndarray       # int32 index of the memory row each planted token follows

    @property
    def N(self):
        return self.spec.n_tokens

    @property
    def pi(self):
        return self.spec.prefix_len

    @property
    def qs(self):
        return self.spec.n_tokens - self.spec.span_len

    @property
    def qe(self):
        return self.spec.n_tokens

    def updates(self, rows_per_update=4):
        """Memory rows grouped as they are fed to ikv_memory_update (4 rows per update)."""
        n = self.mem_rows.shape[0]
        return [self.mem_rows[i:i + rows_per_update] for i in range(0, n, rows_per_update)]


@dataclass
class Workload:
    shape: ModelShape
    n_slots: int
    dead_slot: int
    k_pool: torch.Tensor  # [L, n_slots, Hkv, D] on `device`
    v_pool: torch.Tensor
    sessions: list = field(default_factory=list)
    seed: int = 0


def _gen(seed, device):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def _fill_normal(shape: ModelShape, n_slots, seed, device, outlier_seed, chunk_layers=4):
    """i.i.d. N(0,1) pool with 4 outlier channels (x8) per (layer, kv head)."""
    pool = torch.empty((shape.L, n_slots, shape.Hkv, shape.D), dtype=shape.torch_dtype, device=device)
    g = _gen(seed, device)
    og = _gen(outlier_seed, "cpu")
    for l0 in range(0, shape.L, chunk_layers):
        l1 = min(shape.L, l0 + chunk_layers)
        x = torch.randn((l1 - l0, n_slots, shape.Hkv, shape.D), generator=g, device=device, dtype=torch.float32)
        for l in range(l0, l1):
            for h in range(shape.Hkv):
                ch = torch.randperm(shape.D, generator=og)[:4].to(device)
                x[l - l0, :, h, ch] *= 8.0
        pool[l0:l1] = x.to(shape.torch_dtype)
    return pool


def make_workload(shape: ModelShape, specs, seed: int, device="cpu", outliers=True, spare_pages=2,
                  with_values=True) -> Workload:
    """Build one shared paged pool holding every session in `specs`.

    Seeds: seed+1 keys, +2 values, +3 memory rows, +4 planted positions / noise,
    +7 page permutation, +9/+10 outlier channels.
    Page 0 is reserved: slot 0 is the dead slot s+ (reading R17); logical pages of all sessions are
    placed at seeded random physical pages, so no session is physically contiguous.
    """
    pages_per = [(s.n_tokens + s.decode_tokens + PAGE - 1) // PAGE for s in specs]
    n_pages = 1 + sum(pages_per) + spare_pages
    n_slots = n_pages * PAGE
    if not with_values:     # the pruning pass never reads V (the CPU baseline of bench.py uses the key pool only)
        k_pool = _fill_normal(shape, n_slots, seed + 1, device, seed + 9)
        v_pool = torch.empty((shape.L, 0, shape.Hkv, shape.D), dtype=shape.torch_dtype, device=device)
    elif outliers:
        k_pool = _fill_normal(shape, n_slots, seed + 1, device, seed + 9)
        v_pool = _fill_normal(shape, n_slots, seed + 2, device, seed + 10)
    else:
        k_pool = torch.randn((shape.L, n_slots, shape.Hkv, shape.D), generator=_gen(seed + 1, device),
                             device=device, dtype=torch.float32).to(shape.torch_dtype)
        v_pool = torch.randn((shape.L, n_slots, shape.Hkv, shape.D), generator=_gen(seed + 2, device),
                             device=device, dtype=torch.float32).to(shape.torch_dtype)
    perm = 1 + torch.randperm(n_pages - 1, generator=_gen(seed + 7, "cpu"))
    sessions = []
    page_cursor = 0
    gm = _gen(seed + 3, "cpu")
    gp = _gen(seed + 4, "cpu")
    for spec, npg in zip(specs, pages_per):
        phys = perm[page_cursor:page_cursor + npg]
        page_cursor += npg
        n_pos = spec.n_tokens + spec.decode_tokens
        pos = torch.arange(n_pos)
        slot_map = (phys[pos // PAGE] * PAGE + pos % PAGE).to(torch.int32)
        mem_rows = torch.randn((spec.n_mem_rows, shape.L, shape.Hq, shape.D), generator=gm, dtype=torch.float32)
        # planted evidence: candidate positions only (outside prefix and span)
        lo, hi = spec.prefix_len, spec.n_tokens - spec.span_len
        n_pl = min(spec.n_planted, max(0, hi - lo))
        if n_pl > 0:
            ppos = (lo + torch.randperm(hi - lo, generator=gp)[:n_pl]).sort().values
            # follow a row of the most recent update (the current intent)
            last = max(0, spec.n_mem_rows - 4)
            prow = last + torch.randint(0, spec.n_mem_rows - last, (n_pl,), generator=gp)
            noise = torch.randn((n_pl, shape.L, shape.Hkv, shape.D), generator=gp, dtype=torch.float32)
            # "keys = memory vector + 0.1*noise" (BASELINE.json configs[0]); the memory vector of KV head
            # kvh is the source row at the first query head of its group
            src = mem_rows[prow][:, :, ::shape.G, :]            # [n_pl, L, Hkv, D]
            vals = (src + 0.1 * noise).to(shape.torch_dtype)     # [n_pl, L, Hkv, D]
            slots = slot_map[ppos].long().to(device)
            k_pool[:, slots] = vals.permute(1, 0, 2, 3).to(device)
            planted_pos = ppos.numpy().astype(np.int32)
            planted_row = prow.numpy().astype(np.int32)
        else:
            planted_pos = np.zeros(0, np.int32)
            planted_row = np.zeros(0, np.int32)
        sessions.append(Session(spec, slot_map, mem_rows, planted_pos, planted_row))
    return Workload(shape, n_slots, 0, k_pool, v_pool, sessions, seed)


# ---------------------------------------------------------------------------------------------
# named configurations (BASELINE.json `configs`)
# ---------------------------------------------------------------------------------------------
def tiny(device="cpu", seed=0) -> Workload:
    """configs[0]: 1 layer, 4 Q / 2 KV heads, D=64, fp32, 512 live tokens, M=8, 16 planted, C=128."""
    spec = SessionSpec(session_id=1, n_tokens=512, n_mem_rows=8, budget=128, prefix_len=16, span_len=16,
                       n_planted=16, decode_tokens=16)
    return make_workload(TINY, [spec], seed, device, outliers=False)


def cfg1(device="cpu", seed=1000, n_tokens=32768, budget=8192, decode_tokens=256, shape=QWEN3_8B,
         n_mem_rows=64, with_values=True) -> Workload:
    """configs[1]: Qwen3-8B shape, 32,768 live tokens, M=64, 1% planted, C=8192, 256 decode steps."""
    n_cand = n_tokens - 256 - 64
    spec = SessionSpec(session_id=1, n_tokens=n_tokens, n_mem_rows=n_mem_rows, budget=budget,
                       n_planted=max(1, n_cand // 100), decode_tokens=decode_tokens)
    return make_workload(shape, [spec], seed, device, with_values=with_values)


def cfg2(device="cpu", seed=2000, n_tokens=92160, budget=8192, decode_tokens=256) -> Workload:
    """configs[2]: Qwen2.5-14B shape, 92,160 live tokens, M=256, C=8192."""
    return cfg1(device, seed, n_tokens, budget, decode_tokens, QWEN25_14B, 256)


def small(device="cpu", seed=77, shape=None, n_tokens=1500, budget=400, prefix_len=37, span_len=21,
          n_mem_rows=8, n_planted=12, decode_tokens=5, kv_dtype="bf16") -> Workload:
    """Parity-test size: several tiles plus a ragged tail, finishes in seconds on the oracle."""
    shape = shape or ModelShape(L=3, Hq=8, Hkv=2, D=128, kv_dtype=kv_dtype)
    spec = SessionSpec(session_id=7, n_tokens=n_tokens, n_mem_rows=n_mem_rows, budget=budget,
                       prefix_len=prefix_len, span_len=span_len, n_planted=n_planted,
                       decode_tokens=decode_tokens)
    return make_workload(shape, [spec], seed, device)


def batched(device="cpu", seed=4000, shape=QWEN3_8B, n_sessions=64, median=16384, lo=4096, hi=65536,
            sigma=0.5, budgets=(4096, 8192, 16384), decode_tokens=0, with_values=True) -> Workload:
    """configs[4]: concurrent sessions with lognormal live lengths in one shared pool."""
    g = _gen(seed + 8, "cpu")
    z = torch.randn(n_sessions, generator=g)
    lens = torch.clamp((median * torch.exp(sigma * z)).round(), lo, hi).to(torch.int64).tolist()
    mrows = (4 * torch.randint(8, 65, (n_sessions,), generator=g)).tolist()
    specs = []
    for i, (n, m) in enumerate(zip(lens, mrows)):
        n_cand = n - 256 - 64
        specs.append(SessionSpec(session_id=100 + i, n_tokens=int(n), n_mem_rows=int(m),
                                 budget=budgets[i % len(budgets)], n_planted=max(1, n_cand // 100),
                                 decode_tokens=decode_tokens))
    return make_workload(shape, specs, seed, device, with_values=with_values)


def residual_weights(D: int, seed: int, zero_init: bool = False) -> dict:
    """Residual-head parameters as fp32 numpy arrays, row-major [out][in].

    random: torch-default Linear init U(-1/sqrt(in), 1/sqrt(in)) for all five layers' weights and
    biases, fc2 ~ N(0, 0.02^2), alpha = 1.1.  zero_init: fc2 = 0, b2 = 0, alpha = 1
    (PAPER.md:115).
    """
    g = _gen(seed, "cpu")
    P, DC, HID = 3 * D + 1, 128, 256

    def lin(out, inp):
        b = 1.0 / np.sqrt(inp)
        w = (torch.rand((out, inp), generator=g) * 2 - 1) * b
        bias = (torch.rand((out,), generator=g) * 2 - 1) * b
        return w.numpy().astype(np.float32), bias.numpy().astype(np.float32)

    wq, bq = lin(DC, P)
    wk, bk = lin(DC, D)
    wv, bv = lin(DC, D)
    fc1_w, fc1_b = lin(HID, P + DC)
    if zero_init:
        fc2_w = np.zeros(HID, np.float32)
        fc2_b = np.zeros(1, np.float32)
        alpha = 1.0
    else:
        fc2_w = (torch.randn((HID,), generator=g) * 0.02).numpy().astype(np.float32)
        fc2_b = (torch.randn((1,), generator=g) * 0.02).numpy().astype(np.float32)
        alpha = 1.1
    return dict(wq=wq, bq=bq, wk=wk, bk=bk, wv=wv, bv=bv, fc1_w=fc1_w, fc1_b=fc1_b, fc2_w=fc2_w,
                fc2_b=fc2_b, alpha=alpha)


def decode_queries(shape: ModelShape, n_steps: int, seed: int, device="cpu") -> torch.Tensor:
    """q ~ N(0,1) in bf16, [n_steps, L, Hq, D]."""
    return torch.randn((n_steps, shape.L, shape.Hq, shape.D), generator=_gen(seed + 6, device), device=device,
                       dtype=torch.float32).to(torch.bfloat16)


def to_numpy_bits(t: torch.Tensor) -> np.ndarray:
    """Host numpy view of the exact bits: bf16 -> uint16, fp32 -> float32."""
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16)
    return t.numpy()
