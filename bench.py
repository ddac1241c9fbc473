#!/usr/bin/env python
"""bench.py -- IntentKV hot path on B200: history tokens scored+pruned per second at C=8k.

One "step" = one pass of the whole hot path over one synthetic Qwen3-8B-shaped session (BASELINE.json
configs[1]): ikv_memory_update (4 rows) -> ikv_score (LEARNABLE: rule + residual head) -> ikv_select_evict
(C = 8192) -> 256 decode steps x 36 layers of ikv_decode_attn through the pruned slot map (CUDA graph).
`value` = live history tokens / time of the pruning pass (memory update + score + select/evict), the metric
BASELINE.json names; the decode stage is reported beside it (`decode`, `roofline_decode`), and configs[2] / configs[4]
as sub-objects `cfg2` / `cfg4` of the same line; `next` holds the widened rows (multi-row scorer, baselines, prefill).

  python bench.py [--gpus N] [--steps K] [--warmup W]            # our arm (N>1: under torchrun, replicas)
  python bench.py --impl reference ...                           # the CPU oracle timed on the host cores
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "history tokens scored+pruned/sec at C=8k"
UNIT = "tokens/s"
NOMINAL_HBM_GBS = 8000.0
TRAFFIC_CSV = "r2_ncu_full.csv"       # profiles/: `ncu --set full` capture of this workload (command in r2_summary.md)
CFG1_TEXT = ("configs[1] Qwen3-8B-shaped single session per GPU: 36 layers, 32 Q / 8 KV heads, head_dim 128, bf16 K/V, "
             "32,768 live tokens in 16-token pages, M=64 memory rows, 1% planted, C=8192, one prune pass then 256 decode "
             "steps")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, REPLAYED from the committed `ncu --set full`
    capture of this same workload (profiles/r2_ncu_full.csv; the command is in profiles/r2_summary.md): a number taken
    under a profiler cannot be measured inside this run.  Returns (bytes or None, source string)."""
    import csv
    path = os.path.join(ROOT, "profiles", TRAFFIC_CSV)
    if not os.path.exists(path):
        return None, None
    rows = list(csv.reader(open(path)))
    hdr, units = rows[0], rows[1]
    scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}
    ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    vals = [float(r[ir]) * scale[units[ir]] + float(r[iw]) * scale[units[iw]] for r in rows[2:] if kernel in r[0]]
    return (sum(vals) / len(vals) if vals else None), f"profiles/{TRAFFIC_CSV} (replayed ncu capture)"


def max_over_ranks(times_ms, world, device):
    """Replicas-only multi-GPU (DESIGN.md section 2, 8(e)): no data-path collective; the only exchange is this MAX of
    the device-timed milliseconds, so that `value` = units of all ranks / slowest rank's time."""
    import torch
    import torch.distributed as dist
    tt = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return tt.tolist()


def whole_job_value(units_per_rank, world, steps, total_ms):
    """Weak scaling: every rank processes `units_per_rank` per step; total_ms is the max-over-ranks time of `steps`."""
    return world * units_per_rank * steps / (total_ms * 1e-3)


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_pass(w, sess, kp_host, wts):
    """One pruning pass of the oracle, as it stands, on ALL layers and ALL tokens of the workload: memory update,
    partition, rule score, mean keys, residual head, select, rewrite.  Returns seconds."""
    import numpy as np
    from oracle import ikv_oracle as o
    shape = w.shape
    g = o.Geometry(shape.L, shape.Hq, shape.Hkv, shape.D, w.n_slots, o.BF16, w.dead_slot)
    M = np.zeros((shape.L, shape.Hq, shape.D))
    rows = sess.mem_rows.numpy()
    S = sess.slot_map[:sess.N].numpy().copy()
    t0 = time.perf_counter()
    o.memory_update(M, rows[-4:], 0.5)
    cls, _ = o.partition(S, w.dead_slot, sess.pi, sess.qs, sess.qe)
    rule = o.rule_score(g, kp_host, M, S, cls)
    cand = np.nonzero(cls == o.CAND)[0].astype(np.int32)
    kbar = o.mean_key(g, kp_host, S, cand)
    qpos = np.array([j for j in range(sess.qs, sess.qe) if S[j] != w.dead_slot], np.int32)
    Kq = o.mean_key(g, kp_host, S, qpos)
    s_c = o.residual(rule[cand], kbar, o.mean_memory(M), Kq, wts)
    scores = np.where(cls == o.FORCED, np.inf, -np.inf).astype(np.float32)
    scores[cand] = s_c.astype(np.float32)
    keep, _ = o.select(scores, cls, sess.spec.budget)
    o.rewrite(S, w.dead_slot, keep, sess.pi, w.n_slots)
    return time.perf_counter() - t0


def oracle_workload(tokens, budget):
    """The CPU copy of configs[1] for the oracle: all 36 layers of keys (2.4 GB of host memory; V is not read by the
    pruning pass and is not generated)."""
    from oracle import ikv_oracle as o
    from paper_2606_09916_b200 import workloads as wl
    w = wl.cfg1(device="cpu", decode_tokens=0, n_tokens=tokens, budget=budget, with_values=False)
    kp = wl.to_numpy_bits(w.k_pool)
    wts = o.ResidualWeights(**wl.residual_weights(w.shape.D, w.seed + 5))
    return w, kp, wts


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; every step is one full pruning pass (all layers,
    all tokens: no extrapolation)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, kp, wts = oracle_workload(args.tokens, args.budget)
    sess = w.sessions[0]
    for _ in range(min(args.warmup, 1)):
        oracle_pass(w, sess, kp, wts)
    times = [oracle_pass(w, sess, kp, wts) for _ in range(args.steps)]
    t_mean = sum(times) / len(times)
    value = sess.N / t_mean
    sample = (f"oracle pruning pass (memory update + learnable score + select + rewrite) on all {sess.N} tokens and all "
              f"{w.shape.L} layers per step, {args.steps} steps (1 warm-up pass)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_mean * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": CFG1_TEXT, "n_tokens": sess.N, "budget": sess.spec.budget, "mode": "learnable"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ our arm
class Rig:
    """One context over one workload: the prune pass, the decode loops and their timings."""

    def __init__(self, w, shape, tokens, budget, dec_steps, mode, dev, tune=()):
        import torch
        from paper_2606_09916_b200 import ikv, workloads as wl
        self.torch, self.ikv, self.wl = torch, ikv, wl
        self.w, self.shape, self.T, self.C, self.DEC, self.dev = w, shape, tokens, budget, dec_steps, dev
        self.sess = sess = w.sessions[0]
        L, Hq, Hkv, D = shape.L, shape.Hq, shape.Hkv, shape.D
        self.ctx = ctx = ikv.Context(L, Hq, Hkv, D, w.k_pool, w.v_pool, dead_slot=w.dead_slot)
        for kv in tune:                                   # experiment knobs (ikv_tune), e.g. --tune 3=0
            k, v = kv.split("=")
            ctx.tune(int(k), int(v))
        ctx.reserve(tokens + dec_steps, 1)
        ctx.residual_load(wl.residual_weights(D, w.seed + 5))
        self.sid = sess.spec.session_id
        ctx.session_open(self.sid)
        ups = [u.to(dev).contiguous() for u in sess.updates()]
        for u in ups[:-1]:
            ctx.memory_update(self.sid, u)
        self.new_rows = ups[-1]
        self.mode = ikv.MODE_LEARNABLE if mode == "learnable" else ikv.MODE_MEMORY
        self.pristine = sess.slot_map.to(dev)
        self.S_dev = self.pristine.clone()
        self.valid = torch.empty(tokens + dec_steps, dtype=torch.uint8, device=dev)
        self.scores = torch.empty(tokens, device=dev)
        self.freed = torch.empty(tokens, dtype=torch.int32, device=dev)
        self.nf = torch.zeros(1, dtype=torch.int32, device=dev)
        self.nk = torch.zeros(1, dtype=torch.int32, device=dev)
        self.req = ikv.make_request(self.sid, self.S_dev, tokens, sess.pi, sess.qs, sess.qe, budget, sess.pi,
                                    valid_mask=self.valid)
        self.scale = 1.0 / math.sqrt(D)
        self.stream = torch.cuda.Stream(device=dev)

    def prune(self, mode=None):
        c, st = self.ctx, self.stream
        c.memory_update(self.sid, self.new_rows, st)
        c.score([self.req], self.mode if mode is None else mode, self.scores, None, st)
        c.select_evict([self.req], self.scores, self.freed, self.nf, self.nk, st)

    def ev(self):
        return self.torch.cuda.Event(enable_timing=True)

    def time_prune(self, n, mode=None):
        ts = []
        for _ in range(n):
            with self.torch.cuda.stream(self.stream):
                self.S_dev.copy_(self.pristine)
                a, b = self.ev(), self.ev()
                a.record(self.stream)
                self.prune(mode)
                b.record(self.stream)
            self.stream.synchronize()
            ts.append(a.elapsed_time(b))
        return ts

    def capture_decode(self, steps, dq, dout, dependent):
        """All L layers x `steps` decode steps in one CUDA graph.  dependent=False: precomputed queries, the calls carry
        IKV_REQ_INPUTS_COMPLETE and consecutive layer calls overlap.  dependent=True: the query of every call is copied
        from the previous call's output (a real inter-layer dependency) and the calls use the default flags."""
        torch, ikv, sess, L = self.torch, self.ikv, self.sess, self.shape.L
        flags = 0 if dependent else ikv.REQ_INPUTS_COMPLETE
        qbuf = torch.zeros_like(dq[0, 0:1]) if dependent else None
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=self.stream):
            for t in range(steps):
                r = ikv.make_request(self.sid, self.S_dev, self.T + t + 1, sess.pi, sess.qs, sess.qe, self.C, sess.pi,
                                     flags=flags)
                for l in range(L):
                    if dependent:
                        qbuf.copy_(dout[t, l - 1] if l > 0 else dq[t, 0:1])      # q of this layer <- previous output
                        self.ctx.decode_attn(l, [r], qbuf, dout[t, l], self.scale, self.stream)
                    else:
                        self.ctx.decode_attn(l, [r], dq[t, l:l + 1], dout[t, l], self.scale, self.stream)
        self.stream.synchronize()
        return g


def prune_breakdown(rig, reps=10):
    """Per-kernel microseconds of the prune pass from the library's own events (profile level 2: the events between the
    launches take away the programmatic overlap, so the sum exceeds the timed pass)."""
    rig.ctx.profile_enable(2)
    rig.time_prune(2)
    rig.ctx.profile_read()
    rig.time_prune(reps)
    pr = rig.ctx.profile_read()
    rig.ctx.profile_enable(0)
    return {k: round(1e3 * ms / n, 2) for k, (ms, n) in pr["slots"].items()}


def run_next(rig, hbm_peak):
    """The widened rows of SURVEY section 8(f), measured on the headline workload (configs[1]) through the C-ABI: NEXT-1
    multi-row scorer (R = 4, 32), NEXT-3 baseline scorers, NEXT-2 one chunk of prefill attention through the pruned slot
    map with its KV-read counters.  Each entry carries its own roofline: the time the algorithmic bytes (or flops) would
    take at the measured peaks."""
    torch, ikv = rig.torch, rig.ikv
    ctx, st, dev, shape, T = rig.ctx, rig.stream, rig.dev, rig.shape, rig.T
    L, Hq, Hkv, D = shape.L, shape.Hq, shape.Hkv, shape.D
    key_bytes = L * Hkv * T * D * shape.elem_bytes
    hbm_ms = key_bytes / (hbm_peak * 1e9) * 1e3
    tensor_peak = 1679.3e12
    mp = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(mp):
        tensor_peak = float(json.load(open(mp)).get("bf16_tflops", 1679.3)) * 1e12

    def timed(fn, n=3):
        ts = []
        for i in range(n + 1):
            with torch.cuda.stream(st):
                a, b = rig.ev(), rig.ev()
                a.record(st); fn(); b.record(st)
            st.synchronize()
            ts.append(a.elapsed_time(b))
        return statistics.median(ts[1:])

    with torch.cuda.stream(st):
        rig.S_dev.copy_(rig.pristine)
    st.synchronize()
    res = {"workload": "configs[1], un-pruned 32k-token map for the scorers; pruned map (C = 8k) for the prefill chunk"}
    gen = torch.Generator(device="cpu").manual_seed(4242)
    for R in (4, 32):
        rows = torch.randn((R, L, Hq, D), generator=gen).to(dev).contiguous()
        wts = [1.0 / R] * R
        ms = timed(lambda: ctx.score_rows([rig.req], rows, wts, rig.scores, st))
        # the bank is a bf16 hi + lo pair: two tensor passes per product; the keys are read twice (statistics, sums)
        flop_ms = 2 * 2 * 2.0 * R * L * Hq * T * D / tensor_peak * 1e3
        tc = R >= 4
        roof = max(hbm_ms, flop_ms)
        res[f"multirow_R{R}"] = {"ms": ms, "roofline_ms": roof, "frac_of_roofline": roof / ms,
                                 "bound": "hbm" if hbm_ms >= flop_ms else "tensor",
                                 "passes_over_the_keys": 2 if tc else R,
                                 "what": ("ikv_score_rows on tcgen05: one bank of 128 bank rows, two sweeps over the keys (TMA gather4)"
                                          if tc else "ikv_score_rows: R passes of the single-row key pass (below 4 rows)")}
    rows32 = torch.randn((32, L, Hq, D), generator=gen).to(dev).contiguous()
    res["baseline_streaming"] = {"ms": timed(lambda: ctx.score_baseline([rig.req], ikv.BASE_STREAMING, rig.scores, n_sink=4,
                                                                        stream=st)),
                                 "what": "sink 4 + recency scores: no keys are read"}
    for name, kind, kw in (("baseline_snapkv", ikv.BASE_SNAPKV, {"pool_kernel": 7}),
                           ("baseline_h2o", ikv.BASE_H2O, {"recent_ratio": 0.5, "recent_floor": 64})):
        ms = timed(lambda: ctx.score_baseline([rig.req], kind, rig.scores, rows=rows32, stream=st, **kw), n=2)
        res[name] = {"ms": ms, "roofline_ms": hbm_ms, "frac_of_roofline": hbm_ms / ms,
                     "what": "window of 32 query rows through the tcgen05 multi-row scorer + pooling / recency rule"}
    # NEXT-2: prune, then one chunk of 64 prefill rows at layer 0 through the pruned map
    with torch.cuda.stream(st):
        rig.prune()
    st.synchronize()
    n_kept = int(rig.nk.item())
    for n_q in (64, 2048):
        q = torch.randn((n_q, Hq, D), generator=gen).to(torch.bfloat16).to(dev)
        out = torch.empty_like(q)
        reads = torch.zeros(2, dtype=torch.int64, device=dev)
        S_map = rig.S_dev
        if T + n_q > S_map.numel():   # the workload's map ends 256 positions after T: the new positions reuse live slots
            head_map = rig.S_dev[:T]
            S_map = torch.cat([head_map, head_map[head_map != rig.w.dead_slot][:n_q]]).contiguous()
        r = ikv.make_request(rig.sid, S_map, T + n_q, rig.sess.pi, rig.sess.qs, rig.sess.qe, rig.C, rig.sess.pi)
        n_rep = 4
        ms = timed(lambda: ctx.prefill_attn(0, r, T, q, out, rig.scale, reads, st), n=n_rep - 1)
        raw, eff = [int(x) // n_rep for x in reads.cpu().tolist()]
        kv_bytes = (n_kept + n_q) * Hkv * D * 2 * shape.elem_bytes      # the survivors' K and V rows, read once per chunk
        flops = 2 * 2.0 * Hq * D * eff                                  # QK^T and PV over the (row, visible item) pairs
        hbm_t, mma_t = kv_bytes / (hbm_peak * 1e9) * 1e3, flops / tensor_peak * 1e3
        roof = max(hbm_t, mma_t)
        res[f"prefill_chunk_{n_q}"] = {"n_q": n_q, "layer_calls": 1, "live_tokens": n_kept, "ms": ms, "roofline_ms": roof,
                                       "bound": "hbm" if hbm_t >= mma_t else "tensor",
                                       "frac_of_roofline": roof / ms, "raw_kv_reads": raw, "effective_kv_reads": eff,
                                       "what": "ikv_prefill_attn on tcgen05 (k_prefill_tc): K/V tiles by TMA gather4 into swizzled "
                                               "operands; 128 / G query rows x G heads per M tile, two M tiles per CTA from "
                                               "eight tiles of rows on; counters per PAPER.md:163-175"}
    return res


def run_cfg2(args, dev, hbm_peak):
    """configs[2] (Qwen2.5-14B shape, 92,160 live tokens, M=256, C=8192) as a sub-object: prune pass, key pass, decode."""
    import torch
    from paper_2606_09916_b200 import workloads as wl
    shape = wl.QWEN25_14B
    T, C, DEC = 92160, 8192, 32
    w = wl.cfg2(device="cuda", n_tokens=T, budget=C, decode_tokens=DEC)
    rig = Rig(w, shape, T, C, DEC, "learnable", dev, args.tune)
    rig.time_prune(3)
    rig.ctx.profile_enable(1)
    ts = rig.time_prune(10)
    pr = rig.ctx.profile_read()
    rig.ctx.profile_enable(0)
    prune_ms = statistics.median(ts)
    key_ms = pr["score_logits_ms"] / max(1, pr["score_logits_n"])
    key_bytes = shape.L * shape.Hkv * T * shape.D * shape.elem_bytes
    n_kept = int(rig.nk.item())
    dq = wl.decode_queries(shape, DEC, w.seed, device="cuda")
    dout = torch.empty((DEC, shape.L, 1, shape.Hq, shape.D), dtype=torch.bfloat16, device=dev)
    g = rig.capture_decode(DEC, dq, dout, dependent=False)
    tt = []
    for _ in range(4):
        with torch.cuda.stream(rig.stream):
            a, b = rig.ev(), rig.ev()
            a.record(rig.stream); g.replay(); b.record(rig.stream)
        rig.stream.synchronize()
        tt.append(a.elapsed_time(b))
    dec_ms = statistics.median(tt[1:]) / DEC
    dec_bytes = sum(n_kept + t + 1 for t in range(DEC)) / DEC * shape.L * shape.Hkv * shape.D * 2 * shape.elem_bytes
    out = {"workload": "configs[2] Qwen2.5-14B-shaped single session: 48 layers, 40 Q / 8 KV heads (G = 5), head_dim 128, "
                       "92,160 live tokens, M=256, C=8192", "mode": "learnable", "prune_ms": prune_ms,
           "tokens_per_s": T / (prune_ms * 1e-3), "key_pass_ms": key_ms, "key_pass_gbs": key_bytes / (key_ms * 1e-3) / 1e9,
           "key_pass_frac_of_measured_peak": key_bytes / (key_ms * 1e-3) / 1e9 / hbm_peak,
           # 92k tokens exceed the on-chip capacity of the layer-major kernel: k_key_pass also writes L*Hq*T fp32 logits
           "key_pass_traffic_frac_of_measured_peak": (key_bytes + shape.L * shape.Hq * T * 4) / (key_ms * 1e-3) / 1e9 / hbm_peak,
           "prune_frac_of_measured_peak": key_bytes / (prune_ms * 1e-3) / 1e9 / hbm_peak, "n_kept": n_kept,
           "decode_ms_per_step": dec_ms, "decode_kv_gbs": dec_bytes / (dec_ms * 1e-3) / 1e9,
           "decode_frac_of_measured_peak": dec_bytes / (dec_ms * 1e-3) / 1e9 / hbm_peak,
           "prune_breakdown_us": prune_breakdown(rig, 5)}
    del rig, w, g
    torch.cuda.empty_cache()
    return out


def run_cfg4(args, dev, hbm_peak):
    """configs[4] (64 concurrent sessions, lognormal lengths, budgets {4096, 8192, 16384}) as a sub-object, on L_res = 24
    resident layers (all 36 layers of K+V of 1.12 M tokens are 165 GB: they do not fit beside anything else).  Batched
    score / select / evict, then batched decode, all through the C-ABI with n_req = 64."""
    import torch
    from paper_2606_09916_b200 import ikv, workloads as wl
    L_RES = 24      # K+V of 1.12 M tokens: 4.6 GB per layer; 24 layers = 110 GB of the 180 GB
    shape = wl.ModelShape(L_RES, 32, 8, 128)
    w = wl.batched(device="cuda", shape=shape, decode_tokens=1)
    ctx = ikv.Context(shape.L, shape.Hq, shape.Hkv, shape.D, w.k_pool, w.v_pool, dead_slot=w.dead_slot)
    ctx.residual_load(wl.residual_weights(shape.D, w.seed + 5))
    tot = sum(s.N for s in w.sessions)
    ctx.reserve(max(s.N for s in w.sessions) + 1, len(w.sessions))
    stream = torch.cuda.Stream(device=dev)
    maps0 = [s.slot_map.to(dev) for s in w.sessions]
    maps = [m.clone() for m in maps0]
    reqs = []
    for s, m in zip(w.sessions, maps):
        ctx.session_open(s.spec.session_id)
        for u in s.updates():
            ctx.memory_update(s.spec.session_id, u.to(dev).contiguous())
        reqs.append(ikv.make_request(s.spec.session_id, m, s.N, s.pi, s.qs, s.qe, s.spec.budget, s.pi))
    scores = torch.empty(tot, device=dev)
    freed = torch.empty(tot, dtype=torch.int32, device=dev)
    nf = torch.zeros(len(reqs), dtype=torch.int32, device=dev)
    nk = torch.zeros(len(reqs), dtype=torch.int32, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    ts = []
    for it in range(4):
        with torch.cuda.stream(stream):
            for m, m0 in zip(maps, maps0):
                m.copy_(m0)
            a, b = ev(), ev()
            a.record(stream)
            ctx.score(reqs, ikv.MODE_LEARNABLE, scores, None, stream)
            ctx.select_evict(reqs, scores, freed, nf, nk, stream)
            b.record(stream)
        stream.synchronize()
        ts.append(a.elapsed_time(b))
    prune_ms = statistics.median(ts[1:])
    kept = int(nk.sum().item())
    key_bytes = shape.L * shape.Hkv * tot * shape.D * 2
    # batched decode: one step, every resident layer, 64 requests per call (chunks of 32 inside the library)
    q = torch.randn((shape.L, len(reqs), shape.Hq, shape.D), device=dev).to(torch.bfloat16)
    out = torch.empty_like(q)
    dreqs = [ikv.make_request(s.spec.session_id, m, s.N + 1, s.pi, s.qs, s.qe, s.spec.budget, s.pi,
                              flags=ikv.REQ_INPUTS_COMPLETE) for s, m in zip(w.sessions, maps)]
    scale = 1.0 / math.sqrt(shape.D)
    with torch.cuda.stream(stream):
        for l in range(shape.L):
            ctx.decode_attn(l, dreqs, q[l], out[l], scale, stream)
    stream.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=stream):
        for rep in range(4):
            for l in range(shape.L):
                ctx.decode_attn(l, dreqs, q[l], out[l], scale, stream)
    tt = []
    for _ in range(4):
        with torch.cuda.stream(stream):
            a, b = ev(), ev()
            a.record(stream); g.replay(); b.record(stream)
        stream.synchronize()
        tt.append(a.elapsed_time(b))
    dec_ms = statistics.median(tt[1:]) / 4
    dec_bytes = (kept + len(reqs)) * shape.L * shape.Hkv * shape.D * 2 * 2
    res = {"workload": "configs[4] 64 concurrent Qwen3-8B-shaped sessions in one pool, lognormal live lengths (median 16k, "
                       "4k-64k), budgets {4096, 8192, 16384}, learnable scorer",
           "resident_layers": L_RES, "sessions": len(reqs), "tokens": tot, "kept": kept,
           "prune_ms_resident_layers": prune_ms, "tokens_per_s_resident_layers": tot / (prune_ms * 1e-3),
           "prune_gbs": key_bytes / (prune_ms * 1e-3) / 1e9,
           "prune_frac_of_measured_peak": key_bytes / (prune_ms * 1e-3) / 1e9 / hbm_peak,
           "decode_ms_per_step_resident_layers": dec_ms, "decode_kv_gbs": dec_bytes / (dec_ms * 1e-3) / 1e9,
           "decode_frac_of_measured_peak": dec_bytes / (dec_ms * 1e-3) / 1e9 / hbm_peak}
    del ctx, w, g
    torch.cuda.empty_cache()
    return res


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_09916_b200 import ikv, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    hbm_peak, peak_src = peaks()

    T, C, DEC = args.tokens, args.budget, args.decode_steps
    shape = wl.QWEN3_8B
    w = wl.cfg1(device="cuda", seed=1000 + rank, n_tokens=T, budget=C, decode_tokens=DEC)
    rig = Rig(w, shape, T, C, DEC, args.mode, dev, args.tune)
    sess, ctx, stream = rig.sess, rig.ctx, rig.stream
    L, Hq, Hkv, D = shape.L, shape.Hq, shape.Hkv, shape.D
    dq = wl.decode_queries(shape, DEC, w.seed, device="cuda")
    dout = torch.empty((DEC, L, 1, Hq, D), dtype=torch.bfloat16, device=dev)

    # un-captured warm-up pass (sizes every lazily grown buffer), then capture the decode loop in a graph
    with torch.cuda.stream(stream):
        rig.S_dev.copy_(rig.pristine)
        rig.prune()
        r0 = ikv.make_request(rig.sid, rig.S_dev, T + 1, sess.pi, sess.qs, sess.qe, C, sess.pi)
        ctx.decode_attn(0, [r0], dq[0, 0:1], dout[0, 0], rig.scale, stream)
    stream.synchronize()
    graph = rig.capture_decode(DEC, dq, dout, dependent=False)

    def one_step(record):
        with torch.cuda.stream(stream):
            rig.S_dev.copy_(rig.pristine)       # untimed restore of the slot map (a new turn's map)
            e0, e1, e2 = rig.ev(), rig.ev(), rig.ev()
            e0.record(stream)
            rig.prune()
            e1.record(stream)
            graph.replay()
            e2.record(stream)
        if record is not None:
            record.append((e0, e1, e2))

    for _ in range(args.warmup):
        one_step(None)
    stream.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ctx.profile_enable(1)                        # CUDA events around the dominant kernels, inside the timed region
    recs = []
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        one_step(recs)
    stream.synchronize()
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    prof = ctx.profile_read()
    ctx.profile_enable(0)
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    prune_ms = [a.elapsed_time(b) for a, b, _ in recs]
    dec_ms = [b.elapsed_time(c) for _, b, c in recs]
    step_ms = [a.elapsed_time(c) for a, _, c in recs]
    tot_prune, tot_dec, tot_step = sum(prune_ms), sum(dec_ms), sum(step_ms)
    n_kept = int(rig.nk.item())

    # ---- end-to-end through ikv_prune_host with pinned HOST buffers
    h_map0 = sess.slot_map[:T].clone().pin_memory()
    h_map = torch.empty_like(h_map0).pin_memory()
    h_rows = sess.updates()[-1].to(torch.bfloat16).contiguous().pin_memory()   # post-RoPE Q rows in the model's dtype
    h_valid = torch.empty(T, dtype=torch.uint8).pin_memory()
    h_freed = torch.empty(T, dtype=torch.int32).pin_memory()
    req_h = ikv.make_request(rig.sid, None, T, sess.pi, sess.qs, sess.qe, C, sess.pi)
    e2e_t = []
    n_e2e = max(args.steps, 20)     # a call takes well under a millisecond of wall clock: at least 20 of them, mean
    for i in range(args.warmup + n_e2e):
        h_map.copy_(h_map0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.prune_host(req_h, h_rows, rig.mode, h_map, h_valid, None, h_freed, stream)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            e2e_t.append(dt)
    e2e_total = sum(e2e_t) * args.steps / n_e2e     # scaled to the K steps of the device-timed region
    h2d = T * 4 + h_rows.numel() * h_rows.element_size()
    d2h = 16 + ((T + 1023) // 1024 * 1024) * 8 + T     # one copy: counts | slot map | freed list (capacity) | valid mask

    # ---- beside the headline: the pass without the events of the key-pass profile, phase 1 (memory mode), the breakdown
    plain_ms = statistics.median(rig.time_prune(3 + 10)[3:])
    p1_ms = statistics.median(rig.time_prune(3 + 5, ikv.MODE_MEMORY)[3:])
    breakdown = prune_breakdown(rig)

    # ---- decode: the dependent chain (q of every call = output of the previous call) and one call in isolation
    CH = min(DEC, 32)
    with torch.cuda.stream(stream):
        rig.S_dev.copy_(rig.pristine)
        rig.prune()
    stream.synchronize()
    chain = rig.capture_decode(CH, dq, dout, dependent=True)
    tt = []
    for _ in range(5):
        with torch.cuda.stream(stream):
            a, b = rig.ev(), rig.ev()
            a.record(stream); chain.replay(); b.record(stream)
        stream.synchronize()
        tt.append(a.elapsed_time(b))
    chain_ms = statistics.median(tt[1:]) / CH
    ctx.profile_enable(2)
    r_iso = ikv.make_request(rig.sid, rig.S_dev, T + 1, sess.pi, sess.qs, sess.qe, C, sess.pi)
    for i in range(3 + 36):
        if i == 3:
            ctx.profile_read()
        with torch.cuda.stream(stream):
            ctx.decode_attn(i % L, [r_iso], dq[0, i % L:i % L + 1], dout[0, i % L], rig.scale, stream)
        stream.synchronize()                  # every call alone on the device
    iso = ctx.profile_read()["slots"]
    ctx.profile_enable(0)
    iso_us = sum(1e3 * ms / n for k, (ms, n) in iso.items() if k.startswith("decode"))

    # ---- max over ranks
    tot_prune, tot_dec, tot_step, e2e_ms_total = max_over_ranks([tot_prune, tot_dec, tot_step, e2e_total * 1e3], world, dev)

    if rank == 0:
        K = args.steps
        default_wl = (T == 32768 and C == 8192 and args.mode == "learnable")  # the ncu capture's workload
        key_bytes = L * Hkv * T * D * shape.elem_bytes                 # algorithmic bytes of the key pass
        dec_tokens_sum = sum(n_kept + t + 1 for t in range(DEC))        # live tokens read over the decode loop
        dec_bytes_step = dec_tokens_sum * L * Hkv * D * 2 * shape.elem_bytes
        value = whole_job_value(T, world, K, tot_prune)
        key_ms = prof["score_logits_ms"] / max(1, prof["score_logits_n"])
        ach = key_bytes / (key_ms * 1e-3) / 1e9 if key_ms > 0 else 0.0
        dec_kernel_ms = tot_dec / K / (DEC * L)                         # split + merge + launch gap per layer call
        dec_bytes_call = dec_bytes_step / (DEC * L)
        dec_ach = dec_bytes_call / (dec_kernel_ms * 1e-3) / 1e9
        n_prune_launch = len(breakdown)                                 # kernels of one prune pass (library's own count)
        n_decode_launch = DEC * L * 2
        tr_key, tr_src = ncu_traffic("k_key_pass") if default_wl else (None, None)
        tr_dec, _ = ncu_traffic("k_decode_mma") if default_wl else (None, None)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": tot_step / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16 keys/values, f32 accumulate", "data": "synthetic",
            "config": {"workload": CFG1_TEXT, "n_tokens": T, "budget": C, "decode_steps": DEC, "mode": args.mode,
                       "n_kept": n_kept,
                       "l2": "inputs larger than L2 (2.4 GB of keys per prune, 1.2 GB of K/V per decode step; 126 MB L2)",
                       "parallelism": f"replicas x{world}" if world > 1 else "single GPU"},
            "prune_ms": tot_prune / K, "prune_ms_without_profile_events": plain_ms, "prune_ms_memory_mode": p1_ms,
            "prune_hbm_gbs": key_bytes / (tot_prune / K * 1e-3) / 1e9,
            "prune_frac_of_measured_peak": key_bytes / (tot_prune / K * 1e-3) / 1e9 / hbm_peak,
            "prune_frac_of_nominal_8TBs": key_bytes / (tot_prune / K * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "prune_breakdown_us": breakdown,
            "decode": {"ms_per_decode_step": tot_dec / K / DEC, "kv_gbs": dec_bytes_step / (tot_dec / K * 1e-3) / 1e9,
                       "tokens_per_s": world * DEC * K / (tot_dec * 1e-3),
                       "frac_of_nominal_8TBs": dec_bytes_step / (tot_dec / K * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
                       "what": "graph of 256 steps x 36 layer calls with precomputed queries (IKV_REQ_INPUTS_COMPLETE): "
                               "consecutive calls overlap",
                       "dependent_chain_ms": chain_ms,
                       "dependent_chain_frac_of_measured_peak": dec_bytes_call * L / (chain_ms * 1e-3) / 1e9 / hbm_peak,
                       "dependent_chain_what": f"graph of {CH} steps x 36 calls, the query of every call copied from the "
                                               "previous call's output, default request flags",
                       "isolated_call_us": iso_us,
                       "isolated_call_frac_of_measured_peak": dec_bytes_call / (iso_us * 1e-6) / 1e9 / hbm_peak},
            "e2e": {"value": world * T * K / (e2e_ms_total * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h,
                    "what": "ikv_prune_host: slot map + bf16 query rows H2D, memory update + score + select/evict, "
                            "slot map + valid mask + freed list + counts D2H; the K/V pool is device-resident state; "
                            "wall clock around each call, mean of max(steps, 20) calls"},
            "gpu_launches": K * (n_prune_launch + n_decode_launch),
            "roofline": {"kernel": "k_key_pass_lm (layer-major key pass: logits, rule sums, mean keys)", "bound": "hbm",
                         "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                         "frac_of_nominal_8TBs": ach / NOMINAL_HBM_GBS, "peak_source": peak_src,
                         "traffic": tr_key, "traffic_source": tr_src, "algorithmic_bytes": key_bytes, "ms": key_ms},
            "roofline_decode": {"kernel": "k_decode_mma (+k_decode_merge4, per-layer launch gap included)",
                                "bound": "hbm", "achieved": dec_ach, "peak": hbm_peak, "unit": "GB/s",
                                "frac": dec_ach / hbm_peak, "frac_of_nominal_8TBs": dec_ach / NOMINAL_HBM_GBS,
                                "algorithmic_bytes": dec_bytes_call, "traffic": tr_dec, "traffic_source": tr_src,
                                "ms": dec_kernel_ms},
            "clocks": clocks, "wall_s_timed_region": t_wall,
        }
        if not args.no_extra and world == 1:
            try:
                line["next"] = run_next(rig, hbm_peak)
            except Exception as e:  # a sub-object must not take the headline down
                line["next"] = {"error": repr(e)}
        del rig, graph, chain, w
        torch.cuda.empty_cache()
        if not args.no_extra and world == 1:
            try:
                line["cfg2"] = run_cfg2(args, dev, hbm_peak)
            except Exception as e:  # a sub-object must not take the headline down
                line["cfg2"] = {"error": repr(e)}
            try:
                line["cfg4"] = run_cfg4(args, dev, hbm_peak)
            except Exception as e:
                line["cfg4"] = {"error": repr(e)}
        if not args.no_cpu_baseline:
            wc, kp_host, wts = oracle_workload(T, C)
            oracle_pass(wc, wc.sessions[0], kp_host, wts)          # first touch of the pool
            ts, tsec = [], 0.0
            while len(ts) < 10 and tsec < 15.0:                     # ~15 s of oracle time, bounded
                ts.append(oracle_pass(wc, wc.sessions[0], kp_host, wts)); tsec += ts[-1]
            line["cpu_baseline"] = {
                "value": T / (sum(ts) / len(ts)), "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                "sample": f"oracle pruning pass (learnable mode) on all {T} tokens and all {L} layers, "
                          f"{len(ts)} passes (mean) after one warm-up pass",
                "sample_seconds": tsec}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="learnable", choices=["learnable", "memory"])
    ap.add_argument("--tokens", type=int, default=32768)
    ap.add_argument("--budget", type=int, default=8192)
    ap.add_argument("--decode-steps", type=int, default=256)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the cfg2 / cfg4 sub-objects")
    ap.add_argument("--tune", action="append", default=[], help="ikv_tune knob=value (A/B experiments)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
