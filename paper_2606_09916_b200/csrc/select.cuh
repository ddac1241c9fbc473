// select.cuh -- budgeted top-k (Eq. 1) and slot-map eviction with prefix-safe
// free (Eq. 7).  One CTA of 1024 threads per request.
#pragma once
#include <limits.h>
#include "common.cuh"

namespace ikv {

// Order-preserving map fp32 -> uint32 (larger score -> larger key); -0 == +0; NaN below everything (R13).
__device__ __forceinline__ uint32_t score_key(float s) {
  if (s != s) return 0u;
  if (s == 0.f) s = 0.f;  // folds -0.0 onto +0.0
  const uint32_t u = __float_as_uint(s);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

struct SelParams {
  int32_t* S;            // slot map, in place
  uint8_t* valid;        // optional
  const float* scores;   // [N] by position
  int N, pi, qs, qe, C, radix;
  int32_t dead;
  int32_t* freed;        // [N] capacity
  int32_t* n_freed;      // scalar
  int32_t* n_kept;       // scalar
  int32_t* live_slots;   // compact survivor list for decode, capacity N
  int32_t* n_live;       // scalar
  // scratch
  uint32_t* kept_bits;   // n_slots bits, all zero on entry and on exit
  int32_t* firstpos;     // n_slots ints, all INT_MAX on entry and on exit
  uint8_t* keepflag;     // [N]
  int32_t* tmp_slot;     // [N]
};

__global__ __launch_bounds__(1024) void k_select_evict(SelParams p) {
  __shared__ int hist[256];
  __shared__ int warp_tot[32];
  __shared__ int sh_cnt[2];
  __shared__ uint32_t sh_prefix;
  __shared__ int sh_remaining;
  const int tid = threadIdx.x, lane = tid & 31;
  const int N = p.N;

  // ---- phase A: |F| and |A| over the live set
  if (tid < 2) sh_cnt[tid] = 0;
  __syncthreads();
  {
    int nf = 0, nc = 0;
    for (int j = tid; j < N; j += 1024) {
      const int cls = classify(p.S[j], j, p.dead, p.pi, p.qs, p.qe);
      nf += (cls == CLS_FORCED);
      nc += (cls == CLS_CAND);
    }
    nf = warp_sum_i(nf);
    nc = warp_sum_i(nc);
    if (lane == 0) { atomicAdd(&sh_cnt[0], nf); atomicAdd(&sh_cnt[1], nc); }
  }
  __syncthreads();
  const int nF = sh_cnt[0], nC = sh_cnt[1];
  // skip rule (R15): N <= C keeps every live position
  int cstar = (N <= p.C) ? nC : max(0, p.C - nF);  // R14
  cstar = min(cstar, nC);
  const bool keep_all = (cstar == nC), keep_none = (cstar == 0);

  // ---- phase B: radix select of the cstar-th largest key, 4 passes of 8 bits, MSB first
  uint32_t thr = 0;
  int need_eq = 0;
  if (!keep_all && !keep_none) {
    if (tid == 0) { sh_prefix = 0u; sh_remaining = cstar; }
    for (int pass = 3; pass >= 0; --pass) {
      const int shift = pass * 8;
      const uint32_t mask = (pass == 3) ? 0u : (0xffffffffu << (shift + 8));
      if (tid < 256) hist[tid] = 0;
      __syncthreads();
      const uint32_t prefix = sh_prefix;
      for (int j0 = 0; j0 < N; j0 += 1024) {
        const int j = j0 + tid;
        bool on = false;
        uint32_t digit = 0;
        if (j < N && classify(p.S[j], j, p.dead, p.pi, p.qs, p.qe) == CLS_CAND) {
          const uint32_t key = score_key(p.scores[j]);
          if ((key & mask) == prefix) { on = true; digit = (key >> shift) & 255u; }
        }
        // warp-aggregated histogram: one atomic per distinct digit per warp
        const uint32_t act = __ballot_sync(0xffffffffu, on);
        if (on) {
          const uint32_t peers = __match_any_sync(act, digit);
          if (lane == (__ffs(peers) - 1)) atomicAdd(&hist[digit], __popc(peers));
        }
      }
      __syncthreads();
      if (tid == 0) {
        int remaining = sh_remaining, cum = 0, d = 255;
        for (; d > 0; --d) {
          if (cum + hist[d] >= remaining) break;
          cum += hist[d];
        }
        sh_remaining = remaining - cum;
        sh_prefix = prefix | ((uint32_t)d << shift);
      }
      __syncthreads();
    }
    thr = sh_prefix;
    need_eq = sh_remaining;  // how many keys equal to thr survive (lowest positions first)
  }

  // ---- sweep 1 (position order): keep flags, kept-slot bitmap, first dropped position per slot
  int eq_base = 0;
  for (int j0 = 0; j0 < N; j0 += 1024) {
    const int j = j0 + tid;
    int cls = CLS_DEAD, slot = p.dead;
    uint32_t key = 0;
    if (j < N) {
      slot = p.S[j];
      cls = classify(slot, j, p.dead, p.pi, p.qs, p.qe);
      if (cls == CLS_CAND) key = score_key(p.scores[j]);
    }
    const int is_eq = (cls == CLS_CAND && !keep_all && !keep_none && key == thr) ? 1 : 0;
    int tot;
    const int ex = block_excl_scan_1024(is_eq, warp_tot, &tot);
    bool keep = false;
    if (cls == CLS_FORCED) keep = true;
    else if (cls == CLS_CAND) keep = keep_all || (!keep_none && (key > thr || (is_eq && eq_base + ex < need_eq)));
    eq_base += tot;
    if (j < N) {
      p.keepflag[j] = keep ? 1 : 0;
      if (keep) atomicOr(&p.kept_bits[slot >> 5], 1u << (slot & 31));
      else if (cls != CLS_DEAD && j >= p.radix) atomicMin(&p.firstpos[slot], j);
    }
  }
  __threadfence();
  __syncthreads();

  // ---- sweep 2 (position order): rewrite S, valid mask, live list, freed list (R21, R22)
  int live_base = 0, freed_base = 0;
  for (int j0 = 0; j0 < N; j0 += 1024) {
    const int j = j0 + tid;
    int keep = 0, is_freed = 0, slot = p.dead;
    if (j < N) {
      keep = p.keepflag[j];
      slot = p.S[j];
      int dropped_slot = -1;
      if (!keep && slot != p.dead) {  // newly dropped
        dropped_slot = slot;
        p.S[j] = p.dead;
        if (j >= p.radix) {
          const uint32_t bits = __ldcg(&p.kept_bits[slot >> 5]);
          const int fp = __ldcg(&p.firstpos[slot]);
          is_freed = (!((bits >> (slot & 31)) & 1u) && fp == j) ? 1 : 0;
        }
      }
      p.tmp_slot[j] = dropped_slot;
      if (p.valid) p.valid[j] = keep ? 1 : 0;
    }
    int tot;
    const int ex = block_excl_scan_1024(keep | (is_freed << 16), warp_tot, &tot);
    if (keep) p.live_slots[live_base + (ex & 0xffff)] = slot;
    if (is_freed) p.freed[freed_base + (ex >> 16)] = slot;
    live_base += tot & 0xffff;
    freed_base += tot >> 16;
  }
  __syncthreads();

  // ---- sweep 3: restore the scratch invariants
  for (int j = tid; j < N; j += 1024) {
    if (p.keepflag[j]) {
      const int slot = p.S[j];
      p.kept_bits[slot >> 5] = 0u;
    } else {
      const int ds = p.tmp_slot[j];
      if (ds >= 0) p.firstpos[ds] = INT_MAX;
    }
  }
  for (int i = live_base + tid; i < N; i += 1024) p.live_slots[i] = p.dead;  // padded for decode (host-side bound)
  if (tid == 0) {
    *p.n_kept = live_base;
    *p.n_freed = freed_base;
    *p.n_live = live_base;
  }
}

// Compact survivor list straight from a slot map (used when no ikv_select_evict preceded the decode).
__global__ __launch_bounds__(1024) void k_build_live(const int32_t* __restrict__ S, int N, int32_t dead,
                                                     int32_t* __restrict__ live_slots, int32_t* __restrict__ n_live) {
  __shared__ int warp_tot[32];
  int base = 0;
  for (int j0 = 0; j0 < N; j0 += 1024) {
    const int j = j0 + threadIdx.x;
    const int slot = (j < N) ? S[j] : dead;
    int tot;
    const int ex = block_excl_scan_1024(slot != dead ? 1 : 0, warp_tot, &tot);
    if (slot != dead) live_slots[base + ex] = slot;
    base += tot;
  }
  for (int i = base + threadIdx.x; i < N; i += 1024) live_slots[i] = dead;  // padded for decode (host-side bound)
  if (threadIdx.x == 0) *n_live = base;
}

}  // namespace ikv
