// select_cluster.cuh -- a1 / a6 / a7 as thread-block-cluster kernels (sm_100a): partition,
// budgeted top-k (Eq. 1) and slot-map eviction with prefix-safe free (Eq. 7, PAPER.md:121-132,
// 491-493).  One cluster of CL_CTAS CTAs x 1024 threads per request; every thread keeps MAXI consecutive positions in
// registers (blocked layout, so order-preserving compaction is one block scan plus a rank offset exchanged through
// distributed shared memory).  Requests longer than CL_CTAS * 1024 * 16 positions take the single-CTA kernels of
// select.cuh / score.cuh.  Semantics are identical to k_select_evict / k_partition (R13-R15, R21, R22).
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
#include "pipe.cuh"
#include "select.cuh"

namespace ikv {

namespace cg = cooperative_groups;

constexpr int CL_CTAS = 8;
constexpr int CL_MAX_ITEMS = 16;
constexpr int CL_MAX_N = CL_CTAS * 1024 * CL_MAX_ITEMS;
constexpr int SEL_MAX_REQ = 16;  // requests per launch of k_select_evict_cl (parameters travel by value)
struct SelBatch {
  SelParams p[SEL_MAX_REQ];
};

// Lifetime barrier of distributed shared memory: a CTA may not exit while another rank can still read its shared memory.
// It orders no memory (arrive.relaxed: no fence over the output writes still in flight) and is split, so that the global
// writes between arrive and wait overlap the other ranks' last remote reads.
// `dep` = a value computed from this rank's last remote loads: the arrive cannot issue before they have returned.
__device__ __forceinline__ void cluster_arrive_relaxed(int dep) {
  asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::"r"(dep) : "memory");
}
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.aligned;" ::: "memory"); }

// sum over the cluster of one int per CTA, and the exclusive prefix of this CTA's rank
__device__ __forceinline__ void cluster_offsets(cg::cluster_group& cl, int* sh_val, int crank, int* before, int* total) {
  int b = 0, t = 0;
#pragma unroll
  for (int rk = 0; rk < CL_CTAS; ++rk) {
    const int v = *cl.map_shared_rank(sh_val, rk);
    if (rk < crank) b += v;
    t += v;
  }
  *before = b;
  *total = t;
}

// ---------------------------------------------------------------------------------------------------------------
// a1 partition: score fillers (R6), zeroed rule_out, candidates compacted in ascending position.
// ---------------------------------------------------------------------------------------------------------------
template <int MAXI>
__global__ __cluster_dims__(CL_CTAS, 1, 1) __launch_bounds__(1024) void k_partition_cl(
    const int32_t* __restrict__ S, int N, int32_t dead, int pi, int qs, int qe, float* __restrict__ scores,
    float* __restrict__ rule_out, int32_t* __restrict__ cand_pos, int32_t* __restrict__ cand_slot,
    int32_t* __restrict__ n_cand, const int32_t* __restrict__ xattn_pos, int n_x, int32_t* __restrict__ xq_slot,
    int32_t* __restrict__ n_xq) {
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  cg::cluster_group cl = cg::this_cluster();
  const int crank = (int)cl.block_rank();
  __shared__ int warp_tot[32];
  __shared__ int sh_tot;
  const int tid = threadIdx.x;
  if (blockIdx.x >= CL_CTAS) {
    // second cluster (launched when n_x > 0): rank 0 compacts the live cross-attention positions
    if (crank != 0) return;
    int xb = 0;
    for (int i0 = 0; i0 < n_x; i0 += 1024) {
      const int i = i0 + tid;
      int sl = dead;
      if (i < n_x) {
        const int pos = xattn_pos ? xattn_pos[i] : qs + i;
        if (pos >= 0 && pos < N) sl = S[pos];
      }
      int tot;
      const int ex = block_excl_scan_1024(sl != dead ? 1 : 0, warp_tot, &tot);
      if (sl != dead) xq_slot[xb + ex] = sl;
      xb += tot;
    }
    if (tid == 0) *n_xq = xb;
    return;
  }
  const int base = (crank * 1024 + tid) * MAXI;
  int slot[MAXI];
  int cnt = 0;
  uint32_t cmask = 0;
  const bool vec = (MAXI % 4 == 0) && ((reinterpret_cast<uintptr_t>(S) & 15) == 0) && (base + MAXI <= N);
  if (vec) {
#pragma unroll
    for (int i = 0; i < MAXI; i += 4) {
      const int4 v = *reinterpret_cast<const int4*>(S + base + i);
      slot[i] = v.x; slot[i + 1] = v.y; slot[i + 2] = v.z; slot[i + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int i = 0; i < MAXI; ++i) slot[i] = (base + i < N) ? S[base + i] : dead;
  }
#pragma unroll
  for (int i = 0; i < MAXI; ++i) {
    const int j = base + i;
    if (j < N) {
      const int cls = classify(slot[i], j, dead, pi, qs, qe);
      if (cls == CLS_CAND) { cmask |= 1u << i; ++cnt; }
      else scores[j] = (cls == CLS_FORCED) ? CUDART_INF_F : -CUDART_INF_F;
      if (rule_out) rule_out[j] = 0.f;
    }
  }
  int tot;
  const int ex = block_excl_scan_1024(cnt, warp_tot, &tot);
  if (tid == 0) sh_tot = tot;
  cl.sync();
  int before, total;
  cluster_offsets(cl, &sh_tot, crank, &before, &total);
  int o = before + ex;
#pragma unroll
  for (int i = 0; i < MAXI; ++i)
    if ((cmask >> i) & 1u) {
      cand_pos[o] = base + i;
      cand_slot[o] = slot[i];
      ++o;
    }
  if (crank == 0 && tid == 0) *n_cand = total;
  cl.sync();  // keep sh_tot alive until every rank has read it
}

// ---------------------------------------------------------------------------------------------------------------
// a6 + a7 select and evict.  Phases (cluster barriers between them):
//   counts |F|, |A|  ->  4 x 8-bit radix-select passes (per-CTA histograms summed through DSMEM, every CTA resolves
//   the digit redundantly)  ->  rank of threshold ties in position order  ->  keep flags, kept-slot bitmap and
//   first-dropped-position table (global scratch)  ->  freed test (a)(b)(c)  ->  ordered writes  ->  scratch restore.
// ---------------------------------------------------------------------------------------------------------------
template <int MAXI>
__global__ __cluster_dims__(CL_CTAS, 1, 1) __launch_bounds__(1024) void k_select_evict_cl(const SelBatch batch) {
  // Never triggers its dependents early: the decode kernel that may follow reads the survivor list written here.  The
  // wait on the predecessor (the producer of the scores) comes after the prologue: the slot map is not modified between
  // ikv_score and ikv_select_evict of one event (ikv.h), so loading and classifying it overlaps the predecessor's tail.
  // one cluster per request of the batch.  Requests run concurrently on the shared kept-slot bitmap and
  // first-dropped-position table: they may share slots only below their radix_protected_len (forks, R19), where neither
  // structure is consulted, and every request clears exactly the bits it set.
  const SelParams p = batch.p[blockIdx.x / CL_CTAS];
  cg::cluster_group cl = cg::this_cluster();
  const int crank = (int)cl.block_rank();
  __shared__ int hist[2][256];
  __shared__ int comb[256];
  __shared__ int warp_tot[32];
  __shared__ int sh_cnt[2];   // |F|, |A| of this CTA
  __shared__ int sh_kf[2];    // kept, freed of this CTA
  __shared__ uint32_t sh_prefix;
  __shared__ int sh_remaining;
  const int tid = threadIdx.x, lane = tid & 31;
  const int N = p.N;
  const int base = (crank * 1024 + tid) * MAXI;

  int slot[MAXI];
  uint32_t key[MAXI];
  uint32_t cand_m = 0, forced_m = 0;  // bit i: item i is a candidate / forced
  const bool vec_s = (MAXI % 4 == 0) && (base + MAXI <= N) && ((reinterpret_cast<uintptr_t>(p.S) & 15) == 0);
  if (vec_s) {
#pragma unroll
    for (int i = 0; i < MAXI; i += 4) {
      const int4 v = *reinterpret_cast<const int4*>(p.S + base + i);
      slot[i] = v.x; slot[i + 1] = v.y; slot[i + 2] = v.z; slot[i + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int i = 0; i < MAXI; ++i) slot[i] = (base + i < N) ? p.S[base + i] : p.dead;
  }
#pragma unroll
  for (int i = 0; i < MAXI; ++i) {
    const int j = base + i;
    if (j < N) {
      const int cls = classify(slot[i], j, p.dead, p.pi, p.qs, p.qe);
      if (cls == CLS_CAND) cand_m |= 1u << i;
      else if (cls == CLS_FORCED) forced_m |= 1u << i;
    }
  }
  if (tid < 2) sh_cnt[tid] = 0;
  if (tid < 256) { hist[0][tid] = 0; hist[1][tid] = 0; }
  __syncthreads();
  {  // |F| and |A| of this CTA; summed over the cluster together with the first histogram
    const int nf = warp_sum_i(__popc(forced_m)), nc = warp_sum_i(__popc(cand_m));
    if (lane == 0) { atomicAdd(&sh_cnt[0], nf); atomicAdd(&sh_cnt[1], nc); }
  }
  pdl_wait();  // the scores are complete
  {
    const bool vec = (MAXI % 4 == 0) && (base + MAXI <= N) && ((reinterpret_cast<uintptr_t>(p.scores) & 15) == 0);
    float sc[MAXI];
    if (vec) {
#pragma unroll
      for (int i = 0; i < MAXI; i += 4) {
        const float4 f = *reinterpret_cast<const float4*>(p.scores + base + i);
        sc[i] = f.x; sc[i + 1] = f.y; sc[i + 2] = f.z; sc[i + 3] = f.w;
      }
    } else {
#pragma unroll
      for (int i = 0; i < MAXI; ++i) sc[i] = (base + i < N) ? p.scores[base + i] : 0.f;
    }
#pragma unroll
    for (int i = 0; i < MAXI; ++i) key[i] = ((cand_m >> i) & 1u) ? score_key(sc[i]) : 0u;
  }

  // ---- radix select of the cstar-th largest key, MSB first; the first pass does not depend on C*
  int nF = 0, nC = 0, cstar = 0;
  bool keep_all = false, keep_none = false;
  uint32_t thr = 0;
  int need_eq = 0;
  {
    uint32_t prefix = 0u;
    int remaining = 0;
    for (int pass = 3; pass >= 0; --pass) {
      const int shift = pass * 8;
      const uint32_t mask = (pass == 3) ? 0u : (0xffffffffu << (shift + 8));
      int* h = hist[pass & 1];
#pragma unroll
      for (int i = 0; i < MAXI; ++i) {
        const bool on = ((cand_m >> i) & 1u) && ((key[i] & mask) == prefix);
        const uint32_t digit = (key[i] >> shift) & 255u;
        // upper digits are almost always the same over a warp (scores share sign and exponent): one atomic per warp;
        // otherwise the digits are spread over the bins and plain shared-memory atomics do not collide much
        const uint32_t act = __ballot_sync(0xffffffffu, on);
        if (act) {
          const int first = __ffs(act) - 1;
          const uint32_t d0 = __shfl_sync(0xffffffffu, digit, first);
          if (__all_sync(0xffffffffu, !on || digit == d0)) {
            if (lane == first) atomicAdd(&h[d0], __popc(act));
          } else if (on) {
            atomicAdd(&h[digit], 1);
          }
        }
      }
      cl.sync();
      if (pass == 3) {
#pragma unroll
        for (int rk = 0; rk < CL_CTAS; ++rk) {
          nF += *cl.map_shared_rank(&sh_cnt[0], rk);
          nC += *cl.map_shared_rank(&sh_cnt[1], rk);
        }
        cstar = (N <= p.C) ? nC : max(0, p.C - nF);  // R15, R14
        cstar = min(cstar, nC);
        keep_all = (cstar == nC); keep_none = (cstar == 0);
        remaining = cstar;
        if (keep_all || keep_none) break;  // uniform over the cluster: no threshold to find
      }
      if (tid < 256) {
        int v = 0;
#pragma unroll
        for (int rk = 0; rk < CL_CTAS; ++rk) v += *cl.map_shared_rank(&h[tid], rk);
        comb[tid] = v;
        hist[(pass & 1) ^ 1][tid] = 0;  // next pass's buffer: last read before the barrier above
      }
      __syncthreads();
      if (tid < 32) {
        // lane l covers digits 255 - 8 l .. 248 - 8 l (descending)
        int s = 0;
#pragma unroll
        for (int e = 0; e < 8; ++e) s += comb[255 - (lane * 8 + e)];
        int inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int n = __shfl_up_sync(0xffffffffu, inc, o);
          if (lane >= o) inc += n;
        }
        const int excl = inc - s;
        const uint32_t hit = __ballot_sync(0xffffffffu, inc >= remaining);
        const int src = hit ? (__ffs(hit) - 1) : 31;
        if (lane == src) {
          int cum = excl, d = 255 - lane * 8;
          for (int e = 0; e < 7; ++e, --d) {
            if (cum + comb[d] >= remaining) break;
            cum += comb[d];
          }
          sh_remaining = remaining - cum;
          sh_prefix = prefix | ((uint32_t)d << shift);
        }
      }
      __syncthreads();
      prefix = sh_prefix;
      remaining = sh_remaining;
      __syncthreads();
    }
    if (!keep_all && !keep_none) {
      thr = prefix;
      need_eq = remaining;  // ties at the threshold survive lowest positions first (R13)
    }
  }

  // ---- ties in position order
  uint32_t eq_m = 0;
  if (!keep_all && !keep_none) {
#pragma unroll
    for (int i = 0; i < MAXI; ++i)
      if (((cand_m >> i) & 1u) && key[i] == thr) eq_m |= 1u << i;
  }
  int eq_before = 0;
  {
    // ties of the lower ranks: their last-pass histograms (pass 0 counted, in bin thr & 255, exactly the keys equal to
    // the threshold) are complete since that pass' cluster barrier and are not written again -- no barrier of its own
    int tot;
    const int ex = block_excl_scan_1024(__popc(eq_m), warp_tot, &tot);
    int before = 0;
    if (!keep_all && !keep_none)
      for (int rk = 0; rk < crank; ++rk) before += *cl.map_shared_rank(&hist[0][thr & 255u], rk);
    eq_before = before + ex;
  }

  // ---- keep flags, kept-slot bitmap, first dropped position per slot
  uint32_t keep_m = forced_m, drop_m = 0;  // drop_m: live and not kept (newly dropped)
  {
    int e = eq_before;
#pragma unroll
    for (int i = 0; i < MAXI; ++i) {
      if ((cand_m >> i) & 1u) {
        bool keep = keep_all;
        if (!keep_all && !keep_none) {
          if (key[i] > thr) keep = true;
          else if ((eq_m >> i) & 1u) { keep = e < need_eq; ++e; }
        }
        if (keep) keep_m |= 1u << i; else drop_m |= 1u << i;
      }
    }
#pragma unroll
    for (int i = 0; i < MAXI; ++i) {
      const int j = base + i;
      if ((keep_m >> i) & 1u) atomicOr(&p.kept_bits[slot[i] >> 5], 1u << (slot[i] & 31));
      else if (((drop_m >> i) & 1u) && j >= p.radix) atomicMin(&p.firstpos[slot[i]], j);
    }
  }
  cl.sync();  // arrive.release / wait.acquire at cluster scope: the bitmap and table updates are visible to every rank

  // ---- freed test (PAPER.md:132 (a)(b)(c)), ordered compaction of survivors and freed slots
  uint32_t freed_m = 0;
#pragma unroll
  for (int i = 0; i < MAXI; ++i) {
    const int j = base + i;
    if (((drop_m >> i) & 1u) && j >= p.radix) {
      const uint32_t bits = __ldcg(&p.kept_bits[slot[i] >> 5]);
      const int fp = __ldcg(&p.firstpos[slot[i]]);
      if (!((bits >> (slot[i] & 31)) & 1u) && fp == j) freed_m |= 1u << i;
    }
  }
  int live_o, freed_o, n_kept_all, n_freed_all;
  {
    int tot;
    const int ex = block_excl_scan_1024(__popc(keep_m) | (__popc(freed_m) << 16), warp_tot, &tot);
    if (tid == 0) { sh_kf[0] = tot & 0xffff; sh_kf[1] = tot >> 16; }
    cl.sync();  // also: every rank has finished reading kept_bits / firstpos
    int b0, b1;
    cluster_offsets(cl, &sh_kf[0], crank, &b0, &n_kept_all);
    cluster_offsets(cl, &sh_kf[1], crank, &b1, &n_freed_all);
    live_o = b0 + (ex & 0xffff);
    freed_o = b1 + (ex >> 16);
  }
#pragma unroll
  for (int i = 0; i < MAXI; ++i) {
    const int j = base + i;
    if (j < N) {
      const bool keep = (keep_m >> i) & 1u;
      if (keep) {
        p.live_slots[live_o++] = slot[i];
        atomicAnd(&p.kept_bits[slot[i] >> 5], ~(1u << (slot[i] & 31)));  // restore the scratch invariant
      } else if ((drop_m >> i) & 1u) {
        p.S[j] = p.dead;
        if (j >= p.radix) p.firstpos[slot[i]] = INT_MAX;
        if ((freed_m >> i) & 1u) p.freed[freed_o++] = slot[i];
      }
      if (p.valid) p.valid[j] = keep ? 1 : 0;
    }
  }
  // pad the survivor list with the dead slot up to N: decode sizes its splits from a host-side bound
  for (int i = n_kept_all + crank * 1024 + tid; i < N; i += CL_CTAS * 1024) p.live_slots[i] = p.dead;
  if (crank == 0 && tid == 0) {
    *p.n_kept = n_kept_all;
    *p.n_freed = n_freed_all;
    *p.n_live = n_kept_all;
  }
  cl.sync();  // shared memory stays mapped until every rank has read it
}

}  // namespace ikv
