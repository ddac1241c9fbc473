// fused_small.cuh -- the small per-call kernels around the key pass, fused into two launches (each launch costs
// ~1.2 us of stream latency on B200, and several of these bodies are latency-bound on their own):
//   k_mem_prep : B fragments of M / sqrt(D) for the key pass  |  partial sums of mbar (Eq. 5)
//   k_post_key : lse[l,h] from the per-CTA partials (Eq. 3), a warp per row
//   k_rule_fused : rule_c (Eq. 3)  |  folded W_Q / fc1 operands  |  Kc / Vc fragments (Eq. 6); the block index selects the body.
#pragma once
#include "residual_mma.cuh"
#include "residual_tc.cuh"
#include "score.cuh"
#include "score_mma.cuh"

namespace ikv {

template <int D, int G>
__global__ __launch_bounds__(128) void k_mem_prep(const float* __restrict__ M, int L, int Hkv, float inv_sqrt_d,
                                                  uint4* __restrict__ frag, int n_frag_blocks, int LH,
                                                  float* __restrict__ mpart, int32_t* __restrict__ layer_cnt) {
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  const int bid = blockIdx.x;
  if (bid == 0 && layer_cnt)  // per-layer arrival counters of the layer-major key pass
    for (int l = threadIdx.x; l < L; l += 128) layer_cnt[l] = 0;
  if (bid < n_frag_blocks) {
    memory_frags_item<D, G>(bid * 128 + threadIdx.x, M, L, Hkv, inv_sqrt_d, frag);
    return;
  }
  mean_memory_part_block(bid - n_frag_blocks, M, LH, D, mpart);
}
template <int D, int G>
inline int mem_prep_frag_blocks(int L, int Hkv) {
  constexpr int NT = (G <= 4) ? 1 : 2;
  return (L * Hkv * NT * (D / 32) * 32 + 127) / 128;
}

struct PostKeyParams {
  const float2* partials; int n_part; float* lse; int n_lse;          // lse rows
  const float* mpart; int n_mpart; int LH; FoldOut fold; int n_fold;  // fold blocks (0: not a learnable call)
  int mbar_ready;  // rt.mbar was reduced by the layer-major key pass
  const float* kq; const int32_t* n_xq; int nks; uint4 *kc_frag, *vc_frag; int n_kv;  // Kc / Vc blocks
  int tc; int nxp; RtFoldOut rt;  // tc != 0: operands of k_residual_tc instead (n_fold fc1 blocks, n_kv cross-attention blocks)
};

// lse[l,h] = log sum_c exp(x[l,h,c]) from the per-CTA (max, sum) partials of the key pass: one warp per (l,h) row, no
// block barrier (the row has one partial per key-pass CTA, 148 of them).  TC: the launch also carries the fold bodies of
// k_tail_tc (blocks of 256 threads; the lse and fc1 bodies use the first 128): n_fold fc1 blocks, then n_kv cross-attention
// blocks, which need the mean keys of the query positions and hence the finished key pass.
__device__ __forceinline__ void lse_rows_block(int bid, const float2* __restrict__ partials, int n_part,
                                               float* __restrict__ lse, int n_lse) {
  const int row = bid * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (row >= n_lse) return;
  const float2* pp = partials + (int64_t)row * n_part;
  float mx = -CUDART_INF_F;
  for (int i = lane; i < n_part; i += 32) mx = fmaxf(mx, pp[i].x);
  mx = warp_max(mx);
  float s = 0.f;
  for (int i = lane; i < n_part; i += 32) {
    const float2 v = pp[i];
    if (v.y > 0.f) s += v.y * expf(v.x - mx);
  }
  s = warp_sum(s);
  if (lane == 0) lse[row] = mx + logf(s);
}
template <int D, bool TC>
__global__ __launch_bounds__(TC ? 256 : 128) void k_post_key(const PostKeyParams p, const ResidW w) {
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  int bid = blockIdx.x;
  const int n_lse_blocks = (p.n_lse + 3) / 4;
  if (bid < n_lse_blocks) {
    if (threadIdx.x < 128) lse_rows_block(bid, p.partials, p.n_part, p.lse, p.n_lse);
    return;
  }
  if constexpr (TC) {
    bid -= n_lse_blocks;
    if (bid < p.n_fold) {
      if (threadIdx.x < 128) rt_fold_fc1_block<D>(bid, p.mpart, p.n_mpart, p.LH, w, p.rt, p.mbar_ready != 0);
      return;
    }
    rt_fold_xattn_block<D>(bid - p.n_fold, p.mpart, p.n_mpart, p.LH, p.kq, p.n_xq, p.nxp, w, p.rt, p.mbar_ready != 0);
  }
}

struct RuleParams {
  const float* logits; int64_t ldc; int LH; const float* lse; const int32_t* n_cand; const int32_t* cand_pos;
  float* rule_c; float* scores; int scatter_scores; float* rule_out; int n_rule;  // rule blocks (256 threads)
  int l2_hints;
};

// rule_c of Eq. 3 (HBM-bound, 256-thread blocks) and, for a learnable call, the folded W_Q / fc1 operands and the
// Kc / Vc fragments (latency-bound 128-thread bodies, warps 4-7 of their blocks exit) in one launch: the residual
// kernel needs all three, and the small bodies hide under the rule blocks' stream of the logits.
template <int D>
__global__ __launch_bounds__(256, 4) void k_rule_fused(const RuleParams r, const PostKeyParams p, const ResidW w) {
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  int bid = blockIdx.x;
  if (bid < r.n_rule) {
    score_rule4_block(bid, r.n_rule, r.logits, r.ldc, r.LH, r.lse, r.n_cand, r.cand_pos, r.rule_c, r.scores,
                      r.scatter_scores, r.rule_out, r.l2_hints);
    return;
  }
  bid -= r.n_rule;
  if (threadIdx.x >= 128) return;
  if (bid < p.n_fold) { resid_fold_block<D>(bid, p.mpart, p.n_mpart, p.LH, w, p.fold); return; }
  bid -= p.n_fold;
  resid_kv_frags_block(bid, p.kq, p.n_xq, D, w, p.nks, p.kc_frag, p.vc_frag);
}

}  // namespace ikv
