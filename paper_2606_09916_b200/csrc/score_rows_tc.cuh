// score_rows_tc.cuh -- NEXT-1, the multi-row scorer (PAPER.md:91 "window of W tail Q rows", :159 "tail window W=32",
// :310) in two sweeps over the keys, the (R*G) x T x D contraction on tcgen05:
//
//   score[t] = sum_r w_r sum_{l,h} softmax_t( rows[r,l,h] . K[l,kv(h),t] / sqrt(D) )[t]        (R28)
//
// Up to 128 / G rows form a BANK: per (layer l, KV head) a 128 x D operand whose row c = r*G + g is row r's query head
// kvh*G + g (scaled by log2(e)/sqrt(D), split into bf16 hi + lo; rows beyond R*G are zero).  A CTA owns fixed
// 128-token tiles (two at a time) and walks (layer, KV head) items with the bank of the item resident in shared memory
// (double-buffered bulk copies); per (item, tile) = sub-item the gather warps copy the tile's keys of that head
// through the slot map straight into the canonical K-major operand layout (8-token x 16-byte core matrices, cp.async),
// and one thread issues 2 * D/16 tcgen05.mma (hi, lo) into a 128-column TMEM accumulator.  Three key buffers and
// three accumulators: the MMAs of one sub-item run under the statistics of the previous ones and the gathers of the
// next two.  The gather is the limit: 256-byte pieces of random rows arrive at ~15 bytes per cycle per SM whatever the
// copy instruction (measured: cp.async 16 B, bulk copies of 256 B), a third of what 2 KB rows reach in the key pass.
//   sweep 1 (statistics):  D[bank row, token] = bank . keys^T   -- thread = bank row: (max, sum 2^x) over the tile's
//                          tokens is thread-local; partials per (item, slot) -> k_rows_lse -> lse[item, c].
//   sweep 2 (sums):        D[token, bank row] = keys . bank^T   -- thread = token: sum_c w_c 2^(x - lse_c) is
//                          thread-local and accumulates in a register over all items; written to rule_c per tile pair.
// The same two shared-memory operands serve both sweeps with the A / B roles exchanged (both are K-major, no swizzle).
// Sixteen compute warps: warps w, w + 4, w + 8, w + 12 own the same 32 TMEM lanes and take a quarter of the
// accumulator's columns each (the statistics are MUFU-bound: 8 cycles per ex2 warp instruction per SM sub-partition,
// measured); eight more warps gather the keys.
#pragma once
#include <cuda.h>
#include "residual_tc.cuh"
#include "score_lm.cuh"

namespace ikv {

constexpr int RB_ROWS = 128;                 // bank rows = MMA M (sweep 1) / N (sweep 2)
constexpr int RB_TOK = 128;                  // tokens per tile
constexpr int RB_TAIL = 1024;                // bytes after the operands: lse[128] | w[128]
constexpr int RB_CWARPS = 16;                // compute warps
constexpr int RB_CQ = RB_CWARPS / 4;         // column groups of the accumulator (one warp per lane quarter each)
constexpr int RB_CG = 128 / RB_CQ;           // columns per group
constexpr int RB_PWARPS = 8;                 // key gather warps: warp (token quarter, half of the row's chunks)
constexpr int RB_THREADS = (RB_CWARPS + 2 + RB_PWARPS) * 32;  // + the bank loader warp + the MMA issuer warp
constexpr int RB_KBUF = 3;                   // key operand buffers
constexpr int RB_TB = 3;                     // TMEM accumulators (128 columns each; exchange columns behind them)
__host__ __device__ constexpr int rb_part(int D) { return RB_ROWS * D * 2; }          // bytes of hi (or lo)
__host__ __device__ constexpr int rb_item(int D) { return 2 * rb_part(D) + RB_TAIL; }  // bank bytes per (l, kvh)
// canonical K-major offset of the 16-byte entry (row n, 8 consecutive k starting at 8 * k8) of an [rows x D] operand
__host__ __device__ __forceinline__ int rb_entry(int n, int k8, int D) { return (n >> 3) * (D / 8) * 128 + k8 * 128 + (n & 7) * 16; }
inline size_t rb_smem(int D) { return 2 * (size_t)rb_item(D) + RB_KBUF * (size_t)RB_TOK * D * 2 + 256; }

struct RowsWeights { float w[RB_ROWS]; };  // weight of bank row c (0 for padding rows)

// bank[item = l*Hkv + kvh] = [hi 128 x D | lo 128 x D | lse[128] (written by k_rows_lse) | w[128]]
template <int D>
__global__ void k_rows_prep(const float* __restrict__ rows, int n_rows, int L, int Hkv, int G, RowsWeights wts,
                            unsigned char* __restrict__ bank) {
  const int item = blockIdx.x, l = item / Hkv, kvh = item % Hkv, Hq = Hkv * G;
  unsigned char* dst = bank + (size_t)item * rb_item(D);
  const float inv = 1.4426950408889634f / sqrtf((float)D);  // logits in the log2 domain: exp(x) = exp2(x log2 e)
  for (int e = threadIdx.x; e < RB_ROWS * (D / 8); e += blockDim.x) {
    const int c = e / (D / 8), k8 = e % (D / 8), r = c / G, g = c % G;
    uint32_t hi[4] = {0, 0, 0, 0}, lo[4] = {0, 0, 0, 0};
    if (r < n_rows) {
      const float* src = rows + (((int64_t)r * L + l) * Hq + kvh * G + g) * D + k8 * 8;
#pragma unroll
      for (int j = 0; j < 4; ++j) split_bf16(src[2 * j] * inv, src[2 * j + 1] * inv, hi[j], lo[j]);
    }
    *reinterpret_cast<uint4*>(dst + rb_entry(c, k8, D)) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(dst + rb_part(D) + rb_entry(c, k8, D)) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  }
  float* tail = reinterpret_cast<float*>(dst + 2 * rb_part(D));
  for (int c = threadIdx.x; c < RB_ROWS; c += blockDim.x) { tail[c] = 0.f; tail[RB_ROWS + c] = wts.w[c]; }
}

// lse[item, c] = log2 sum 2^x over all candidates, from the partials of sweep 1.  Block = item, 1,024 threads: thread
// (c, sg) folds the slots sg, sg + 8, ... in ascending order, the eight folds are combined in sg order (deterministic).
template <int D>
__global__ __launch_bounds__(1024) void k_rows_lse(const float2* __restrict__ partials, int n_slots,
                                                   unsigned char* __restrict__ bank) {
  __shared__ float2 part_s[8][RB_ROWS];
  const int item = blockIdx.x, c = threadIdx.x & (RB_ROWS - 1), sg = threadIdx.x >> 7;
  const float2* p = partials + (size_t)item * n_slots * RB_ROWS + c;
  float m = -CUDART_INF_F, s = 0.f;
  auto fold = [&](float2 v) {
    if (v.y > 0.f) {
      const float mn = fmaxf(m, v.x);
      s = s * exp2f(m - mn) + v.y * exp2f(v.x - mn);
      m = mn;
    }
  };
  for (int j = sg; j < n_slots; j += 8) fold(p[(size_t)j * RB_ROWS]);
  part_s[sg][c] = make_float2(m, s);
  __syncthreads();
  if (sg == 0) {
    for (int k = 1; k < 8; ++k) fold(part_s[k][c]);
    reinterpret_cast<float*>(bank + (size_t)item * rb_item(D) + 2 * rb_part(D))[c] = m + log2f(s);  // no candidates: unused
  }
}

// K-major, 128-byte-swizzled operand written by TMA (1 KB atoms of 8 rows), and the gather4 instruction itself
__device__ __forceinline__ uint64_t rb_desc_sw128(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3fff) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)2 << 61);
}
__device__ __forceinline__ void rb_gather4(uint32_t dst, const CUtensorMap* tm, uint64_t* bar, int col, int r0, int r1, int r2, int r3) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(dst),
      "l"(tm), "r"(smem_u32(bar)), "r"(col), "r"(r0), "r"(r1), "r"(r2), "r"(r3)
      : "memory");
}

struct RowsPassParams {
  const bf16* k_pool;
  int64_t layer_stride;  // elements
  int L, Hkv, n_cols;    // n_cols = bank rows in use (R*G)
  const unsigned char* bank;
  const int32_t* cand_slot;
  const int32_t* n_cand;
  float2* partials;      // sweep 1: [item][slot][128], slot = (pair, cta, column group)
  int n_slots, n_pairs;
  float* rule_c;         // sweep 2
  int accumulate;        // sweep 2: add to rule_c (second and later banks)
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void tmem_ld32f(uint32_t taddr, float* v) {
  tmem_ld16(taddr, v);
  tmem_ld16(taddr + 16, v + 16);
}
__device__ __forceinline__ void cp_async16_zfill(uint32_t dst_smem, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst_smem), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Roles: warps [0, RB_CWARPS) take the statistics from TMEM; then one warp streams the banks, one issues the MMAs and
// RB_PWARPS warps gather the keys.
// Sub-item K = (pair of tiles, item, tile t): key buffer K % 3, TMEM buffer K & 1, bank buffer (item count) & 1.
template <int D, int SWEEP, bool TG>
__global__ __launch_bounds__(RB_THREADS, 1) void k_rows_pass(const RowsPassParams p, const __grid_constant__ CUtensorMap tmk) {
  constexpr int CH = D / 8;                      // 16-byte chunks of a key row of one head
  constexpr int PART = rb_part(D), ITEM = rb_item(D);
  constexpr int COPY = SWEEP == 1 ? 2 * PART : ITEM;
  constexpr int KB = RB_TOK * D * 2;              // key operand bytes
  constexpr uint32_t SBO = (uint32_t)(D / 8) * 128u;
  constexpr int CT = RB_CWARPS * 32;
  extern __shared__ __align__(1024) unsigned char rb_smem_raw[];
  unsigned char* bank_s = rb_smem_raw;                    // [2][ITEM]
  unsigned char* keys_s = rb_smem_raw + 2 * ITEM;         // [RB_KBUF][KB]
  uint64_t* bars = reinterpret_cast<uint64_t*>(keys_s + RB_KBUF * KB);
  uint64_t* bank_full = bars;             // [2]  bulk copy landed
  uint64_t* bank_empty = bars + 2;        // [2]  sweep 1: the item's MMAs completed; sweep 2: every thread read lse / w
  uint64_t* mma_done = bars + 4;          // [RB_TB]  accumulator of the TMEM buffer complete
  uint64_t* tmem_free = mma_done + RB_TB; // [RB_TB]  every compute thread has read the accumulator
  uint64_t* keys_ready = tmem_free + RB_TB;   // [RB_KBUF] every gather thread's part of the operand is in shared memory
  uint64_t* keys_free = keys_ready + RB_KBUF; // [RB_KBUF] the MMAs that read the operand completed
  uint32_t* tmem_base_p = reinterpret_cast<uint32_t*>(keys_free + RB_KBUF);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int b = 0; b < 2; ++b) {
      mbar_init(&bank_full[b], 1);
      mbar_init(&bank_empty[b], SWEEP == 1 ? 1 : CT);
    }
    for (int b = 0; b < RB_TB; ++b) { mbar_init(&mma_done[b], 1); mbar_init(&tmem_free[b], CT); }
    for (int b = 0; b < RB_KBUF; ++b) { mbar_init(&keys_ready[b], TG ? 1 : RB_PWARPS * 32); mbar_init(&keys_free[b], 1); }
    mbar_fence_init();
  }
  if (warp == 0) {  // columns [0, 384): three accumulators; [384, 400): exchange between the column groups (sweep 2)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_p)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_base_p;
  const int n_items = p.L * p.Hkv;
  const int n_sub = 2 * n_items;               // sub-items per pair of tiles
  const int total = p.n_pairs * n_sub;
  const int nc = *p.n_cand;

  if (warp == RB_CWARPS) {
    // ------------------------------------------------------------------ bank loader: one bulk copy per item
    if (lane == 0) {
      int j = 0;
      for (int pr = 0; pr < p.n_pairs; ++pr)
        for (int it = 0; it < n_items; ++it, ++j) {
          const int b = j & 1;
          mbar_wait(&bank_empty[b], ((uint32_t)(j >> 1) & 1u) ^ 1u);
          mbar_arrive_expect_tx(&bank_full[b], (uint32_t)COPY);
          bulk_g2s(bank_s + (size_t)b * ITEM, p.bank + (size_t)it * ITEM, (uint32_t)COPY, &bank_full[b]);
        }
    }
  } else if (warp == RB_CWARPS + 1) {
    // ------------------------------------------------------------------ MMA issuer (one thread)
    if (lane == 0) {
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
      const uint32_t keys_u32 = smem_u32(keys_s), bank_u32 = smem_u32(bank_s);
      int kb = 0;
      uint32_t kph = 0u;
      for (int K = 0; K < total; ++K) {
        const int j = K >> 1, t = K & 1, b = j & 1;      // j = item count over the pairs
        const uint32_t buf = (uint32_t)(K % RB_TB);
        mbar_wait(&keys_ready[kb], kph);
        if (t == 0) mbar_wait(&bank_full[b], (uint32_t)(j >> 1) & 1u);
        mbar_wait(&tmem_free[buf], ((uint32_t)(K / RB_TB) & 1u) ^ 1u);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint64_t d_keys0 = umma_desc(keys_u32 + (uint32_t)(kb * KB), 128, SBO);
        const uint64_t d_hi = umma_desc(bank_u32 + (uint32_t)(b * ITEM), 128, SBO);
        const uint64_t d_lo = d_hi + (uint64_t)(PART >> 4);
        const uint32_t td = tmem + buf * 128u;
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint64_t o = (uint64_t)((ks * 256) >> 4);
          // tensor-map gathers: keys as [column half][128 tokens][128 B], 128-byte swizzle, 32 B per 16 k inside an atom
          const uint64_t d_keys = TG ? rb_desc_sw128(keys_u32 + (uint32_t)(kb * KB + (ks >> 2) * (RB_TOK * 128) + (ks & 3) * 32)) - o
                                     : d_keys0;
          if (SWEEP == 1) {
            umma_bf16(td, d_hi + o, d_keys + o, idesc, ks ? 1u : 0u);
            umma_bf16(td, d_lo + o, d_keys + o, idesc, 1u);
          } else {
            umma_bf16(td, d_keys + o, d_hi + o, idesc, ks ? 1u : 0u);
            umma_bf16(td, d_keys + o, d_lo + o, idesc, 1u);
          }
        }
        umma_commit(&mma_done[buf]);
        umma_commit(&keys_free[kb]);
        if (SWEEP == 1 && t == 1) umma_commit(&bank_empty[b]);   // arrives when every MMA issued so far has completed
        if (++kb == RB_KBUF) { kb = 0; kph ^= 1u; }
      }
    }
  } else if (TG && warp >= RB_CWARPS + 2) {
    // ------------------------------------------------------------------ key gather warps, tensor-map path: OPW lanes of
    // each warp issue one TMA gather4 per sub-item (four tokens x 128 bytes of one column half of the head's keys; the
    // issue costs a warp ~75 cycles per instruction whatever the lane count, hence eight warps); tokens beyond the
    // candidates get an out-of-range row (zero fill).  The mbarrier of the buffer counts the bytes.
    constexpr int HALVES = D / 64, OPS = (RB_TOK / 4) * HALVES, OPW = OPS / RB_PWARPS;
    const int o = (warp - (RB_CWARPS + 2)) * OPW + lane, quad = o / HALVES, half = o % HALVES;
    if (lane < OPW) {
      const uint32_t keys_u32 = smem_u32(keys_s);
      const int rows_per_layer = (int)(p.layer_stride / D);
      int rw[2][4];   // slot * H_kv of this lane's four tokens in tile 0 / 1 of the pair; -1: no candidate
      auto load_slots = [&](int pr) {
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          const int t0 = ((2 * pr + t) * (int)gridDim.x + (int)blockIdx.x) * RB_TOK;
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int tok = t0 + quad * 4 + e;
            rw[t][e] = tok < nc ? p.cand_slot[tok] * p.Hkv : -1;
          }
        }
      };
      int g_l = 0, g_kvh = 0, g_sub = 0, g_pr = 0, kb = 0;
      uint32_t kph = 0u;
      if (total > 0) load_slots(0);
      for (int K = 0; K < total; ++K) {
        const int t = K & 1;
        mbar_wait(&keys_free[kb], kph ^ 1u);
        if (o == 0) mbar_arrive_expect_tx(&keys_ready[kb], (uint32_t)KB);
        const int base = g_l * rows_per_layer + g_kvh;
        int r[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int v = t ? rw[1][e] : rw[0][e];
          r[e] = v >= 0 ? v + base : -1;
        }
        rb_gather4(keys_u32 + (uint32_t)(kb * KB + half * (RB_TOK * 128) + quad * 512), &tmk, &keys_ready[kb], half * 64, r[0], r[1],
                   r[2], r[3]);
        if (++kb == RB_KBUF) { kb = 0; kph ^= 1u; }
        if (t == 1) {
          if (++g_kvh == p.Hkv) { g_kvh = 0; if (++g_l == p.L) g_l = 0; }
        }
        if (++g_sub == n_sub) { g_sub = 0; if (++g_pr < p.n_pairs) load_slots(g_pr); }
      }
    }
  } else if (warp >= RB_CWARPS + 2) {
    // ------------------------------------------------------------------ key gather warps: sub-item K into buffer K % 3
    // as soon as the MMAs of K - 3 have completed; published one iteration later, so that two gathers are in flight and
    // the wait never depends on a sub-item these warps have not published yet
    const int pw = (warp - (RB_CWARPS + 2)) & 3, ph2 = (warp - (RB_CWARPS + 2)) >> 2, tok8 = lane & 7, c4 = lane >> 3;
    const uint32_t keys_u32 = smem_u32(keys_s);
    int64_t slot[2][4];   // lane = (token % 8, chunk % 4): tokens pw*32 + i*8 + tok8 of tile 0 / 1 of the pair
    auto load_slots = [&](int pr) {
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int t0 = ((2 * pr + t) * (int)gridDim.x + (int)blockIdx.x) * RB_TOK;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int tok = t0 + pw * 32 + i * 8 + tok8;
          slot[t][i] = tok < nc ? (int64_t)p.cand_slot[tok] : -1;
        }
      }
    };
    int g_l = 0, g_kvh = 0, g_sub = 0, g_pr = 0, kb = 0;
    uint32_t kph = 0u;
    if (total > 0) load_slots(0);
    for (int K = 0; K < total; ++K) {
      const int t = K & 1;
      mbar_wait(&keys_free[kb], kph ^ 1u);
      const bf16* base = p.k_pool + (int64_t)g_l * p.layer_stride + (int64_t)g_kvh * D;
      const uint32_t dst0 = keys_u32 + (uint32_t)(kb * KB);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int64_t sl = t ? slot[1][i] : slot[0][i];
        const bf16* src = base + (sl >= 0 ? sl : 0) * (int64_t)(p.Hkv * D);
#pragma unroll
        for (int jj = 0; jj < CH / 8; ++jj) {
          const int jc = ph2 * (CH / 8) + jj;
          cp_async16_zfill(dst0 + (uint32_t)rb_entry(pw * 32 + i * 8 + tok8, jc * 4 + c4, D), src + (jc * 4 + c4) * 8,
                           sl >= 0 ? 16u : 0u);  // tokens beyond the candidates: zero rows
        }
      }
      cp_async_commit();
      if (K > 0) {
        cp_async_wait<1>();
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_arrive(&keys_ready[kb == 0 ? RB_KBUF - 1 : kb - 1]);
      }
      if (++kb == RB_KBUF) { kb = 0; kph ^= 1u; }
      if (t == 1) {   // next (layer, head); after the last one the next pair of tiles
        if (++g_kvh == p.Hkv) { g_kvh = 0; if (++g_l == p.L) g_l = 0; }
      }
      if (++g_sub == n_sub) { g_sub = 0; if (++g_pr < p.n_pairs) load_slots(g_pr); }
    }
    if (total > 0) {
      cp_async_wait<0>();
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_arrive(&keys_ready[kb == 0 ? RB_KBUF - 1 : kb - 1]);
    }
  } else {
    // ------------------------------------------------------------------ compute warps: statistics only.  Warp w owns
    // the TMEM lane quarter w % 4 and the column group cq = w / 4 (RB_CG columns of the 128)
    const int wq = warp & 3, cq = warp >> 2, tid = wq * 32 + lane;   // tid = TMEM lane (bank row / token)
    const uint32_t tlane = tmem + ((uint32_t)(wq * 32) << 16);        // this warp's 32 TMEM lanes
    int c_t0[2], c_nv[2];
    auto set_pair = [&](int pr) {
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        c_t0[t] = ((2 * pr + t) * (int)gridDim.x + (int)blockIdx.x) * RB_TOK;
        c_nv[t] = max(0, min(RB_TOK, nc - c_t0[t]));
      }
    };
    float acc[2] = {0.f, 0.f};   // sweep 2: this thread's token of tile 0 / tile 1 of the statistics' pair
    float pm = -CUDART_INF_F, ps = 0.f;   // sweep 1: (max, sum) of tile 0 until tile 1 of the same item is done
    // statistics of sub-item Ks: item `it` of pair `prs`, tile t
    auto stats = [&](int Ks, int it, int prs) {
      const int t = Ks & 1, j = Ks >> 1, b = j & 1;
      const int snv = t ? c_nv[1] : c_nv[0];
      const uint32_t buf = (uint32_t)(Ks % RB_TB);
      mbar_wait(&mma_done[buf], (uint32_t)(Ks / RB_TB) & 1u);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t tl = tlane + buf * 128u + (uint32_t)(cq * RB_CG);
      float x[RB_CG];
      if (SWEEP == 1) {
        float m = -CUDART_INF_F, s = 0.f;
        const int nq = min(RB_CG, snv - cq * RB_CG);   // this warp's share of the token columns
        if (nq > 0) {
#pragma unroll
          for (int c0 = 0; c0 < RB_CG; c0 += 16) tmem_ld16(tl + (uint32_t)c0, x + c0);   // beyond the tile: read, not used
          tmem_ld_wait();
          if (nq == RB_CG) {
            float c0 = x[0], c1 = x[1];
#pragma unroll
            for (int e = 2; e < RB_CG; e += 2) { c0 = fmaxf(c0, x[e]); c1 = fmaxf(c1, x[e + 1]); }
            m = fmaxf(c0, c1);
            float s0 = 0.f, s1 = 0.f;
#pragma unroll
            for (int e = 0; e < RB_CG; e += 2) { s0 += ex2_approx(x[e] - m); s1 += ex2_approx(x[e + 1] - m); }
            s = s0 + s1;
          } else {
#pragma unroll
            for (int e = 0; e < RB_CG; ++e)
              if (e < nq) m = fmaxf(m, x[e]);
#pragma unroll
            for (int e = 0; e < RB_CG; ++e)
              if (e < nq) s += ex2_approx(x[e] - m);
          }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        mbar_arrive(&tmem_free[buf]);
        if (t == 0) {   // the two tiles of the pair are the same bank row of the same item: one partial for both
          pm = m; ps = s;
        } else {
          const float mn = fmaxf(pm, m);
          if (mn > -CUDART_INF_F) { s = ps * ex2_approx(pm - mn) + s * ex2_approx(m - mn); m = mn; }
          const int slot_id = (prs * (int)gridDim.x + (int)blockIdx.x) * RB_CQ + cq;
          p.partials[((size_t)it * p.n_slots + slot_id) * RB_ROWS + tid] = make_float2(m, s);
        }
      } else {
        const int q0 = cq * RB_CG, nq = min(RB_CG, p.n_cols - q0);   // this warp's share of the bank rows
        if (snv > 0 && nq > 0) {
          mbar_wait(&bank_full[b], (uint32_t)(j >> 1) & 1u);   // the bulk copy's bytes (lse, w) are visible to this thread
          const float* tail = reinterpret_cast<const float*>(bank_s + (size_t)b * ITEM + 2 * PART);
          float a0 = 0.f, a1 = 0.f;
#pragma unroll
          for (int c0 = 0; c0 < RB_CG; c0 += 16)
            if (c0 < nq) tmem_ld16(tl + (uint32_t)c0, x + c0);
          tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < RB_CG; e += 4) {
            if (e < nq) {   // groups of four columns: the bank's padding rows have w = 0 and a finite lse
              const float4 ls = *reinterpret_cast<const float4*>(tail + q0 + e);
              const float4 ws = *reinterpret_cast<const float4*>(tail + RB_ROWS + q0 + e);
              a0 = fmaf(ws.x, ex2_approx(x[e] - ls.x), a0);
              a1 = fmaf(ws.y, ex2_approx(x[e + 1] - ls.y), a1);
              a0 = fmaf(ws.z, ex2_approx(x[e + 2] - ls.z), a0);
              a1 = fmaf(ws.w, ex2_approx(x[e + 3] - ls.w), a1);
            }
          }
          if (t) acc[1] += a0 + a1; else acc[0] += a0 + a1;
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        mbar_arrive(&tmem_free[buf]);
        if (t == 1) mbar_arrive(&bank_empty[b]);   // this thread is done with the item's lse / w
      }
    };
    // end of a pair (sweep 2): the column groups of a token meet through spare TMEM columns (four per group; the warps
    // w, w + 4, ... own the same lanes); group 0 adds them in group order and writes the sums
    auto flush = [&]() {
      const uint32_t tx = tlane + (uint32_t)(RB_TB * 128);
      if (cq > 0) {
        const float v4[4] = {acc[0], acc[1], 0.f, 0.f};
        tmem_st4(tx + (uint32_t)(4 * cq), v4);
        tmem_wait_st();
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      bar_sync(1, CT);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      if (cq == 0) {
        float s0 = acc[0], s1 = acc[1];
#pragma unroll
        for (int k = 1; k < RB_CQ; ++k) {
          float o[4];
          tmem_ld4(tx + (uint32_t)(4 * k), o);
          tmem_wait_ld();
          s0 += o[0]; s1 += o[1];
        }
        if (tid < c_nv[0]) { const int tok = c_t0[0] + tid; p.rule_c[tok] = (p.accumulate ? p.rule_c[tok] : 0.f) + s0; }
        if (tid < c_nv[1]) { const int tok = c_t0[1] + tid; p.rule_c[tok] = (p.accumulate ? p.rule_c[tok] : 0.f) + s1; }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      bar_sync(1, CT);
      acc[0] = acc[1] = 0.f;
    };
    set_pair(0);
    int s_sub = 0, s_pr = 0;   // statistics: sub-item inside its pair, pair
    auto stats_next = [&](int Ks) {
      stats(Ks, s_sub >> 1, s_pr);
      if (++s_sub == n_sub) {   // last sub-item of its pair: write the pair's sums, move on to the next pair
        if (SWEEP == 2) flush();
        s_sub = 0;
        if (++s_pr < p.n_pairs) set_pair(s_pr);
      }
    };
    for (int K = 0; K < total; ++K) stats_next(K);
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
  }
}

}  // namespace ikv
