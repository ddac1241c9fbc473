// prefill_tc.cuh -- NEXT-2 on tcgen05: the causal chunk attention of prefill_mma.cuh with both contractions on the 5th-gen
// tensor cores, for G in {1, 2, 4, 8} (128 / G query rows x G heads of one KV head = one 128-row tile).
//
// CTA = (split of the items, KV head, block of MT x BR rows, BR = 128 / G).  M row m = i G + g: chunk row i, query head
// kvh G + g.  Per tile of 64 items:
//   producers            TG = true (default; the pools are covered by the tensor maps ikv_create builds): they do not
//                        touch the data.  Every 64-item tile is fetched by 64 TMA tile::gather4 instructions (four rows of
//                        128 bytes each; the row = (layer, slot, KV head) of the pool seen as a 2-D tensor [rows][D]; dead
//                        items get an out-of-range row: zero fill) with SWIZZLE_128B, which lands K as the K-major and
//                        V as the MN-major 128-byte-swizzled operand of tcgen05.mma: no transposition pass, no staging.
//                        A gather4 costs its issuing warp ~75 cycles whatever the lane count, so the issue is spread:
//                        eight warps x eight lanes (seven warps with two M tiles).  Per SM, 32 KB of random 256-byte
//                        pieces arrive in 1,190-1,730 cycles against 2,150-2,400 for cp.async or 256-byte bulk copies.
//                        TG = false (no tensor map): 2 x 2 warps, alternating tiles, gather the K rows with cp.async
//                        straight into the canonical no-swizzle K-major operand [64 items x D], the V rows into a
//                        row-major staging buffer, then transpose V with ldmatrix.trans into the canonical operand
//                        V^T [D x 64 items] (P V needs items as K);
//   MMA thread           S = Q K^T  (D/16 tcgen05.mma M128 N64 K16, double-buffered in TMEM), then O += P V
//                        (4 tcgen05.mma M128 N=D K16) once P is written; with MT = 2 for both M tiles on each K/V tile;
//   softmax (4 warps     thread = M row: tcgen05.ld of its 64 logits, causal / dead mask, exp2 against a LAZY reference
//   per M tile)          maximum (moved, with a rescale of the row's O and l, only when a tile's maximum exceeds it by
//                        more than 2^8), P as bf16 into the canonical A operand [128 x 64].
// Partials (reference m, l, O) per (row, head, split) as in prefill_mma.cuh; k_prefill_merge combines them.
#pragma once
#include <cuda.h>
#include "prefill_mma.cuh"

namespace ikv {

constexpr int PT_TOK = 64;            // items per tile
constexpr int PT_THREADS = 9 * 32;    // 4 softmax warps, 4 producer warps, MMA warp
constexpr int PT_PW_TG = 8;           // producer warps of the tensor-map path (64 / PT_PW_TG issuing lanes each)
constexpr int PT_THREADS_TG = (5 + PT_PW_TG) * 32;
constexpr int PT_PW_TG2 = 7;          // with two M tiles: 8 softmax + 7 producer + 1 MMA warps = 512 threads (128 registers each)
constexpr int PT_NB = 4;               // K / V^T buffers: the gathers run three tiles ahead of the MMAs
constexpr int PT_NB_TG = 4;            // the same on the tensor-map path (no staging buffers)
constexpr int PT_PB = 1;               // P buffers (shared memory: 4 K / V^T buffers leave room for one)
constexpr float PT_GROW = 8.f;        // log2 units a tile's maximum may exceed the reference before it moves

template <int D>
__host__ __device__ constexpr int pt_vst() { return D * 2 + 16; }   // staged V row stride (conflict-free ldmatrix)
template <int D, bool TG = false, int MT = 1>
__host__ __device__ constexpr int pt_smem() {
  // Q[MT] | K[NB] | V^T[NB] | V staging[2] (cp.async path) | P[MT][1 or 2] | minrow[NB][64] | barriers
  return MT * 128 * D * 2 + (TG ? PT_NB_TG : PT_NB) * (PT_TOK * D * 2 + D * PT_TOK * 2 + PT_TOK * 4) +
         (TG ? 0 : 2 * PT_TOK * pt_vst<D>()) + MT * ((TG && MT == 1) ? 2 : PT_PB) * 128 * PT_TOK * 2 + 256;
}
template <bool TG, int MT>
__host__ __device__ constexpr int pt_threads() { return TG ? (4 * MT + (MT == 2 ? PT_PW_TG2 : PT_PW_TG) + 1) * 32 : PT_THREADS; }
// shared-memory matrix descriptors of the 128-byte-swizzled operands the tensor map writes ([rows][128 B], 8-row atoms of
// 1 KB): K-major (start address advanced by 32 B per 16 k) and MN-major (64 contiguous n per atom, the next 64 at `lbo`)
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((saddr >> 4) & 0x3fff) | ((uint64_t)((lbo >> 4) & 0x3fff) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3fff) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
__device__ __forceinline__ void tma_gather4(uint32_t dst, const CUtensorMap* tm, uint64_t* bar, int col, int r0, int r1, int r2,
                                            int r3) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];" ::"r"(dst),
      "l"(tm), "r"(smem_u32(bar)), "r"(col), "r"(r0), "r"(r1), "r"(r2), "r"(r3)
      : "memory");
}
// canonical K-major (no swizzle) offset of the 16-byte entry (row n, k-group k8) of an operand with kdim elements of K
__host__ __device__ __forceinline__ int pt_entry(int n, int k8, int kdim) { return (n >> 3) * (kdim / 8) * 128 + k8 * 128 + (n & 7) * 16; }

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float* v) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
      "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
      "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
      "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15]))
      : "memory");
}

// MT = 2 (tensor-map path only): two 128-row M tiles per CTA, one softmax warpgroup each, share every K/V tile -- half
// the gather traffic and half the gather instructions per flop; all 512 TMEM columns (S double-buffered and O per M tile).
template <int D, int G, bool TG, int MT>
__global__ __launch_bounds__(pt_threads<TG, MT>(), 1) void k_prefill_tc(const PrefillParams p, const __grid_constant__ CUtensorMap tmk,
                                                              const __grid_constant__ CUtensorMap tmv) {
  static_assert(MT == 1 || TG, "two M tiles per CTA need the tensor-map producers");
  constexpr int BR = 128 / G;                // chunk rows per M tile
  constexpr int NPB = (TG && MT == 1) ? 2 : PT_PB;   // P buffers per M tile
  constexpr int SW = 4 * MT;                 // softmax warps
  constexpr int NB = TG ? PT_NB_TG : PT_NB;  // K / V buffers
  constexpr int NPW = TG ? (MT == 2 ? PT_PW_TG2 : PT_PW_TG) : 4, MMA_WARP = SW + NPW;
  constexpr int CPR = D / 8;                 // 16-byte chunks per K / V row
  constexpr int VST = pt_vst<D>();
  constexpr int QB = 128 * D * 2, KB = PT_TOK * D * 2, VTB = D * PT_TOK * 2, VSB = PT_TOK * VST, PB = 128 * PT_TOK * 2;
  constexpr uint32_t SBO_D = (uint32_t)(D / 8) * 128u, SBO_T = (uint32_t)(PT_TOK / 8) * 128u;
  constexpr uint32_t O_COL = 128, T_COLS = 256;   // TMEM per M tile: S buffers at columns 0 and 64, O at [128, 128 + D)
  extern __shared__ __align__(1024) unsigned char pt_smem_raw[];
  unsigned char* q_s = pt_smem_raw;
  unsigned char* k_s = q_s + MT * QB;            // [NB][KB]
  unsigned char* vt_s = k_s + NB * KB;           // [NB][VTB]: V^T (cp.async path) or V [half][item][128 B] (tensor map)
  unsigned char* vst_s = vt_s + NB * VTB;        // [2][VSB]: one per producer group (cp.async path only)
  unsigned char* p_s = vst_s + (TG ? 0 : 2 * VSB);   // [MT][NPB][PB]
  int* minrow_s = reinterpret_cast<int*>(p_s + MT * NPB * PB);   // [NB][PT_TOK]
  uint64_t* bars = reinterpret_cast<uint64_t*>(minrow_s + NB * PT_TOK);
  uint64_t* kv_full = bars;                 // [NB] operands K, V^T and minrow of a tile are in shared memory (64 threads)
  uint64_t* kv_free = kv_full + NB;      // [NB] the MMAs that read them have completed
  uint64_t* s_full = kv_free + NB;          // [MT][2] S accumulator complete
  uint64_t* s_free = s_full + MT * 2;       // [MT][2] every softmax thread of the M tile has read it
  uint64_t* p_full = s_free + MT * 2;       // [MT][NPB] P written (and O rescaled) by every softmax thread of the M tile
  uint64_t* p_free = p_full + MT * NPB;     // [MT][NPB] P V of the buffer's tile complete
  uint64_t* q_ready = p_free + MT * NPB;
  uint32_t* tmem_base_p = reinterpret_cast<uint32_t*>(q_ready + 1);

  const int split = blockIdx.x, kvh = blockIdx.y, rb = blockIdx.z;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int Hq = p.Hkv * G;
  if (threadIdx.x == 0) {
    for (int b = 0; b < NB; ++b) { mbar_init(&kv_full[b], 64); mbar_init(&kv_free[b], 1); }
    for (int b = 0; b < MT * 2; ++b) { mbar_init(&s_full[b], 1); mbar_init(&s_free[b], 128); }
    for (int b = 0; b < MT * NPB; ++b) { mbar_init(&p_full[b], 128); mbar_init(&p_free[b], 1); }
    mbar_init(q_ready, 128 * MT);
    mbar_fence_init();
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_p)), "n"(MT * 256));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_base_p;
  pdl_launch_dependents();   // the merge grid may be scheduled now; it waits (griddepcontrol.wait) for this grid to complete

  // items of this CTA (as in k_prefill_mma)
  const int n_cached = min(p.n_cached, *p.n_live);
  const int total = n_cached + (p.q_pos0 + p.n_q - p.covered);
  const int lim = min(total, n_cached + (p.q_pos0 + min(p.n_q, (rb + 1) * MT * BR) - p.covered));
  const int tiles_all = (total + PT_TOK - 1) / PT_TOK;
  const int t_begin = (int)(((int64_t)tiles_all * split) / p.n_split);
  const int t_end = min((int)(((int64_t)tiles_all * (split + 1)) / p.n_split), (lim + PT_TOK - 1) / PT_TOK);
  const int n_t = max(0, t_end - t_begin);

  if (TG && warp >= SW && warp < MMA_WARP) {
    // ------------------------------------------------------------------ producers, tensor-map path: lane < LPW of warp
    // SW + pw is thread j = LPW pw + lane < 64: it writes minrow of item j and issues gather4 number o (if o < OPS)
    constexpr int HALVES = D / 64, OPS = 2 * HALVES * 16, LPW = (PT_TOK + NPW - 1) / NPW;
    const int pw = warp - SW, j = pw * LPW + lane;
    if (lane < LPW && j < PT_TOK) {
      const int o = j;
      const int mat = o / (OPS / 2), rem = o % (OPS / 2), quad = rem / HALVES, half = rem % HALVES;
      const bool op = o < OPS;
      auto slot_at = [&](int idx) -> int {
        return idx < lim ? (idx < n_cached ? p.live_slots[idx] : p.S[p.covered + (idx - n_cached)]) : p.dead;
      };
      int sj = p.dead, s4[4] = {p.dead, p.dead, p.dead, p.dead};
      auto load_slots = [&](int tile) {
        sj = slot_at(tile * PT_TOK + j);
        if (op) {
#pragma unroll
          for (int e = 0; e < 4; ++e) s4[e] = slot_at(tile * PT_TOK + quad * 4 + e);
        }
      };
      if (n_t > 0) load_slots(t_begin);
      for (int it = 0; it < n_t; ++it) {
        const int b = it % NB, tile = t_begin + it;
        mbar_wait(&kv_free[b], ((uint32_t)(it / NB) & 1u) ^ 1u);   // P V of tile it - NB has completed
        const int idx = tile * PT_TOK + j;
        minrow_s[b * PT_TOK + j] = sj == p.dead ? INT_MAX : (idx < n_cached ? INT_MIN : p.covered + (idx - n_cached) - p.q_pos0);
        if (j == 0) mbar_arrive_expect_tx(&kv_full[b], (uint32_t)(OPS * 512));
        else mbar_arrive(&kv_full[b]);
        if (op) {
          int r[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) r[e] = s4[e] == p.dead ? -1 : (int)(p.row0 + (int64_t)s4[e] * p.Hkv + kvh);
          const uint32_t dst = smem_u32(mat ? vt_s : k_s) + (uint32_t)(b * KB + half * (PT_TOK * 128) + quad * 512);
          tma_gather4(dst, mat ? &tmv : &tmk, &kv_full[b], half * 64, r[0], r[1], r[2], r[3]);
        }
        if (it + 1 < n_t) load_slots(tile + 1);
      }
    }
  } else if (!TG && warp >= 4 && warp < 8) {
    // ------------------------------------------------------------------ producers: two groups of two warps, group gp
    // takes the tiles it = gp, gp + 2, ...: the gather latency of one group's tile hides under the other group's
    constexpr int CPT = PT_TOK * CPR / 64;      // chunks per thread per matrix
    const int gp = (warp - 4) >> 1, gw = (warp - 4) & 1, gtid = threadIdx.x - 128 - gp * 64;
    int sl[CPT];
    auto load_slots = [&](int tile) {
#pragma unroll
      for (int j = 0; j < CPT; ++j) {
        const int idx = tile * PT_TOK + (gtid + j * 64) / CPR;
        sl[j] = idx < lim ? (idx < n_cached ? p.live_slots[idx] : p.S[p.covered + (idx - n_cached)]) : p.dead;
      }
    };
    const uint32_t vd = smem_u32(vst_s) + (uint32_t)(gp * VSB);   // the group's staging buffer
    if (gp < n_t) load_slots(t_begin + gp);
    for (int it = gp; it < n_t; it += 2) {
      const int b = it % NB, tile = t_begin + it;
      mbar_wait(&kv_free[b], ((uint32_t)(it / NB) & 1u) ^ 1u);   // P V of tile it - 3 has completed
      const uint32_t kd = smem_u32(k_s) + (uint32_t)(b * KB);
#pragma unroll
      for (int j = 0; j < CPT; ++j) {
        const int c = gtid + j * 64, tok = c / CPR, ch = c % CPR;
        const bool live = sl[j] != p.dead;
        const int64_t off = ((int64_t)(live ? sl[j] : 0) * p.Hkv + kvh) * D + ch * 8;
        cp_async16_zfill(kd + (uint32_t)pt_entry(tok, ch, D), p.k_layer + off, live ? 16u : 0u);
        cp_async16_zfill(vd + (uint32_t)(tok * VST + ch * 16), p.v_layer + off, live ? 16u : 0u);
        if (ch == 0) {
          const int idx = tile * PT_TOK + tok;
          minrow_s[b * PT_TOK + tok] = !live ? INT_MAX : (idx < n_cached ? INT_MIN : p.covered + (idx - n_cached) - p.q_pos0);
        }
      }
      cp_async_commit();
      if (it + 2 < n_t) load_slots(tile + 2);
      cp_async_wait<0>();
      bar_sync(2 + gp, 64);   // every thread's copies of the tile have landed
      // V staging [item][d] -> V^T canonical [d][item]: ldmatrix.trans x4 = four 8 x 8 blocks (item groups tg0 .. tg0 + 3
      // of one d group); thread (r, q) receives items 2q, 2q + 1 of d = 8 dg + r and stores them as one 32-bit word
      unsigned char* vt = vt_s + (size_t)b * VTB;
      const int mi = lane >> 3, mr = lane & 7, r = lane >> 2, q4 = lane & 3;
      for (int blk = gw; blk < (D / 8) * 2; blk += 2) {
        const int dg = blk >> 1, tg0 = (blk & 1) * 4;
        uint32_t v0, v1, v2, v3;
        ldsm_x4_t(vd + (uint32_t)(((tg0 + mi) * 8 + mr) * VST + dg * 16), v0, v1, v2, v3);
        unsigned char* dst = vt + pt_entry(dg * 8 + r, tg0, PT_TOK) + q4 * 4;
        *reinterpret_cast<uint32_t*>(dst) = v0;
        *reinterpret_cast<uint32_t*>(dst + 128) = v1;
        *reinterpret_cast<uint32_t*>(dst + 256) = v2;
        *reinterpret_cast<uint32_t*>(dst + 384) = v3;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_arrive(&kv_full[b]);
      bar_sync(2 + gp, 64);   // the staging buffer is free for the group's next tile
    }
  } else if (warp == MMA_WARP) {
    // ------------------------------------------------------------------ MMA issuer (one thread)
    if (lane == 0 && n_t > 0) {
      const uint32_t ibase = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 4) << 24);
      const uint32_t idesc_s = ibase | (((uint32_t)PT_TOK >> 3) << 17), idesc_o = ibase | (((uint32_t)D >> 3) << 17);
      auto issue_s = [&](int it) {
        const int b = it & 1, kb = it % NB;
        mbar_wait(&kv_full[kb], (uint32_t)(it / NB) & 1u);
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
          mbar_wait(&s_free[mt * 2 + b], ((uint32_t)(it >> 1) & 1u) ^ 1u);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint64_t dq = umma_desc(smem_u32(q_s) + (uint32_t)(mt * QB), 128, SBO_D);
          const uint32_t td = tmem + (uint32_t)(mt * T_COLS + b * PT_TOK);
          if constexpr (TG) {
            const uint32_t ka = smem_u32(k_s) + (uint32_t)(kb * KB);
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks)
              umma_bf16(td, dq + (uint64_t)(ks * 16),
                        umma_desc_sw128(ka + (uint32_t)((ks >> 2) * (PT_TOK * 128) + (ks & 3) * 32), 16, 1024), idesc_s, ks ? 1u : 0u);
          } else {
            const uint64_t dk = umma_desc(smem_u32(k_s) + (uint32_t)(kb * KB), 128, SBO_D);
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) umma_bf16(td, dq + (uint64_t)(ks * 16), dk + (uint64_t)(ks * 16), idesc_s, ks ? 1u : 0u);
          }
          umma_commit(&s_full[mt * 2 + b]);
        }
      };
      mbar_wait(q_ready, 0u);
      issue_s(0);
      for (int it = 0; it < n_t; ++it) {
        if (it + 1 < n_t) issue_s(it + 1);      // S of the next tile runs under this tile's softmax
        const int pb = it % NPB;
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
          mbar_wait(&p_full[mt * NPB + pb], (uint32_t)(it / NPB) & 1u);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint64_t dp = umma_desc(smem_u32(p_s) + (uint32_t)((mt * NPB + pb) * PB), 128, SBO_T);
          const uint32_t td = tmem + (uint32_t)(mt * T_COLS) + O_COL;
          if constexpr (TG) {   // V [item][64 d] per column half: MN-major B, 16 items (two 8-row atoms) per instruction
            const uint32_t va = smem_u32(vt_s) + (uint32_t)((it % NB) * VTB);
#pragma unroll
            for (int ks = 0; ks < PT_TOK / 16; ++ks)
              umma_bf16(td, dp + (uint64_t)(ks * 16), umma_desc_sw128(va + (uint32_t)(ks * 2048), PT_TOK * 128, 1024),
                        idesc_o | (1u << 16), (it | ks) ? 1u : 0u);
          } else {
            const uint64_t dv = umma_desc(smem_u32(vt_s) + (uint32_t)((it % NB) * VTB), 128, SBO_T);
#pragma unroll
            for (int ks = 0; ks < PT_TOK / 16; ++ks)
              umma_bf16(td, dp + (uint64_t)(ks * 16), dv + (uint64_t)(ks * 16), idesc_o, (it | ks) ? 1u : 0u);
          }
          umma_commit(&p_free[mt * NPB + pb]);
        }
        umma_commit(&kv_free[it % NB]);
      }
    }
  } else {
    // ------------------------------------------------------------------ softmax warps: thread m = TMEM lane = M row
    // (warpgroup sg = M tile sg of the CTA)
    const int sg = MT == 1 ? 0 : warp >> 2, m = threadIdx.x & 127, i = m / G, g = m % G;
    const int row = (rb * MT + sg) * BR + i, head = kvh * G + g;
    const uint32_t tl = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(sg * T_COLS);
    unsigned char* q_m = q_s + sg * QB;
    uint64_t* s_full_m = s_full + sg * 2;
    uint64_t* s_free_m = s_free + sg * 2;
    uint64_t* p_full_m = p_full + sg * NPB;
    uint64_t* p_free_m = p_free + sg * NPB;
    {  // Q row of this thread into the canonical A operand
      const bf16* src = p.q + ((int64_t)row * Hq + head) * D;
#pragma unroll
      for (int k8 = 0; k8 < CPR; ++k8) {
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (row < p.n_q) v = *reinterpret_cast<const uint4*>(src + k8 * 8);
        *reinterpret_cast<uint4*>(q_m + pt_entry(m, k8, D)) = v;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_arrive(q_ready);
    }
    float m_ref = -CUDART_INF_F, l = 0.f;
    for (int it = 0; it < n_t; ++it) {
      const int b = it & 1;
      const uint32_t par = (uint32_t)(it >> 1) & 1u;
      const int kb = it % NB;
      mbar_wait(&kv_full[kb], (uint32_t)(it / NB) & 1u);   // minrow of the tile
      mbar_wait(&s_full_m[b], par);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      float x[PT_TOK];
#pragma unroll
      for (int c0 = 0; c0 < PT_TOK; c0 += 16) tmem_ld16(tl + (uint32_t)(b * PT_TOK + c0), &x[c0]);
      tmem_ld_wait();
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      mbar_arrive(&s_free_m[b]);
      float tmax = -CUDART_INF_F;
#pragma unroll
      for (int c = 0; c < PT_TOK; c += 4) {
        const int4 mr = *reinterpret_cast<const int4*>(&minrow_s[kb * PT_TOK + c]);
        x[c] = row >= mr.x ? x[c] * p.scale_log2 : -CUDART_INF_F;
        x[c + 1] = row >= mr.y ? x[c + 1] * p.scale_log2 : -CUDART_INF_F;
        x[c + 2] = row >= mr.z ? x[c + 2] * p.scale_log2 : -CUDART_INF_F;
        x[c + 3] = row >= mr.w ? x[c + 3] * p.scale_log2 : -CUDART_INF_F;
        tmax = fmaxf(fmaxf(tmax, fmaxf(x[c], x[c + 1])), fmaxf(x[c + 2], x[c + 3]));
      }
      // lazy reference: move it (and rescale the row's O and l) only when this tile exceeds it by more than 2^PT_GROW
      const bool grow = tmax > m_ref + PT_GROW;   // also the first finite maximum (m_ref = -inf)
      if (__any_sync(0xffffffffu, grow)) {
        const float m_new = grow ? tmax : m_ref;
        const float corr = (m_new == -CUDART_INF_F) ? 1.f : fast_exp2(m_ref - m_new);   // m_ref = -inf: 0
        if (it > 0) {   // O exists from the first P V on; wait for the previous tile's
          mbar_wait(&p_free_m[(it - 1) % NPB], (uint32_t)((it - 1) / NPB) & 1u);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
          for (int c0 = 0; c0 < D; c0 += 32) {
            float o[32];
            tmem_ld16(tl + O_COL + (uint32_t)c0, o);
            tmem_ld16(tl + O_COL + (uint32_t)c0 + 16, o + 16);
            tmem_ld_wait();
#pragma unroll
            for (int e = 0; e < 32; ++e) o[e] *= corr;
            tmem_st16(tl + O_COL + (uint32_t)c0, o);
            tmem_st16(tl + O_COL + (uint32_t)c0 + 16, o + 16);
          }
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
        l *= corr;
        m_ref = m_new;
      }
      const float ms = (m_ref == -CUDART_INF_F) ? 0.f : m_ref;
      float s0 = 0.f, s1 = 0.f;
#pragma unroll
      for (int c = 0; c < PT_TOK; c += 2) {
        x[c] = fast_exp2(x[c] - ms);
        x[c + 1] = fast_exp2(x[c + 1] - ms);
        s0 += x[c]; s1 += x[c + 1];
      }
      l += s0 + s1;
      const int pb = it % NPB;
      mbar_wait(&p_free_m[pb], ((uint32_t)(it / NPB) & 1u) ^ 1u);   // the P V that read this buffer has completed
      unsigned char* pd = p_s + (size_t)(sg * NPB + pb) * PB;
#pragma unroll
      for (int k8 = 0; k8 < PT_TOK / 8; ++k8) {
        const uint4 v = make_uint4(pack2_bf16(x[8 * k8], x[8 * k8 + 1]), pack2_bf16(x[8 * k8 + 2], x[8 * k8 + 3]),
                                   pack2_bf16(x[8 * k8 + 4], x[8 * k8 + 5]), pack2_bf16(x[8 * k8 + 6], x[8 * k8 + 7]));
        *reinterpret_cast<uint4*>(pd + pt_entry(m, k8, PT_TOK)) = v;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      mbar_arrive(&p_full_m[pb]);
    }
    // ---- partials of the split (an empty split writes m = -inf, l = 0: the scratch is not cleared)
    if (n_t > 0) {
      mbar_wait(&p_free_m[(n_t - 1) % NPB], (uint32_t)((n_t - 1) / NPB) & 1u);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    }
    const int64_t ph = ((int64_t)row * Hq + head) * p.n_split + split;
    const bool direct = p.out_direct != nullptr;   // one split: out = O / l, exactly what k_prefill_merge would compute
    if (row < p.n_q && !direct) p.part_ml[ph] = make_float2(m_ref, l);
#pragma unroll 1
    for (int c0 = 0; c0 < D; c0 += 16) {
      float o[16];
      if (n_t > 0) {
        tmem_ld16(tl + O_COL + (uint32_t)c0, o);
        tmem_ld_wait();
      } else {
#pragma unroll
        for (int e = 0; e < 16; ++e) o[e] = 0.f;
      }
      if (direct) {
        if (row < p.n_q) {
          uint32_t w[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) {
            const float a = l > 0.f ? o[2 * e] / l : 0.f, b = l > 0.f ? o[2 * e + 1] / l : 0.f;
            w[e] = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(a)) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(b)) << 16);
          }
          uint4* po = reinterpret_cast<uint4*>(p.out_direct + ((int64_t)row * Hq + head) * D + c0);
          po[0] = make_uint4(w[0], w[1], w[2], w[3]);
          po[1] = make_uint4(w[4], w[5], w[6], w[7]);
        }
      } else if (row < p.n_q) {
        float4* po = reinterpret_cast<float4*>(p.part_o + ph * D + c0);
        po[0] = make_float4(o[0], o[1], o[2], o[3]);     po[1] = make_float4(o[4], o[5], o[6], o[7]);
        po[2] = make_float4(o[8], o[9], o[10], o[11]);   po[3] = make_float4(o[12], o[13], o[14], o[15]);
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(MT * 256));
  }
}

}  // namespace ikv
