// prefill_mma.cuh -- NEXT-2: causal attention of a chunk of n_q query rows through the slot map ("after
// prefill", :163-175 KV-read metrics), dead entries skipped, bf16 pools.  Tiled: the K/V rows of the request are read
// once per 32-row block instead of once per row.
//
// Items of a request = the session's compact survivor list (positions < covered, all of them visible to every row of
// the chunk: the host makes covered <= q_pos0) followed by the positions [covered, q_pos0 + n_q) read through the slot
// map; the item of position pos is visible to chunk row i iff pos <= q_pos0 + i and its slot is not the dead slot.
// CTA = (split of the items, KV head, block of 32 rows), 2 G warps: warp (g, half) owns the m16 tile of rows
// 16 half .. 16 half + 15 of query head kvh G + g.  Per tile of 64 items: K and V rows of the head gathered with
// cp.async (16 bytes per thread, double-buffered, slots prefetched one tile further ahead), S = Q K^T on
// mma.sync.m16n8k16 (K fragments by ldmatrix), online softmax in the log2 domain on the accumulator layout, P cast to
// bf16 straight into A fragments, O += P V (V fragments by ldmatrix.trans).  Partials (m, l, O) per (row, head, split),
// merged by k_prefill_merge.
#pragma once
#include "decode_mma.cuh"
#include "score_rows_tc.cuh"

namespace ikv {

constexpr int PF_BR = 32;      // query rows per CTA
constexpr int PF_TOK = 64;     // items per tile
constexpr int PF_ROWPAD = 16;  // bytes: row stride = 16 (mod 128), conflict-free 8-row ldmatrix reads

struct PrefillParams {
  const bf16* k_layer;
  const bf16* v_layer;
  int Hkv;
  int32_t dead;
  const int32_t* S;           // slot map
  const int32_t* live_slots;  // survivor list of the positions [0, covered); entries past the live count hold the dead slot
  const int32_t* n_live;      // length of the list (device scalar)
  int n_cached, covered;      // host-side upper bound of that length, positions the list covers
  int q_pos0, n_q;
  const bf16* q;              // [n_q][Hq][D]
  float scale_log2;           // sm_scale * log2(e)
  float* part_o;              // [n_q][Hq][n_split][D]
  float2* part_ml;            // [n_q][Hq][n_split]: (m in log2 units, l)
  int n_split;
  int m_tiles;                // host only: 128-row tiles per CTA of k_prefill_tc (1 or 2)
  bf16* out_direct;           // k_prefill_tc with n_split = 1: the output itself ([n_q][Hq][D]); no partials, no merge
  int64_t row0;               // row of (layer, slot 0, KV head 0) in the pool seen as [rows][D] (tensor-map producers)
};

template <int D>
__host__ __device__ constexpr int pf_smem() { return 4 * PF_TOK * (D * 2 + PF_ROWPAD) + 2 * PF_TOK * 4; }

template <int D, int G>
__global__ __launch_bounds__(64 * G) void k_prefill_mma(const PrefillParams p) {
  constexpr int NT = 64 * G;                 // threads
  constexpr int CPR = D / 8;                 // 16-byte chunks per row
  constexpr int STRIDE = D * 2 + PF_ROWPAD;  // bytes per staged row
  constexpr int MAT = PF_TOK * STRIDE;       // bytes of a K (or V) tile
  constexpr int CPT = (PF_TOK * CPR + NT - 1) / NT;  // chunks per thread per matrix
  extern __shared__ __align__(128) unsigned char pf_smem_raw[];
  unsigned char* kv_s = pf_smem_raw;                                 // [2 stages][K | V][PF_TOK][STRIDE]
  int* minrow_s = reinterpret_cast<int*>(pf_smem_raw + 4 * MAT);     // [2][PF_TOK]: first chunk row that sees the item

  const int split = blockIdx.x, kvh = blockIdx.y, rb = blockIdx.z;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = warp >> 1, rh = warp & 1, r = lane >> 2, q4 = lane & 3;
  const int Hq = p.Hkv * G, head = kvh * G + g;
  const int row0 = rb * PF_BR + rh * 16 + r, row1 = row0 + 8;

  // items of this CTA: its share of the 64-item tiles, cut at the last item any row of the block can see.  The list
  // length is read on the device: the host's bound may be the whole prefix (entries past the length are dead padding)
  const int n_cached = min(p.n_cached, *p.n_live);
  const int total = n_cached + (p.q_pos0 + p.n_q - p.covered);
  const int lim = min(total, n_cached + (p.q_pos0 + min(p.n_q, (rb + 1) * PF_BR) - p.covered));
  const int tiles_all = (total + PF_TOK - 1) / PF_TOK;
  const int t_begin = (int)(((int64_t)tiles_all * split) / p.n_split);
  const int t_end = min((int)(((int64_t)tiles_all * (split + 1)) / p.n_split), (lim + PF_TOK - 1) / PF_TOK);

  // Q fragments of the warp's m16 tile, all k-steps
  uint32_t qa[D / 16][4];
  {
    const bf16* q0 = p.q + ((int64_t)row0 * Hq + head) * D + 2 * q4;
    const bf16* q1 = p.q + ((int64_t)row1 * Hq + head) * D + 2 * q4;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
      qa[ks][0] = row0 < p.n_q ? *reinterpret_cast<const uint32_t*>(q0 + ks * 16) : 0u;
      qa[ks][1] = row1 < p.n_q ? *reinterpret_cast<const uint32_t*>(q1 + ks * 16) : 0u;
      qa[ks][2] = row0 < p.n_q ? *reinterpret_cast<const uint32_t*>(q0 + ks * 16 + 8) : 0u;
      qa[ks][3] = row1 < p.n_q ? *reinterpret_cast<const uint32_t*>(q1 + ks * 16 + 8) : 0u;
    }
  }
  // loader state: the slots of this thread's chunks, one tile ahead of the copies
  int sl[CPT];
  auto load_slots = [&](int tile) {
#pragma unroll
    for (int j = 0; j < CPT; ++j) {
      const int c = tid + j * NT, idx = tile * PF_TOK + c / CPR;
      int s = p.dead;
      if (c < PF_TOK * CPR && idx < lim) s = idx < n_cached ? p.live_slots[idx] : p.S[p.covered + (idx - n_cached)];
      sl[j] = s;
    }
  };
  auto issue_tile = [&](int tile, int buf) {
    const uint32_t kb = smem_u32(kv_s) + (uint32_t)(buf * 2 * MAT);
#pragma unroll
    for (int j = 0; j < CPT; ++j) {
      const int c = tid + j * NT;
      if (c < PF_TOK * CPR) {
        const int tok = c / CPR, ch = c % CPR;
        const bool live = sl[j] != p.dead;
        const int64_t off = ((int64_t)(live ? sl[j] : 0) * p.Hkv + kvh) * D + ch * 8;
        const uint32_t dst = kb + (uint32_t)(tok * STRIDE + ch * 16);
        cp_async16_zfill(dst, p.k_layer + off, live ? 16u : 0u);         // dead / beyond the end: zero rows
        cp_async16_zfill(dst + MAT, p.v_layer + off, live ? 16u : 0u);
        if (ch == 0) {
          const int idx = tile * PF_TOK + tok;
          // cached items are visible to every row; a slot-map item at position pos from row pos - q_pos0 on
          minrow_s[buf * PF_TOK + tok] = !live ? INT_MAX : (idx < n_cached ? INT_MIN : p.covered + (idx - n_cached) - p.q_pos0);
        }
      }
    }
    cp_async_commit();
  };

  float oacc[D / 8][4];
#pragma unroll
  for (int i = 0; i < D / 8; ++i) oacc[i][0] = oacc[i][1] = oacc[i][2] = oacc[i][3] = 0.f;
  float m0 = -CUDART_INF_F, m1 = -CUDART_INF_F, l0 = 0.f, l1 = 0.f;  // l: this thread's share of the row sums

  if (t_begin < t_end) {
    load_slots(t_begin);
    issue_tile(t_begin, 0);
    if (t_begin + 1 < t_end) load_slots(t_begin + 1);
  }
  for (int tile = t_begin; tile < t_end; ++tile) {
    const int buf = (tile - t_begin) & 1;
    cp_async_wait<0>();
    __syncthreads();   // tile `tile` is in shared memory for everybody; everybody is done with the other buffer
    if (tile + 1 < t_end) {
      issue_tile(tile + 1, buf ^ 1);
      if (tile + 2 < t_end) load_slots(tile + 2);
    }
    const uint32_t kb = smem_u32(kv_s) + (uint32_t)(buf * 2 * MAT), vb = kb + MAT;
    // ---- S = Q K^T: 8 n-tiles of 8 items
    float sacc[PF_TOK / 8][4];
#pragma unroll
    for (int i = 0; i < PF_TOK / 8; ++i) sacc[i][0] = sacc[i][1] = sacc[i][2] = sacc[i][3] = 0.f;
    {
      // ldmatrix x4: (items 0-7, d 0-7), (items 0-7, d 8-15), (items 8-15, d 0-7), (items 8-15, d 8-15) of a 16 x 16 block
      const int mi = lane >> 3, mr = lane & 7;
      const uint32_t a0 = kb + (uint32_t)(((mi >> 1) * 8 + mr) * STRIDE + (mi & 1) * 16);
#pragma unroll
      for (int ks = 0; ks < D / 16; ++ks)
#pragma unroll
        for (int np = 0; np < PF_TOK / 16; ++np) {
          uint32_t b0, b1, b2, b3;
          ldsm_x4(a0 + (uint32_t)(np * 16 * STRIDE + ks * 32), b0, b1, b2, b3);
          mma_bf16_16816(sacc[2 * np], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b0, b1);
          mma_bf16_16816(sacc[2 * np + 1], qa[ks][0], qa[ks][1], qa[ks][2], qa[ks][3], b2, b3);
        }
    }
    // ---- mask, online softmax (log2 domain); thread: rows row0 / row1, items 8 nt + 2 q4 + {0, 1}
    float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
#pragma unroll
    for (int nt = 0; nt < PF_TOK / 8; ++nt) {
      const int2 mr2 = *reinterpret_cast<const int2*>(&minrow_s[buf * PF_TOK + nt * 8 + 2 * q4]);
      sacc[nt][0] = row0 >= mr2.x ? sacc[nt][0] * p.scale_log2 : -CUDART_INF_F;
      sacc[nt][1] = row0 >= mr2.y ? sacc[nt][1] * p.scale_log2 : -CUDART_INF_F;
      sacc[nt][2] = row1 >= mr2.x ? sacc[nt][2] * p.scale_log2 : -CUDART_INF_F;
      sacc[nt][3] = row1 >= mr2.y ? sacc[nt][3] * p.scale_log2 : -CUDART_INF_F;
      mx0 = fmaxf(mx0, fmaxf(sacc[nt][0], sacc[nt][1]));
      mx1 = fmaxf(mx1, fmaxf(sacc[nt][2], sacc[nt][3]));
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
    const float ms0 = mn0 == -CUDART_INF_F ? 0.f : mn0, ms1 = mn1 == -CUDART_INF_F ? 0.f : mn1;  // nothing seen yet
    const float c0 = fast_exp2(m0 - ms0), c1 = fast_exp2(m1 - ms1);                               // exp2(-inf) = 0
    m0 = mn0; m1 = mn1;
    float s0 = 0.f, s1 = 0.f;
#pragma unroll
    for (int nt = 0; nt < PF_TOK / 8; ++nt) {
      sacc[nt][0] = fast_exp2(sacc[nt][0] - ms0);
      sacc[nt][1] = fast_exp2(sacc[nt][1] - ms0);
      sacc[nt][2] = fast_exp2(sacc[nt][2] - ms1);
      sacc[nt][3] = fast_exp2(sacc[nt][3] - ms1);
      s0 += sacc[nt][0] + sacc[nt][1];
      s1 += sacc[nt][2] + sacc[nt][3];
    }
    l0 = l0 * c0 + s0;
    l1 = l1 * c1 + s1;
#pragma unroll
    for (int i = 0; i < D / 8; ++i) { oacc[i][0] *= c0; oacc[i][1] *= c0; oacc[i][2] *= c1; oacc[i][3] *= c1; }
    // ---- O += P V: P from the accumulator layout straight into A fragments (k = items)
    {
      // ldmatrix.trans x4: (items 0-7, d 0-7), (items 8-15, d 0-7), (items 0-7, d 8-15), (items 8-15, d 8-15)
      const int mi = lane >> 3, mr = lane & 7;
      const uint32_t a0 = vb + (uint32_t)(((mi & 1) * 8 + mr) * STRIDE + (mi >> 1) * 16);
#pragma unroll
      for (int ks = 0; ks < PF_TOK / 16; ++ks) {
        const uint32_t pa0 = pack2_bf16(sacc[2 * ks][0], sacc[2 * ks][1]), pa1 = pack2_bf16(sacc[2 * ks][2], sacc[2 * ks][3]);
        const uint32_t pa2 = pack2_bf16(sacc[2 * ks + 1][0], sacc[2 * ks + 1][1]);
        const uint32_t pa3 = pack2_bf16(sacc[2 * ks + 1][2], sacc[2 * ks + 1][3]);
#pragma unroll
        for (int dp = 0; dp < D / 16; ++dp) {
          uint32_t b0, b1, b2, b3;
          ldsm_x4_t(a0 + (uint32_t)(ks * 16 * STRIDE + dp * 32), b0, b1, b2, b3);
          mma_bf16_16816(oacc[2 * dp], pa0, pa1, pa2, pa3, b0, b1);
          mma_bf16_16816(oacc[2 * dp + 1], pa0, pa1, pa2, pa3, b2, b3);
        }
      }
    }
  }
  // ---- partials of the split (an empty split writes m = -inf, l = 0: the scratch is not cleared)
  l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
  l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
  l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int row = h ? row1 : row0;
    if (row < p.n_q) {
      const int64_t ph = ((int64_t)row * Hq + head) * p.n_split + split;
      if (q4 == 0) p.part_ml[ph] = make_float2(h ? m1 : m0, h ? l1 : l0);
      float* po = p.part_o + ph * D + 2 * q4;
#pragma unroll
      for (int i = 0; i < D / 8; ++i)
        *reinterpret_cast<float2*>(po + i * 8) = make_float2(oacc[i][2 * h], oacc[i][2 * h + 1]);
    }
  }
}

// out[row][head][:] = sum_s 2^(m_s - m) O_s / sum_s 2^(m_s - m) l_s; a row that sees nothing gives zeros (as the decode
// merge does).  grid (Hq, n_q), D threads.
template <int D>
__global__ __launch_bounds__(D) void k_prefill_merge(const float* __restrict__ part_o, const float2* __restrict__ part_ml,
                                                     int n_split, bf16* __restrict__ out) {
  const int64_t ph = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * n_split;
  pdl_wait();   // launched programmatically behind the split kernel: its partials are complete from here on
  float m = -CUDART_INF_F;
  for (int s = 0; s < n_split; ++s) {
    const float2 ml = part_ml[ph + s];
    if (ml.y > 0.f) m = fmaxf(m, ml.x);
  }
  float den = 0.f, acc = 0.f;
  for (int s = 0; s < n_split; ++s) {
    const float2 ml = part_ml[ph + s];
    if (ml.y > 0.f) {
      const float w = fast_exp2(ml.x - m);
      den = fmaf(w, ml.y, den);
      acc = fmaf(w, part_o[(ph + s) * D + threadIdx.x], acc);
    }
  }
  out[((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * D + threadIdx.x] = __float2bfloat16_rn(den > 0.f ? acc / den : 0.f);
}

}  // namespace ikv
