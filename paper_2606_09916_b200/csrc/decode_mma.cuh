// decode_mma.cuh -- bf16 paged GQA decode attention through the slot map, dead entries skipped (
// DESIGN.md R16), split-K over the survivor list, for sm_100a.
//
// One CTA = (token split, request, group of <= 8 KV heads); producer warp + one consumer warp per KV head.
//   producer : slots of 32 tokens per load, two tiles ahead; per 16-token tile one 1-D bulk copy (TMA unit) per token
//              for the K rows into one half-stage of the ring and for the V rows into the next ([heads][D] bf16, 2 KB
//              at Qwen3-8B shape), each half-stage with its own mbarrier pair.
//   consumers: S = K q^T and O^T = V^T P with mma.sync.m16n8k16: the 16 tokens of the tile are the M rows of both
//              products and the G query heads of the group the (padded) N columns, so every accumulator register is
//              useful and O^T takes D/4 registers per thread.  K fragments via ldmatrix, V^T via ldmatrix.trans, P
//              from the accumulator layout to the B layout by one 8x8 movmatrix transpose per half tile; online
//              softmax per column in exp2 units, fp32.
// At ~95 registers and three 33 KB half-stages a CTA takes under half an SM: the CTAs of two consecutive layer calls
// co-reside, so the next call streams its K/V while this one computes, merges and drains (programmatic dependent
// launch).  Partials (m, l, o) per (request, head, split) go to scratch; k_decode_merge4 combines them.
#pragma once
#include "common.cuh"
#include "decode.cuh"
#include "pipe.cuh"

namespace ikv {

constexpr int DM_TOK = 16;     // tokens per tile (one K half-stage + one V half-stage)
constexpr int DM_GRAN = 8;     // split boundaries are multiples of this many tokens
constexpr int DM_CWARPS = 8;   // consumer warps = KV heads per CTA
constexpr int DM_THREADS = (DM_CWARPS + 1) * 32;
constexpr int DM_ROWPAD = 16;  // bytes: row stride = 16 (mod 128) keeps the 8-row ldmatrix reads conflict-free

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(addr));
}
__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack2_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

struct DecMmaParams {
  const bf16* k_layer;
  const bf16* v_layer;
  int Hkv;
  int32_t dead;
  const bf16* q;  // [n_req][Hq][D]
  float sm_scale;
  float* part_o;     // [n_req][Hq][n_split][D]
  float2* part_ml;   // [n_req][Hq][n_split]  (m in natural-log units, l)
  int n_split, n_stage;
};

__device__ __forceinline__ uint32_t movmatrix_t(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}

template <int D, int G>
__global__ __launch_bounds__(DM_THREADS, 2) void k_decode_mma(const DecMmaParams p, const DecBatch batch) {
  constexpr int KS = D / 16, MT = D / 16;
  const int split = blockIdx.x, req = blockIdx.y, hg = blockIdx.z;
  const int Hkv = p.Hkv, Hq = Hkv * G;
  const int h0 = hg * DM_CWARPS;
  const int nh = min(DM_CWARPS, Hkv - h0);
  const int row_bytes = nh * D * 2;
  const int row_stride = row_bytes + DM_ROWPAD;
  const int half_bytes = DM_TOK * row_stride;
  const int HS = p.n_stage;  // half-stages in the ring

  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* ring = smem_raw;
  uint64_t* full = (uint64_t*)(ring + (size_t)HS * half_bytes);
  uint64_t* empty = full + HS;
  uint32_t* vmasks = (uint32_t*)(empty + HS);  // [HS], written for K half-stages

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < HS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], DM_CWARPS); }
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();

  // Programmatic dependent launch: this grid may start while the preceding kernel of the stream is still running.
  // What is read BEFORE griddepcontrol.wait is only what cannot be that kernel's output: the survivor list (rewritten
  // only by ikv_select_evict / the rescan, after which the host launches this kernel without the programmatic attribute)
  // and the K/V rows of positions that list covers.  The caller's inputs of THIS call -- q, the slot-map tail and the K/V
  // rows of the appended positions -- are read after the wait, unless the request carries IKV_REQ_INPUTS_COMPLETE.
  // Everything WRITTEN here (the partial buffers, which the previous merge may still be reading) is written after it.
  const DecReq rq = batch.r[req];
  const int n_cached = rq.n_items;
  const int total = n_cached + (rq.seq_len - rq.covered);
  if (split >= rq.n_split) return;  // requests of a batch get splits in proportion to their length
  const int n_gran = (total + DM_GRAN - 1) / DM_GRAN;
  const int begin = (int)(((int64_t)n_gran * split) / rq.n_split) * DM_GRAN;
  const int end = min(total, (int)(((int64_t)n_gran * (split + 1)) / rq.n_split) * DM_GRAN);
  const int n_tiles = (end > begin) ? (end - begin + DM_TOK - 1) / DM_TOK : 0;

  if (warp == DM_CWARPS) {
    // ------------------------------------------------------------------ producer
    bool waited = (rq.flags & 2) != 0;  // IKV_REQ_INPUTS_COMPLETE
    auto slot_of = [&](int i0) -> int {  // slots i0 .. i0+31, one per lane (warp-uniform i0)
      if (!waited && i0 + 32 > n_cached && i0 < end) { pdl_wait(); waited = true; }  // the slot-map tail is a caller input
      const int i = i0 + lane;
      if (i >= end) return p.dead;
      return (i < n_cached) ? rq.live_slots[i] : rq.S[rq.covered + (i - n_cached)];
    };
    int cur = slot_of(begin), nxt = slot_of(begin + 32);
    int s = 0;
    uint32_t ph = 0;
    for (int t = 0; t < n_tiles; ++t) {
      if (t > 0 && (t & 1) == 0) {
        cur = nxt;
        nxt = slot_of(begin + (t + 2) * DM_TOK);
      }
      const int i = begin + t * DM_TOK + lane;
      const int slot = __shfl_sync(0xffffffffu, cur, (t & 1) * DM_TOK + (lane & (DM_TOK - 1)));
      const bool in_range = lane < DM_TOK && i < end;
      const uint32_t vmask = __ballot_sync(0xffffffffu, in_range && slot != p.dead);
      const uint32_t nrows = __popc(__ballot_sync(0xffffffffu, in_range));
      const int64_t off = ((int64_t)slot * Hkv + h0) * D;
#pragma unroll
      for (int kv = 0; kv < 2; ++kv) {
        if (lane == 0) {
          mbar_wait(&empty[s], ph ^ 1u);
          if (kv == 0) vmasks[s] = vmask;
          mbar_arrive_expect_tx(&full[s], nrows * (uint32_t)row_bytes);
        }
        __syncwarp();
        if (in_range)
          bulk_g2s(ring + (size_t)s * half_bytes + lane * row_stride, (kv == 0 ? p.k_layer : p.v_layer) + off,
                   (uint32_t)row_bytes, &full[s]);
        if (++s == HS) { s = 0; ph ^= 1u; }
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers
    const int r = lane >> 2, q4 = lane & 3;
    const int kvh = h0 + warp;
    const bool active = warp < nh;
    // B fragments of q^T: b0 = q[g = r][16 ks + 2 q4, +1], b1 = q[g = r][16 ks + 8 + 2 q4, +1]; rows g >= G are zero
    uint32_t qb[KS][2];
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) { qb[ks][0] = 0u; qb[ks][1] = 0u; }
    if (!(rq.flags & 2)) pdl_wait();  // q is a caller input of this call (IKV_REQ_INPUTS_COMPLETE: read it right away)
    if (active && r < G) {
      const uint32_t* qp = reinterpret_cast<const uint32_t*>(p.q + ((int64_t)req * Hq + kvh * G + r) * D);
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        qb[ks][0] = qp[8 * ks + q4];
        qb[ks][1] = qp[8 * ks + 4 + q4];
      }
    }
    const float sc = p.sm_scale * 1.4426950408889634f;  // logits in log2 units
    float o[MT][4];  // O^T: [d = 16 mt + r (+8)][g = 2 q4 (+1)]
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) { o[mt][0] = o[mt][1] = o[mt][2] = o[mt][3] = 0.f; }
    float m0 = -CUDART_INF_F, m1 = -CUDART_INF_F, l0 = 0.f, l1 = 0.f;  // columns g = 2 q4, 2 q4 + 1
    const uint32_t ring_u32 = smem_u32(ring);
    const int mi = lane >> 3, mr = lane & 7;
    // K as A (row-major tok x d): matrices (tok 0-7, d 0-7), (tok 8-15, d 0-7), (tok 0-7, d 8-15), (tok 8-15, d 8-15)
    const uint32_t k_lane = (uint32_t)(((mi & 1) * 8 + mr) * row_stride + warp * D * 2 + (mi >> 1) * 16);
    // V^T as A (d x tok) through ldmatrix.trans: (tok 0-7, d 0-7), (tok 0-7, d 8-15), (tok 8-15, d 0-7), (tok 8-15, d 8-15)
    const uint32_t v_lane = (uint32_t)(((mi >> 1) * 8 + mr) * row_stride + warp * D * 2 + (mi & 1) * 16);
    int s = 0;
    uint32_t ph = 0;

    for (int t = 0; t < n_tiles; ++t) {
      // ---- K half-stage: S = K q^T
      mbar_wait(&full[s], ph);
      float pv[4] = {0.f, 0.f, 0.f, 0.f};
      uint32_t vmask = 0;
      float c0 = 1.f, c1 = 1.f;
      if (active) {
        const uint32_t sb = ring_u32 + (uint32_t)(s * half_bytes);
        vmask = vmasks[s];
        float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb2[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int ks = 0; ks < KS; ks += 2) {
          uint32_t a0, a1, a2, a3;
          ldsm_x4(sb + k_lane + (uint32_t)(ks * 32), a0, a1, a2, a3);
          mma_bf16_16816(sa, a0, a1, a2, a3, qb[ks][0], qb[ks][1]);
          ldsm_x4(sb + k_lane + (uint32_t)((ks + 1) * 32), a0, a1, a2, a3);
          mma_bf16_16816(sb2, a0, a1, a2, a3, qb[ks + 1][0], qb[ks + 1][1]);
        }
        const bool v0 = (vmask >> r) & 1u, v1 = (vmask >> (r + 8)) & 1u;
        float x00 = v0 ? (sa[0] + sb2[0]) * sc : -CUDART_INF_F, x01 = v0 ? (sa[1] + sb2[1]) * sc : -CUDART_INF_F;
        float x10 = v1 ? (sa[2] + sb2[2]) * sc : -CUDART_INF_F, x11 = v1 ? (sa[3] + sb2[3]) * sc : -CUDART_INF_F;
        float t0m = fmaxf(x00, x10), t1m = fmaxf(x01, x11);
#pragma unroll
        for (int ofs = 4; ofs < 32; ofs <<= 1) {
          t0m = fmaxf(t0m, __shfl_xor_sync(0xffffffffu, t0m, ofs));
          t1m = fmaxf(t1m, __shfl_xor_sync(0xffffffffu, t1m, ofs));
        }
        const float n0 = fmaxf(m0, t0m), n1 = fmaxf(m1, t1m);
        const float r0 = (n0 == -CUDART_INF_F) ? 0.f : n0, r1 = (n1 == -CUDART_INF_F) ? 0.f : n1;
        c0 = fast_exp2(m0 - r0); c1 = fast_exp2(m1 - r1);
        pv[0] = fast_exp2(x00 - r0); pv[1] = fast_exp2(x01 - r1);
        pv[2] = fast_exp2(x10 - r0); pv[3] = fast_exp2(x11 - r1);
        l0 = l0 * c0 + (pv[0] + pv[2]);
        l1 = l1 * c1 + (pv[1] + pv[3]);
        m0 = n0; m1 = n1;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
      if (++s == HS) { s = 0; ph ^= 1u; }

      // ---- V half-stage: O^T += V^T P
      mbar_wait(&full[s], ph);
      if (active) {
        const uint32_t sb = ring_u32 + (uint32_t)(s * half_bytes);
        if (vmask != 0xffffu) {
          // ragged tile: V rows of masked tokens may hold stale or uninitialised bytes (0 x NaN = NaN): zero them
          constexpr int LPRV = D / 8;
          for (int tok = lane / LPRV; tok < DM_TOK; tok += 32 / LPRV)
            if (!((vmask >> tok) & 1u))
              *reinterpret_cast<uint4*>(ring + (size_t)s * half_bytes + (size_t)tok * row_stride + warp * D * 2 +
                                        (lane % LPRV) * 16) = make_uint4(0u, 0u, 0u, 0u);
          __syncwarp();
        }
        // P (C layout: [tok r | r+8][g 2q4, 2q4+1]) -> B fragments [k = tok][n = g] by an 8x8 transpose each
        const uint32_t b0 = movmatrix_t(pack2_bf16(pv[0], pv[1]));
        const uint32_t b1 = movmatrix_t(pack2_bf16(pv[2], pv[3]));
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
          o[mt][0] *= c0; o[mt][1] *= c1; o[mt][2] *= c0; o[mt][3] *= c1;
          uint32_t a0, a1, a2, a3;
          ldsm_x4_t(sb + v_lane + (uint32_t)(mt * 32), a0, a1, a2, a3);
          mma_bf16_16816(o[mt], a0, a1, a2, a3, b0, b1);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
      if (++s == HS) { s = 0; ph ^= 1u; }
    }
    pdl_wait();
    if (active) {
#pragma unroll
      for (int ofs = 4; ofs < 32; ofs <<= 1) {
        l0 += __shfl_xor_sync(0xffffffffu, l0, ofs);
        l1 += __shfl_xor_sync(0xffffffffu, l1, ofs);
      }
      const int g0 = 2 * q4, g1 = g0 + 1;
      const int64_t ph0 = ((int64_t)req * Hq + kvh * G + g0) * p.n_split + split;
      const int64_t ph1 = ((int64_t)req * Hq + kvh * G + g1) * p.n_split + split;
      if (g0 < G) {
        float* po = p.part_o + ph0 * D;
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) { po[mt * 16 + r] = o[mt][0]; po[mt * 16 + 8 + r] = o[mt][2]; }
        if (r == 0) p.part_ml[ph0] = make_float2(m0 * 0.6931471805599453f, l0);
      }
      if (g1 < G) {
        float* po = p.part_o + ph1 * D;
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) { po[mt * 16 + r] = o[mt][1]; po[mt * 16 + 8 + r] = o[mt][3]; }
        if (r == 0) p.part_ml[ph1] = make_float2(m1 * 0.6931471805599453f, l1);
      }
    }
  }
}

// shared memory of k_decode_mma for `n_half` half-stages
inline size_t decode_mma_smem(int nh, int D, int max_smem, int* n_half) {
  const size_t half = (size_t)DM_TOK * (nh * D * 2 + DM_ROWPAD);
  const size_t per = half + 2 * 8 + 4;
  const size_t fixed = 128;
  if (fixed + 2 * per > (size_t)max_smem) { *n_half = 0; return 0; }
  int n = (int)(((size_t)max_smem - fixed) / per);
  if (n > 12) n = 12;
  *n_half = n;
  return fixed + (size_t)n * per;
}

// grid = (H_q, n_req), block = DMG_THREADS.  Two phases with no serial dependency between splits:
//   1. m* = max_s m_s; w_s = exp(m_s - m*) (0 for empty splits) into shared memory; den = sum_s w_s l_s
//   2. thread (g, d) sums w_s o_s[d] over the splits s = g mod (threads / D) with independent loads; the groups
//      are combined through shared memory.
constexpr int DMG_THREADS = 512;
constexpr int DMG_MAX_SPLIT = 1024;
template <typename T, int D>
__global__ __launch_bounds__(DMG_THREADS) void k_decode_merge4(const float* __restrict__ part_o,
                                                               const float2* __restrict__ part_ml, int stride,
                                                               const DecBatch batch, T* __restrict__ out) {
  constexpr int NG = DMG_THREADS / D;
  __shared__ float ws[DMG_MAX_SPLIT];
  __shared__ float red[DMG_THREADS / 32];
  __shared__ float acc_s[NG][D];
  pdl_launch_dependents();
  pdl_wait();
  const int64_t ph = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * stride;
  const int n_split = batch.r[blockIdx.y].n_split;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  float2 ml[DMG_MAX_SPLIT / DMG_THREADS];
  float mx = -CUDART_INF_F;
#pragma unroll
  for (int i = 0; i < DMG_MAX_SPLIT / DMG_THREADS; ++i) {
    const int sp = tid + i * DMG_THREADS;
    ml[i] = (sp < n_split) ? part_ml[ph + sp] : make_float2(-CUDART_INF_F, 0.f);
    if (ml[i].y > 0.f) mx = fmaxf(mx, ml[i].x);
  }
  mx = warp_max(mx);
  if (lane == 0) red[warp] = mx;
  __syncthreads();
  mx = warp_max(lane < DMG_THREADS / 32 ? red[lane] : -CUDART_INF_F);
  __syncthreads();
  float den = 0.f;
#pragma unroll
  for (int i = 0; i < DMG_MAX_SPLIT / DMG_THREADS; ++i) {
    const int sp = tid + i * DMG_THREADS;
    const float w = (ml[i].y > 0.f) ? __expf(ml[i].x - mx) : 0.f;
    if (sp < n_split) ws[sp] = w;
    den = fmaf(w, ml[i].y, den);
  }
  den = warp_sum(den);
  if (lane == 0) red[warp] = den;
  __syncthreads();
  den = warp_sum(lane < DMG_THREADS / 32 ? red[lane] : 0.f);
  const int g = tid / D, d = tid % D;
  float acc = 0.f;
  const float* po = part_o + ph * D + d;
#pragma unroll 8
  for (int sp = g; sp < n_split; sp += NG) acc = fmaf(ws[sp], po[(int64_t)sp * D], acc);
  acc_s[g][d] = acc;
  __syncthreads();
  if (tid < D) {
    float a = 0.f;
#pragma unroll
    for (int i = 0; i < NG; ++i) a += acc_s[i][tid];
    const float inv = (den > 0.f) ? 1.f / den : 0.f;
    out[((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * D + tid] = (T)(a * inv);
  }
}

}  // namespace ikv
