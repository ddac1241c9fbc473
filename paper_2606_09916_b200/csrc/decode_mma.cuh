// decode_mma.cuh -- bf16 paged GQA decode attention through the slot map, dead entries skipped
// (R16), split-K over the survivor list, for sm_100a.
//
// One CTA = (token split, request, group of <= 8 KV heads):
//   producer warp : per 16-token tile, one 1-D bulk copy (TMA unit) per token for the K row and one for the V row
//                   of the CTA's heads ([heads][D] bf16, 2 KB at Qwen3-8B shape) into an mbarrier ring.
//   consumer warps: warp w owns KV head w.  S^T = q K^T with the G query heads of the group as the (padded) M rows
//                   of mma.sync.m16n8k16 and 8 tokens as N (K fragments via ldmatrix), online softmax in fp32
//                   (exp2), O += P V with P re-used straight from the accumulator layout and V fragments via
//                   ldmatrix.trans.  With G = 4 the FMA pipe could not keep up with HBM (8 FMA per key/value
//                   element); the tensor pipe can.
// Partials (m, l, o) per (request, head, split) go to scratch; k_decode_merge4 combines them.  Both kernels use
// programmatic dependent launch: the next call's K/V prefetch overlaps this call's merge.
#pragma once
#include "common.cuh"
#include "decode.cuh"
#include "pipe.cuh"

namespace ikv {

constexpr int DM_TOK = 16;     // tokens per stage
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

template <int D, int G>
__global__ __launch_bounds__(DM_THREADS, 1) void k_decode_mma(const DecMmaParams p, const DecBatch batch) {
  constexpr int KS = D / 16, NO = D / 8;
  const int split = blockIdx.x, req = blockIdx.y, hg = blockIdx.z;
  const int Hkv = p.Hkv, Hq = Hkv * G;
  const int h0 = hg * DM_CWARPS;
  const int nh = min(DM_CWARPS, Hkv - h0);
  const int row_bytes = nh * D * 2;
  const int row_stride = row_bytes + DM_ROWPAD;
  const int kv_bytes = DM_TOK * row_stride;  // K part of a stage; V part follows
  const int stage_bytes = 2 * kv_bytes + 16;   // + validity mask word
  const int NS = p.n_stage;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* stage_base = smem_raw;
  uint64_t* full = (uint64_t*)(stage_base + (size_t)NS * stage_bytes);
  uint64_t* empty = full + NS;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], DM_CWARPS); }
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();

  // Programmatic dependent launch: this grid may start while the previous decode call (its split and merge grids,
  // the only kernels of the library that trigger their dependents early) is still running.  Everything READ here --
  // slot lists, K/V pools, q -- was produced by kernels that never trigger early, so it is complete at this point;
  // everything WRITTEN here (the partial buffers, which the previous merge may still be reading) is written only
  // after pdl_wait(), which the consumers execute just before their stores.
  const DecReq rq = batch.r[req];
  const int n_cached = rq.n_items;  // the list is padded with the dead slot up to n_items: no device-side length read
  const int total = n_cached + (rq.seq_len - rq.covered);
  const int n_gran = (total + DM_GRAN - 1) / DM_GRAN;
  const int begin = (int)(((int64_t)n_gran * split) / p.n_split) * DM_GRAN;
  const int end = min(total, (int)(((int64_t)n_gran * (split + 1)) / p.n_split) * DM_GRAN);
  const int n_tiles = (end > begin) ? (end - begin + DM_TOK - 1) / DM_TOK : 0;

  if (warp == DM_CWARPS) {
    // ------------------------------------------------------------------ producer
    // slots of 32 tokens (two tiles) per load, fetched two tiles ahead of their bulk copies
    auto slot_of = [&](int i) -> int {
      if (i >= end) return p.dead;
      return (i < n_cached) ? __ldg(rq.live_slots + i) : __ldg(rq.S + rq.covered + (i - n_cached));
    };
    int cur = slot_of(begin + lane), nxt = slot_of(begin + 32 + lane);
    for (int t = 0; t < n_tiles; ++t) {
      const int s = t % NS;
      const uint32_t ph = (uint32_t)(t / NS) & 1u;
      if (t > 0 && (t & 1) == 0) {
        cur = nxt;
        nxt = slot_of(begin + (t + 2) * DM_TOK + lane);
      }
      const int i = begin + t * DM_TOK + lane;
      const int slot = __shfl_sync(0xffffffffu, cur, (t & 1) * DM_TOK + (lane & (DM_TOK - 1)));
      const bool in_range = lane < DM_TOK && i < end;
      const bool copy = in_range;  // rows past the end are never copied; the consumers zero their V slices
      const uint32_t vmask = __ballot_sync(0xffffffffu, in_range && slot != p.dead);
      const uint32_t cmask = __ballot_sync(0xffffffffu, copy);
      unsigned char* sb = stage_base + (size_t)s * stage_bytes;
      if (lane == 0) {
        mbar_wait(&empty[s], ph ^ 1u);
        *reinterpret_cast<uint32_t*>(sb + 2 * kv_bytes) = vmask;
        mbar_arrive_expect_tx(&full[s], (uint32_t)(__popc(cmask) * 2 * row_bytes));
      }
      __syncwarp();
      if (copy) {
        const int64_t off = ((int64_t)slot * Hkv + h0) * D;
        bulk_g2s(sb + lane * row_stride, p.k_layer + off, (uint32_t)row_bytes, &full[s]);
        bulk_g2s(sb + kv_bytes + lane * row_stride, p.v_layer + off, (uint32_t)row_bytes, &full[s]);
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers
    const int r = lane >> 2, q4 = lane & 3;
    const int kvh = h0 + warp;
    const bool active = warp < nh;
    // A fragments of q (rows g = r < G; rows >= G are zero)
    uint32_t qa[KS][2];
#pragma unroll
    for (int s = 0; s < KS; ++s) { qa[s][0] = 0u; qa[s][1] = 0u; }
    if (active && r < G) {
      const uint32_t* qp = reinterpret_cast<const uint32_t*>(p.q + ((int64_t)req * Hq + kvh * G + r) * D);
#pragma unroll
      for (int s = 0; s < KS; ++s) {
        qa[s][0] = qp[8 * s + q4];
        qa[s][1] = qp[8 * s + 4 + q4];
      }
    }
    const float sc = p.sm_scale * 1.4426950408889634f;  // logits in log2 units
    float o[NO][4];
#pragma unroll
    for (int n = 0; n < NO; ++n) { o[n][0] = o[n][1] = o[n][2] = o[n][3] = 0.f; }
    float m = -CUDART_INF_F, lsum = 0.f;
    const uint32_t stage_u32 = smem_u32(stage_base);
    // per-lane ldmatrix row: matrix mi = lane/8, row lane%8
    const int mi = lane >> 3, mr = lane & 7;
    const uint32_t k_lane = (uint32_t)(mr * row_stride + warp * D * 2 + mi * 16);                       // + tok8*8 rows + 64*v
    const uint32_t v_lane = (uint32_t)(((mi & 1) * 8 + mr) * row_stride + warp * D * 2 + (mi >> 1) * 16);  // + 32*j

    for (int t = 0; t < n_tiles; ++t) {
      const int s = t % NS;
      const uint32_t ph = (uint32_t)(t / NS) & 1u;
      mbar_wait(&full[s], ph);
      if (active) {
        const uint32_t sb = stage_u32 + (uint32_t)(s * stage_bytes);
        const uint32_t vmask = *reinterpret_cast<const uint32_t*>(stage_base + (size_t)s * stage_bytes + 2 * kv_bytes);
        if (vmask != 0xffffu) {
          // ragged tile: V rows of masked tokens may hold stale or uninitialised bytes (0 x NaN = NaN): zero this
          // head's slice of them (D * 2 bytes = D / 8 lanes x 16 bytes per row, two rows per pass when D = 128)
          constexpr int LPRV = D / 8;
          for (int tok = lane / LPRV; tok < DM_TOK; tok += 32 / LPRV)
            if (!((vmask >> tok) & 1u))
              *reinterpret_cast<uint4*>(stage_base + (size_t)s * stage_bytes + kv_bytes + (size_t)tok * row_stride +
                                        warp * D * 2 + (lane % LPRV) * 16) = make_uint4(0u, 0u, 0u, 0u);
          __syncwarp();
        }
        // S^T tiles: [g][tokens 0-7], [g][tokens 8-15]
        float sacc[2][4];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
          sacc[nt][0] = sacc[nt][1] = sacc[nt][2] = sacc[nt][3] = 0.f;
#pragma unroll
          for (int v = 0; v < KS / 2; ++v) {
            uint32_t b0, b1, b2, b3;
            ldsm_x4(sb + k_lane + (uint32_t)(nt * 8 * row_stride + v * 64), b0, b1, b2, b3);
            mma_bf16_16816(sacc[nt], qa[2 * v][0], 0u, qa[2 * v][1], 0u, b0, b1);
            mma_bf16_16816(sacc[nt], qa[2 * v + 1][0], 0u, qa[2 * v + 1][1], 0u, b2, b3);
          }
        }
        // online softmax over the 16 tokens of row g = r
        float sv[4];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int tok = nt * 8 + 2 * q4 + e;
            sv[nt * 2 + e] = ((vmask >> tok) & 1u) ? sacc[nt][e] * sc : -CUDART_INF_F;
          }
        float tmax = fmaxf(fmaxf(sv[0], sv[1]), fmaxf(sv[2], sv[3]));
        tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
        tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
        const float mn = fmaxf(m, tmax);
        const float mref = (mn == -CUDART_INF_F) ? 0.f : mn;
        const float corr = fast_exp2(m - mref);
        float pv[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) pv[e] = fast_exp2(sv[e] - mref);
        lsum = lsum * corr + (pv[0] + pv[1] + pv[2] + pv[3]);
        m = mn;
        const uint32_t pa0 = pack2_bf16(pv[0], pv[1]), pa2 = pack2_bf16(pv[2], pv[3]);
#pragma unroll
        for (int n = 0; n < NO; ++n) { o[n][0] *= corr; o[n][1] *= corr; }
        // O += P V
#pragma unroll
        for (int j = 0; j < NO / 2; ++j) {
          uint32_t v0, v1, v2, v3;
          ldsm_x4_t(sb + (uint32_t)kv_bytes + v_lane + (uint32_t)(j * 32), v0, v1, v2, v3);
          mma_bf16_16816(o[2 * j], pa0, 0u, pa2, 0u, v0, v1);
          mma_bf16_16816(o[2 * j + 1], pa0, 0u, pa2, 0u, v2, v3);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
    }
    pdl_wait();
    if (active) {
      lsum += __shfl_xor_sync(0xffffffffu, lsum, 1);
      lsum += __shfl_xor_sync(0xffffffffu, lsum, 2);
      if (r < G) {
        const int64_t phd = ((int64_t)req * Hq + kvh * G + r) * p.n_split + split;
        float2* po = reinterpret_cast<float2*>(p.part_o + phd * D);
#pragma unroll
        for (int n = 0; n < NO; ++n) po[4 * n + q4] = make_float2(o[n][0], o[n][1]);
        if (q4 == 0) p.part_ml[phd] = make_float2(m * 0.6931471805599453f, lsum);
      }
    }
  }
}

inline size_t decode_mma_smem(int nh, int D, int max_smem, int* n_stage) {
  const size_t stage = 2 * (size_t)DM_TOK * (nh * D * 2 + DM_ROWPAD) + 16;
  const size_t fixed = 2 * 8 * 8 + 128;
  if (fixed + 2 * stage > (size_t)max_smem) { *n_stage = 0; return 0; }
  int ns = (int)(((size_t)max_smem - fixed) / stage);
  if (ns > 8) ns = 8;
  *n_stage = ns;
  return fixed + (size_t)ns * stage;
}

// grid = (H_q, n_req), block = DMG_THREADS.  Two phases with no serial dependency between splits:
//   1. m* = max_s m_s; w_s = exp(m_s - m*) (0 for empty splits) into shared memory; den = sum_s w_s l_s
//   2. thread (g, d) sums w_s o_s[d] over the splits s = g mod (threads / D) with independent loads; the groups
//      are combined through shared memory.
constexpr int DMG_THREADS = 512;
constexpr int DMG_MAX_SPLIT = 1024;
template <typename T, int D>
__global__ __launch_bounds__(DMG_THREADS) void k_decode_merge4(const float* __restrict__ part_o,
                                                               const float2* __restrict__ part_ml, int n_split,
                                                               T* __restrict__ out) {
  constexpr int NG = DMG_THREADS / D;
  __shared__ float ws[DMG_MAX_SPLIT];
  __shared__ float red[DMG_THREADS / 32];
  __shared__ float acc_s[NG][D];
  pdl_launch_dependents();
  pdl_wait();
  const int64_t ph = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * n_split;
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
