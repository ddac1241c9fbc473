// decode.cuh -- paged GQA decode attention through the slot map, dead entries skipped
// (R16).  Split-K over the survivor list + a merge kernel.
#pragma once
#include "common.cuh"

namespace ikv {

constexpr int DEC_MAX_REQ = 32;  // requests per launch (parameters travel by value)

struct DecReq {
  const int32_t* S;           // slot map
  const int32_t* live_slots;  // compact survivor list covering positions [0, covered)
  const int32_t* n_live;      // its length (device scalar)
  int seq_len, covered;
  int n_split;                // splits of this request (<= the launch's n_split, which is the scratch stride)
  int n_items;                // host-side upper bound of the list length; entries past *n_live hold the dead slot
  int flags;                  // IKV_REQ_* of the request
};
struct DecBatch {
  DecReq r[DEC_MAX_REQ];
};

template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<bf16>(bf16 v) { return __bfloat162float(v); }

// grid = (n_split, H_kv, n_req), block = 128 (4 warps).  A row of D elements is spread over LPR lanes
// (16-byte loads); each group of LPR lanes runs its own online softmax over its share of the tokens for the
// G query heads of this KV head; groups are merged through shared memory into one partial (m, l, o) per
// (request, head, split).
template <typename T, int D, int G>
__global__ __launch_bounds__(128) void k_decode_split(const T* __restrict__ k_layer, const T* __restrict__ v_layer,
                                                      int Hkv, int32_t dead, DecBatch batch,
                                                      const T* __restrict__ q, float sm_scale,
                                                      float* __restrict__ part_o, float2* __restrict__ part_ml,
                                                      int n_split) {
  constexpr int VEC = Elem<T>::VEC;
  constexpr int LPR = D / VEC;
  constexpr int RPW = 32 / LPR;
  constexpr int NGRP = 4 * RPW;  // softmax groups per CTA
  constexpr int UNR = 2;
  extern __shared__ float smem[];
  float* s_o = smem;                       // [NGRP][G][D]
  float* s_m = s_o + NGRP * G * D;         // [NGRP][G]
  float* s_l = s_m + NGRP * G;             // [NGRP][G]

  const int split = blockIdx.x, kvh = blockIdx.y, req = blockIdx.z;
  const int Hq = Hkv * G;
  const DecReq rq = batch.r[req];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int sub = lane % LPR, rw = lane / LPR;
  const int grp = warp * RPW + rw;

  const int n_cached = *rq.n_live;
  const int total = n_cached + (rq.seq_len - rq.covered);
  const int begin = (int)(((int64_t)total * split) / n_split);
  const int end = (int)(((int64_t)total * (split + 1)) / n_split);

  float qv[G][VEC];
#pragma unroll
  for (int g = 0; g < G; ++g)
#pragma unroll
    for (int i = 0; i < VEC; ++i)
      qv[g][i] = to_f32<T>(q[((int64_t)req * Hq + kvh * G + g) * D + sub * VEC + i]) * sm_scale;

  float m[G], l[G], o[G][VEC];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    m[g] = -CUDART_INF_F;
    l[g] = 0.f;
#pragma unroll
    for (int i = 0; i < VEC; ++i) o[g][i] = 0.f;
  }

  for (int i0 = begin; i0 < end; i0 += NGRP * UNR) {
    uint4 kr[UNR], vr[UNR];
    bool ok[UNR];
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      const int i = i0 + u * NGRP + grp;
      int slot = dead;
      if (i < end) slot = (i < n_cached) ? rq.live_slots[i] : rq.S[rq.covered + (i - n_cached)];
      ok[u] = (slot != dead);
      const int64_t off = ((int64_t)slot * Hkv + kvh) * D + sub * VEC;
      kr[u] = ld_stream16(k_layer + off);
      vr[u] = ld_stream16(v_layer + off);
    }
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      float k[VEC], v[VEC];
      Elem<T>::unpack(kr[u], k);
      Elem<T>::unpack(vr[u], v);
      float s[G];
#pragma unroll
      for (int g = 0; g < G; ++g) {
        s[g] = 0.f;
#pragma unroll
        for (int i = 0; i < VEC; ++i) s[g] = fmaf(k[i], qv[g][i], s[g]);
      }
#pragma unroll
      for (int g = 0; g < G; ++g)
#pragma unroll
        for (int x = LPR / 2; x > 0; x >>= 1) s[g] += __shfl_xor_sync(0xffffffffu, s[g], x);
      if (ok[u]) {
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const float mn = fmaxf(m[g], s[g]);
          const float corr = __expf(m[g] - mn);  // m = -inf on the first token -> 0
          const float pj = __expf(s[g] - mn);
          l[g] = l[g] * corr + pj;
#pragma unroll
          for (int i = 0; i < VEC; ++i) o[g][i] = fmaf(pj, v[i], o[g][i] * corr);
          m[g] = mn;
        }
      }
    }
  }

  // merge the NGRP groups
#pragma unroll
  for (int g = 0; g < G; ++g) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) s_o[(grp * G + g) * D + sub * VEC + i] = o[g][i];
    if (sub == 0) { s_m[grp * G + g] = m[g]; s_l[grp * G + g] = l[g]; }
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < G * D; idx += 128) {
    const int g = idx / D, d = idx % D;
    float mx = -CUDART_INF_F;
#pragma unroll
    for (int r = 0; r < NGRP; ++r) mx = fmaxf(mx, s_m[r * G + g]);
    float acc = 0.f, den = 0.f;
    if (mx > -CUDART_INF_F) {
#pragma unroll
      for (int r = 0; r < NGRP; ++r) {
        const float w = __expf(s_m[r * G + g] - mx);
        acc = fmaf(w, s_o[(r * G + g) * D + d], acc);
        den = fmaf(w, s_l[r * G + g], den);
      }
    }
    const int64_t ph = ((int64_t)req * Hq + kvh * G + g) * n_split + split;
    part_o[ph * D + d] = acc;
    if (d == 0) part_ml[ph] = make_float2(mx, den);
  }
}

}  // namespace ikv
