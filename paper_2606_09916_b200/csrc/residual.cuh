// residual.cuh -- residual head of Eq. 4-6, fp32 ("FP32 residual head").
// Topology per DESIGN.md R9-R12.  Weights are stored TRANSPOSED on the device ([in][out]) so that
// consecutive threads (output units) read consecutive addresses.
#pragma once
#include "common.cuh"

namespace ikv {

constexpr int R_DC = 128;   // d_c
constexpr int R_HC = 4;     // H_c
constexpr int R_DH = 32;    // d_c / H_c
constexpr int R_HID = 256;  // hidden width
constexpr int R_TOK = 16;   // candidates per CTA

struct ResidW {
  const float *wq_t, *bq, *wk_t, *bk, *wv_t, *bv, *fc1_t, *fc1_b, *fc2_w, *fc2_b;
  float alpha;  // already clipped to [-5,5]
};

// Kc = W_K K^q + b_K, Vc = W_V K^q + b_V   (Eq. 6).  grid = capacity of the list, block = 128.
__global__ void k_resid_kv(const float* __restrict__ kq, const int32_t* __restrict__ n_xq, int D, ResidW w,
                           float* __restrict__ kc, float* __restrict__ vc) {
  const int i = blockIdx.x, o = threadIdx.x;
  if (i >= *n_xq) return;
  float ak = w.bk[o], av = w.bv[o];
  for (int d = 0; d < D; ++d) {
    const float x = kq[(int64_t)i * D + d];
    ak = fmaf(w.wk_t[d * R_DC + o], x, ak);
    av = fmaf(w.wv_t[d * R_DC + o], x, av);
  }
  kc[(int64_t)i * R_DC + o] = ak;
  vc[(int64_t)i * R_DC + o] = av;
}

__device__ __forceinline__ float gelu_erf(float x) { return 0.5f * x * (1.f + erff(x * 0.70710678118654752f)); }

// One CTA of 256 threads scores R_TOK candidates:
//   phi = [kbar | mbar | kbar*mbar | rule]            (Eq. 5)
//   c   = 4-head cross-attention of W_Q phi over (Kc, Vc)   (Eq. 6)
//   z   = fc2(GELU(fc1(phi (+) c)));   s = rule + alpha z    (Eq. 4)
// x is staged in shared memory as [IN][R_TOK] so that a row is read with broadcast 16-byte loads.
template <int D>
__global__ __launch_bounds__(256) void k_residual(const float* __restrict__ rule_c, const float* __restrict__ kbar,
                                                  const float* __restrict__ mbar, const float* __restrict__ kc,
                                                  const float* __restrict__ vc, const int32_t* __restrict__ n_xq_p,
                                                  const int32_t* __restrict__ n_cand_p,
                                                  const int32_t* __restrict__ cand_pos, ResidW w, int use_xattn,
                                                  float* __restrict__ scores) {
  constexpr int P = 3 * D + 1, IN = P + R_DC, TOK = R_TOK;
  __shared__ __align__(16) float x[IN][TOK];
  __shared__ __align__(16) float qs[TOK][R_DC];  // Q projection (two half-sums, added in turn)
  __shared__ float zred[8][TOK];
  const int tid = threadIdx.x;
  const int nc = *n_cand_p;
  const int c0 = blockIdx.x * TOK;
  if (c0 >= nc) return;
  const int nvalid = min(TOK, nc - c0);

  for (int idx = tid; idx < D * TOK; idx += 256) {
    const int t = idx / D, d = idx % D;
    const float k = (t < nvalid) ? kbar[(int64_t)(c0 + t) * D + d] : 0.f;
    const float m = mbar[d];
    x[d][t] = k;
    x[D + d][t] = m;
    x[2 * D + d][t] = k * m;
  }
  if (tid < TOK) x[3 * D][tid] = (tid < nvalid) ? rule_c[c0 + tid] : 0.f;
  for (int idx = tid; idx < R_DC * TOK; idx += 256) x[P + idx / TOK][idx % TOK] = 0.f;
  __syncthreads();

  const int nq = use_xattn ? *n_xq_p : 0;
  if (nq > 0) {
    // Q = W_Q phi + b_Q : thread (o, half) sums half of the input range
    {
      const int o = tid & 127, half = tid >> 7;
      const int i0 = half ? (P + 1) / 2 : 0, i1 = half ? P : (P + 1) / 2;
      float acc[TOK];
#pragma unroll
      for (int t = 0; t < TOK; ++t) acc[t] = 0.f;
      for (int i = i0; i < i1; ++i) {
        const float wv = w.wq_t[i * R_DC + o];
        const float4* xr = reinterpret_cast<const float4*>(&x[i][0]);
#pragma unroll
        for (int t4 = 0; t4 < TOK / 4; ++t4) {
          const float4 v = xr[t4];
          acc[t4 * 4 + 0] = fmaf(wv, v.x, acc[t4 * 4 + 0]);
          acc[t4 * 4 + 1] = fmaf(wv, v.y, acc[t4 * 4 + 1]);
          acc[t4 * 4 + 2] = fmaf(wv, v.z, acc[t4 * 4 + 2]);
          acc[t4 * 4 + 3] = fmaf(wv, v.w, acc[t4 * 4 + 3]);
        }
      }
      if (half == 0) {
        const float b = w.bq[o];
#pragma unroll
        for (int t = 0; t < TOK; ++t) qs[t][o] = acc[t] + b;
      }
      __syncthreads();
      if (half == 1) {
#pragma unroll
        for (int t = 0; t < TOK; ++t) qs[t][o] += acc[t];
      }
    }
    __syncthreads();
    // cross attention: 4 threads per (token, head) pair; thread r takes keys i = r mod 4
    {
      const int pair = tid >> 2, r = tid & 3;
      const int t = pair / R_HC, hc = pair % R_HC;
      float q[R_DH];
#pragma unroll
      for (int e = 0; e < R_DH; ++e) q[e] = qs[t][hc * R_DH + e] * 0.17677669529663689f;
      float mx = -CUDART_INF_F;
      for (int i = r; i < nq; i += 4) {
        const float4* kr = reinterpret_cast<const float4*>(kc + (int64_t)i * R_DC + hc * R_DH);
        float dot = 0.f;
#pragma unroll
        for (int e4 = 0; e4 < R_DH / 4; ++e4) {
          const float4 k = kr[e4];
          dot = fmaf(q[e4 * 4], k.x, dot); dot = fmaf(q[e4 * 4 + 1], k.y, dot);
          dot = fmaf(q[e4 * 4 + 2], k.z, dot); dot = fmaf(q[e4 * 4 + 3], k.w, dot);
        }
        mx = fmaxf(mx, dot);
      }
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
      float acc[R_DH];
#pragma unroll
      for (int e = 0; e < R_DH; ++e) acc[e] = 0.f;
      float den = 0.f;
      for (int i = r; i < nq; i += 4) {
        const float4* kr = reinterpret_cast<const float4*>(kc + (int64_t)i * R_DC + hc * R_DH);
        const float4* vr = reinterpret_cast<const float4*>(vc + (int64_t)i * R_DC + hc * R_DH);
        float dot = 0.f;
#pragma unroll
        for (int e4 = 0; e4 < R_DH / 4; ++e4) {
          const float4 k = kr[e4];
          dot = fmaf(q[e4 * 4], k.x, dot); dot = fmaf(q[e4 * 4 + 1], k.y, dot);
          dot = fmaf(q[e4 * 4 + 2], k.z, dot); dot = fmaf(q[e4 * 4 + 3], k.w, dot);
        }
        const float p = expf(dot - mx);
        den += p;
#pragma unroll
        for (int e4 = 0; e4 < R_DH / 4; ++e4) {
          const float4 v = vr[e4];
          acc[e4 * 4] = fmaf(p, v.x, acc[e4 * 4]); acc[e4 * 4 + 1] = fmaf(p, v.y, acc[e4 * 4 + 1]);
          acc[e4 * 4 + 2] = fmaf(p, v.z, acc[e4 * 4 + 2]); acc[e4 * 4 + 3] = fmaf(p, v.w, acc[e4 * 4 + 3]);
        }
      }
      den += __shfl_xor_sync(0xffffffffu, den, 1);
      den += __shfl_xor_sync(0xffffffffu, den, 2);
#pragma unroll
      for (int e = 0; e < R_DH; ++e) {
        acc[e] += __shfl_xor_sync(0xffffffffu, acc[e], 1);
        acc[e] += __shfl_xor_sync(0xffffffffu, acc[e], 2);
      }
      const float inv = 1.f / den;
#pragma unroll
      for (int e = 0; e < R_DH; ++e)
        if ((e >> 3) == r) x[P + hc * R_DH + e][t] = acc[e] * inv;
    }
    __syncthreads();
  }

  // fc1 -> GELU -> fc2 : thread u owns hidden unit u
  {
    const int u = tid;
    float acc[TOK];
#pragma unroll
    for (int t = 0; t < TOK; ++t) acc[t] = 0.f;
    for (int i = 0; i < IN; ++i) {
      const float wv = w.fc1_t[i * R_HID + u];
      const float4* xr = reinterpret_cast<const float4*>(&x[i][0]);
#pragma unroll
      for (int t4 = 0; t4 < TOK / 4; ++t4) {
        const float4 v = xr[t4];
        acc[t4 * 4 + 0] = fmaf(wv, v.x, acc[t4 * 4 + 0]);
        acc[t4 * 4 + 1] = fmaf(wv, v.y, acc[t4 * 4 + 1]);
        acc[t4 * 4 + 2] = fmaf(wv, v.z, acc[t4 * 4 + 2]);
        acc[t4 * 4 + 3] = fmaf(wv, v.w, acc[t4 * 4 + 3]);
      }
    }
    const float b1 = w.fc1_b[u], w2 = w.fc2_w[u];
#pragma unroll
    for (int t = 0; t < TOK; ++t) {
      float hz = w2 * gelu_erf(acc[t] + b1);
      hz = warp_sum(hz);
      if ((tid & 31) == 0) zred[tid >> 5][t] = hz;
    }
  }
  __syncthreads();
  if (tid < nvalid) {
    float z = w.fc2_b[0];
#pragma unroll
    for (int wi = 0; wi < 8; ++wi) z += zred[wi][tid];
    scores[cand_pos[c0 + tid]] = x[3 * D][tid] + w.alpha * z;
  }
}

}  // namespace ikv
