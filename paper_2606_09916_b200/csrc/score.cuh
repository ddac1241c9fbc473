// score.cuh -- QueryMemory update and the rule-score key pass (Eq. 2-3; k_bar of Eq. 5).
#pragma once
#include "common.cuh"

namespace ikv {

// ---------------------------------------------------------------------------------------------
// a0  M <- normalize(e^{-lambda} M + Enc),  Enc = mean of n query rows      (Eq. 2)
// grid = L*Hq, block = D threads.  qenc <- normalize(Enc) (IKV_MODE_QUERY).
// ---------------------------------------------------------------------------------------------
template <typename TQ>
__global__ void k_memory_update(float* __restrict__ M, float* __restrict__ qenc, const TQ* __restrict__ q_rows,
                                int n, int64_t row_stride /* L*Hq*D */, int D, float decay) {
  __shared__ float red[2][4];
  const int lh = blockIdx.x, d = threadIdx.x;
  const int64_t off = (int64_t)lh * D + d;
  float enc = 0.f;
  for (int r = 0; r < n; ++r) enc += (float)q_rows[(int64_t)r * row_stride + off];
  enc /= (float)n;
  const float m = decay * M[off] + enc;
  float s0 = warp_sum(m * m), s1 = warp_sum(enc * enc);
  if ((d & 31) == 0) { red[0][d >> 5] = s0; red[1][d >> 5] = s1; }
  __syncthreads();
  float t0 = 0.f, t1 = 0.f;
  for (int w = 0; w < (D + 31) / 32; ++w) { t0 += red[0][w]; t1 += red[1][w]; }
  M[off] = m / fmaxf(sqrtf(t0), 1e-12f);
  qenc[off] = enc / fmaxf(sqrtf(t1), 1e-12f);
}

// ---------------------------------------------------------------------------------------------
// a1  partition: one CTA of 1024 threads per request.  Writes the score
// fillers (R6), zeroes rule_out, and compacts the candidates in ascending position:
// cand_pos[c], cand_slot[c], *n_cand.
// ---------------------------------------------------------------------------------------------
__global__ __launch_bounds__(1024) void k_partition(const int32_t* __restrict__ S, int N, int32_t dead, int pi,
                                                    int qs, int qe, float* __restrict__ scores,
                                                    float* __restrict__ rule_out, int32_t* __restrict__ cand_pos,
                                                    int32_t* __restrict__ cand_slot, int32_t* __restrict__ n_cand) {
  __shared__ int warp_tot[32];
  int base = 0;
  for (int j0 = 0; j0 < N; j0 += 1024) {
    const int j = j0 + threadIdx.x;
    int slot = dead, cls = CLS_DEAD;
    if (j < N) {
      slot = S[j];
      cls = classify(slot, j, dead, pi, qs, qe);
      if (cls != CLS_CAND) scores[j] = (cls == CLS_FORCED) ? CUDART_INF_F : -CUDART_INF_F;
      if (rule_out) rule_out[j] = 0.f;
    }
    int tot;
    const int ex = block_excl_scan_1024(cls == CLS_CAND ? 1 : 0, warp_tot, &tot);
    if (cls == CLS_CAND) {
      cand_pos[base + ex] = j;
      cand_slot[base + ex] = slot;
    }
    base += tot;
  }
  if (threadIdx.x == 0) *n_cand = base;
}

// ---------------------------------------------------------------------------------------------
// a2 (+a4)  logit pass: x[l,h,c] = <M[l,h], K[l, h div G, slot_c]> / sqrt(D)
// One CTA (256 threads, 8 warps) owns a tile of TILE candidates and loops over all layers.
// Warp w handles KV heads w, w+8, ...; a row of D elements is spread over LPR = D/VEC lanes
// (16-byte loads), RPW = 32/LPR rows per warp instruction.  Per layer the tile's logits are
// staged in shared memory, written out coalesced, and reduced to one (max, sum-exp) pair per head.
// KBAR: also accumulates sum_{l,kvh} K[l,kvh,slot] per token (mean key of Eq. 5).
// ---------------------------------------------------------------------------------------------
constexpr int SCORE_TILE = 64;

template <typename T, int D, int G, bool KBAR>
__global__ __launch_bounds__(256) void k_score_logits(
    const T* __restrict__ k_pool, int64_t layer_stride, int L, int Hkv, const float* __restrict__ M,
    const int32_t* __restrict__ cand_slot, const int32_t* __restrict__ n_cand_p, int32_t dead,
    float* __restrict__ logits, int64_t ldc, float2* __restrict__ partials, int n_tiles,
    float* __restrict__ kbar, float inv_sqrt_d) {
  constexpr int VEC = Elem<T>::VEC;
  constexpr int LPR = D / VEC;   // lanes per row
  constexpr int RPW = 32 / LPR;  // rows per warp instruction
  constexpr int TILE = SCORE_TILE;
  constexpr int UNR = 4;
  static_assert(TILE % (RPW * UNR) == 0, "tile / unroll mismatch");
  const int Hq = Hkv * G;
  extern __shared__ float smem[];
  float* xs = smem;                                  // [Hq][TILE+1]
  int32_t* slots = (int32_t*)(xs + Hq * (TILE + 1)); // [TILE]
  float* kb = (float*)(slots + TILE);                // [TILE][D] if KBAR

  const int tile = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int sub = lane % LPR, rw = lane / LPR;
  const int nc = *n_cand_p;
  const int c0 = tile * TILE;
  const int nvalid = min(TILE, nc - c0);  // may be <= 0
  if (threadIdx.x < TILE) slots[threadIdx.x] = (threadIdx.x < nvalid) ? cand_slot[c0 + threadIdx.x] : dead;
  if (KBAR)
    for (int i = threadIdx.x; i < TILE * D; i += 256) kb[i] = 0.f;
  __syncthreads();

  for (int l = 0; l < L; ++l) {
    const T* kl = k_pool + (int64_t)l * layer_stride;
    if (nvalid > 0) {
      for (int kvh = warp; kvh < Hkv; kvh += 8) {
        float m[G][VEC];
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
          for (int i = 0; i < VEC; ++i)
            m[g][i] = M[((int64_t)l * Hq + kvh * G + g) * D + sub * VEC + i] * inv_sqrt_d;
        for (int t0 = 0; t0 < TILE; t0 += RPW * UNR) {
          uint4 raw[UNR];
#pragma unroll
          for (int u = 0; u < UNR; ++u) {
            const int t = t0 + u * RPW + rw;
            raw[u] = ld_stream16(kl + ((int64_t)slots[t] * Hkv + kvh) * D + sub * VEC);
          }
#pragma unroll
          for (int u = 0; u < UNR; ++u) {
            const int t = t0 + u * RPW + rw;
            float k[VEC];
            Elem<T>::unpack(raw[u], k);
            float acc[G];
#pragma unroll
            for (int g = 0; g < G; ++g) {
              acc[g] = 0.f;
#pragma unroll
              for (int i = 0; i < VEC; ++i) acc[g] = fmaf(k[i], m[g][i], acc[g]);
            }
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
              for (int o = LPR / 2; o > 0; o >>= 1) acc[g] += __shfl_xor_sync(0xffffffffu, acc[g], o);
#pragma unroll
            for (int g = 0; g < G; ++g)
              if (sub == (g % LPR)) xs[(kvh * G + g) * (TILE + 1) + t] = acc[g];
            if (KBAR && t < nvalid) {
#pragma unroll
              for (int i = 0; i < VEC; ++i) atomicAdd(&kb[t * D + sub * VEC + i], k[i]);
            }
          }
        }
      }
    }
    __syncthreads();
    // per-head tile reduction and coalesced write-out
    for (int h = warp; h < Hq; h += 8) {
      float mx = -CUDART_INF_F;
      float v[TILE / 32];
#pragma unroll
      for (int r = 0; r < TILE / 32; ++r) {
        const int t = lane + 32 * r;
        v[r] = (t < nvalid) ? xs[h * (TILE + 1) + t] : -CUDART_INF_F;
        mx = fmaxf(mx, v[r]);
      }
      mx = warp_max(mx);
      float s = 0.f;
#pragma unroll
      for (int r = 0; r < TILE / 32; ++r) {
        const int t = lane + 32 * r;
        if (t < nvalid) {
          s += expf(v[r] - mx);
          logits[((int64_t)l * Hq + h) * ldc + c0 + t] = v[r];
        }
      }
      s = warp_sum(s);
      if (lane == 0) partials[((int64_t)l * Hq + h) * n_tiles + tile] = make_float2(mx, s);
    }
    __syncthreads();
  }
  if (KBAR) {
    const float inv = 1.f / (float)(L * Hkv);
    for (int i = threadIdx.x; i < nvalid * D; i += 256) kbar[(int64_t)c0 * D + i] = kb[i] * inv;
  }
}

// live cross-attention positions ("positions evicted in a prior round are excluded"):
// compacts the slots of the live entries of xattn_pos (or of [qs,qe) when xattn_pos == NULL).  1 CTA of 1024.
__global__ __launch_bounds__(1024) void k_xattn_compact(const int32_t* __restrict__ S, int N, int32_t dead,
                                                        const int32_t* __restrict__ xattn_pos, int n_x, int qs,
                                                        int32_t* __restrict__ xq_slot, int32_t* __restrict__ n_xq) {
  __shared__ int warp_tot[32];
  int base = 0;
  for (int i0 = 0; i0 < n_x; i0 += 1024) {
    const int i = i0 + threadIdx.x;
    int slot = dead;
    if (i < n_x) {
      const int pos = xattn_pos ? xattn_pos[i] : qs + i;
      if (pos >= 0 && pos < N) slot = S[pos];
    }
    int tot;
    const int ex = block_excl_scan_1024(slot != dead ? 1 : 0, warp_tot, &tot);
    if (slot != dead) xq_slot[base + ex] = slot;
    base += tot;
  }
  if (threadIdx.x == 0) *n_xq = base;
}

// K^q rows: mean over layers and KV heads of the keys at the listed slots (R8).  grid = n_x, block = D.
template <typename T>
__global__ void k_mean_key_list(const T* __restrict__ k_pool, int64_t layer_stride, int L, int Hkv, int D,
                                const int32_t* __restrict__ xq_slot, const int32_t* __restrict__ n_xq,
                                float* __restrict__ kq) {
  const int i = blockIdx.x;
  if (i >= *n_xq) return;
  const int64_t slot = xq_slot[i];
  float acc = 0.f;
  for (int l = 0; l < L; ++l)
    for (int h = 0; h < Hkv; ++h)
      acc += (float)k_pool[(int64_t)l * layer_stride + (slot * Hkv + h) * D + threadIdx.x];
  kq[(int64_t)i * D + threadIdx.x] = acc / (float)(L * Hkv);
}

}  // namespace ikv
