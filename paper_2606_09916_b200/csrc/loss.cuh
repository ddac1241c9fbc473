// loss.cuh -- NEXT-4: the training objective of the residual head, Eq. 8, and dL/ds for one
// (session, turn) row of scores; readings R34-R37.  One CTA of 1,024 threads (n <= 131,072), every reduction a fixed
// tree: run-to-run deterministic.  Not a hot path: the point is the arithmetic on the GPU, next to the scores.
//   L = L_BCE + rho L_rank + gamma mean sigma(s) + eta mean_r (||row_r|| - 1)^2
#pragma once
#include "common.cuh"

namespace ikv {

constexpr int LOSS_MAX_N = 131072;
constexpr int LOSS_HN = 64;   // hard negatives of the rank term

struct LossParams {
  const float* s;         // [n] scores (logits)
  const int32_t* y;       // [n] 1 / 0 / anything else = excluded
  int n;
  const float* mem_rows;  // [n_rows][row_dim] or NULL
  int n_rows, row_dim;
  float rho, gamma, eta;
  float* terms;           // [5]: L, L_BCE, L_rank, keep, norm
  float* grad;            // [n]
};

__device__ __forceinline__ float softplus_f(float x) { return x > 0.f ? x + log1pf(expf(-x)) : log1pf(expf(x)); }
__device__ __forceinline__ float sigmoid_f(float x) { return x >= 0.f ? 1.f / (1.f + expf(-x)) : expf(x) / (1.f + expf(x)); }

// sum over the block, same value in every thread; red: 32 floats of shared memory
__device__ __forceinline__ float block_sum_1024(float v, float* red) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();   // red may still be read from the previous call
  if (lane == 0) red[warp] = v;
  __syncthreads();
  float t = red[lane];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  return t;
}

__global__ __launch_bounds__(1024) void k_train_loss(const LossParams p) {
  __shared__ float red[32];
  __shared__ float best_s[32];
  __shared__ int best_i[32];
  __shared__ float hn_s[LOSS_HN];
  __shared__ int hn_i[LOSS_HN];
  __shared__ float gh[LOSS_HN];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // ---- counts
  float nv = 0.f, np = 0.f;
  for (int i = tid; i < p.n; i += 1024) {
    const int y = p.y[i];
    if (y == 0 || y == 1) { nv += 1.f; np += (float)y; }
  }
  const float n_v = block_sum_1024(nv, red), n_p = block_sum_1024(np, red);
  float bce = 0.f, keep = 0.f, rank = 0.f;
  int n_h = 0;
  if (n_v > 0.f) {
    const float pr = n_p / n_v, pt = fminf(fmaxf(pr, 0.02f), 0.5f), wp = (1.f - pt) / pt;
    // ---- BCE and keep terms, their gradients
    for (int i = tid; i < p.n; i += 1024) {
      const int y = p.y[i];
      float g = 0.f;
      if (y == 0 || y == 1) {
        const float s = p.s[i], sg = sigmoid_f(s);
        if (y == 1) { bce += wp * softplus_f(-s); g = -wp * sigmoid_f(-s) / n_v; }
        else { bce += softplus_f(s); g = sg / n_v; }
        keep += sg;
        g += p.gamma * sg * (1.f - sg) / n_v;
      }
      p.grad[i] = g;
    }
    bce = block_sum_1024(bce, red) / n_v;
    keep = block_sum_1024(keep, red) / n_v;
    // ---- the 64 highest negatives, one per round: the largest (score, lower position first) below the previous pick
    float prev_s = CUDART_INF_F;
    int prev_i = -1;
    for (int k = 0; k < LOSS_HN; ++k) {
      float bs = -CUDART_INF_F;
      int bi = -1;
      for (int i = tid; i < p.n; i += 1024) {
        if (p.y[i] != 0) continue;
        const float s = p.s[i];
        const bool below = s < prev_s || (s == prev_s && i > prev_i);
        if (below && (bi < 0 || s > bs)) { bs = s; bi = i; }   // ascending i: the first of equal scores stays
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const float os = __shfl_xor_sync(0xffffffffu, bs, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (oi >= 0 && (bi < 0 || os > bs || (os == bs && oi < bi))) { bs = os; bi = oi; }
      }
      __syncthreads();
      if (lane == 0) { best_s[warp] = bs; best_i[warp] = bi; }
      __syncthreads();
      bs = best_s[lane]; bi = best_i[lane];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const float os = __shfl_xor_sync(0xffffffffu, bs, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (oi >= 0 && (bi < 0 || os > bs || (os == bs && oi < bi))) { bs = os; bi = oi; }
      }
      if (bi < 0) break;   // uniform: fewer than 64 negatives
      if (tid == 0) { hn_s[k] = bs; hn_i[k] = bi; }
      prev_s = bs; prev_i = bi;
      n_h = k + 1;
    }
    __syncthreads();
    // ---- rank term: every positive against the hard negatives
    if (n_p > 0.f && n_h > 0) {
      const float c = 1.f / (n_p * (float)n_h);
      for (int i = tid; i < p.n; i += 1024) {
        if (p.y[i] != 1) continue;
        const float s = p.s[i];
        float gi = 0.f;
        for (int k = 0; k < n_h; ++k) {
          const float z = hn_s[k] - s;
          rank += softplus_f(z);
          gi += sigmoid_f(z) * c * p.rho;
        }
        p.grad[i] -= gi;
      }
      rank = block_sum_1024(rank, red) * c;
      for (int k = 0; k < n_h; ++k) {   // gradient of hard negative k: the same pairs, summed over the positives
        float v = 0.f;
        for (int i = tid; i < p.n; i += 1024)
          if (p.y[i] == 1) v += sigmoid_f(hn_s[k] - p.s[i]) * c * p.rho;
        const float t = block_sum_1024(v, red);
        if (tid == 0) gh[k] = t;
      }
      __syncthreads();
      if (tid < n_h) p.grad[hn_i[tid]] += gh[tid];
    }
  } else {
    for (int i = tid; i < p.n; i += 1024) p.grad[i] = 0.f;
  }
  // ---- norm term: warp per row
  float nr = 0.f;
  for (int r = warp; r < p.n_rows; r += 32) {
    float q = 0.f;
    for (int d = lane; d < p.row_dim; d += 32) { const float v = p.mem_rows[(int64_t)r * p.row_dim + d]; q = fmaf(v, v, q); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) q += __shfl_xor_sync(0xffffffffu, q, o);
    const float e = sqrtf(q) - 1.f;
    if (lane == 0) nr += e * e;
  }
  float norm = block_sum_1024(nr, red);
  if (p.n_rows > 0) norm /= (float)p.n_rows;
  if (tid == 0) {
    p.terms[0] = bce + p.rho * rank + p.gamma * keep + p.eta * norm;
    p.terms[1] = bce; p.terms[2] = rank; p.terms[3] = keep; p.terms[4] = norm;
  }
}

}  // namespace ikv
