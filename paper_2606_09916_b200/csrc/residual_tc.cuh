// residual_tc.cuh -- the residual head of Eq. 4-6 as two dense tcgen05 contractions per 128-token
// tile, for calls with at most RT_NXMAX live cross-attention positions (the actionable span is 64 tokens; longer
// lists take k_residual_mma).  Topology per DESIGN.md R9-R12; every GEMM operand is a bf16 hi + bf16 lo pair and each
// product is hi*hi + lo*hi + hi*lo with fp32 accumulation in TMEM ("FP32 residual head").
//
// Folding.  mbar and K^q are constant over the call (n_x live query positions), hence
//   S[j, (h,i)] = Q_{j,h} . Kc_{i,h} / sqrt(32) = kbar_j . W_S[:, (h,i)] + rule_j s_r[(h,i)] + s_b[(h,i)]
//       W_S[:, (h,i)] = W_Q'_h^T Kc_{i,h},  s_r = w_qr,h . Kc_{i,h},  s_b = b_Q',h . Kc_{i,h}      (all x log2(e)/sqrt(32))
//   fc1(phi_j (+) c_j) = W_1k' kbar_j + sum_{h,i} P[j,(h,i)] U[(h,i), :] + rule_j w_r + b_1',   U[(h,i), :] = W_1c,h Vc_{i,h}
// with W_Q' = W_Qk + W_Qkm diag(mbar), b_Q' = b_Q + W_Qm mbar (same for fc1), P = per-head softmax of S over i.
// The head is then  S = kbar W_S  (128 x 4n_x x D)  and  hid = [kbar | P] [W_1k' ; U]  (128 x 256 x (D + 4n_x)).
//
// Kernel: warp 8 = MMA issuer, warp 9 = bulk-copy chunk loader (one elected thread each), warps 0-7 = tile loader,
// softmax and epilogue.
//   A operand  [kbar | P] in shared memory, canonical K-major layout (8 x 16-byte core matrices), hi and lo parts;
//   B operand  streamed in chunks of [N <= 256 rows x 16 k] (hi 8 KB | lo 8 KB) through a 5-stage bulk-copy ring;
//   TMEM       columns [0, 4 n_x) = S, [256, 512) = fc1 accumulator; tcgen05.ld.32x32b hands every thread its own token
//              row, so the four per-head softmaxes are thread-local.
// fc1's kbar chunks are multiplied while the softmax warps work; P of heads 2, 3 reuses the kbar rows' shared memory
// once those MMAs have completed.
#pragma once
#include "residual_mma.cuh"

namespace ikv {

constexpr int RT_M = 128;            // tokens per CTA
constexpr int RT_NXMAX = 64;         // live query positions taken by this kernel (4 * 64 = 256 S columns)
constexpr int RT_PART = 8192;        // bytes of one part (hi or lo) of a chunk: 256 rows x 16 k bf16
constexpr int RT_CHUNK = 2 * RT_PART;
constexpr int RT_STAGES = 5;
constexpr int RT_THREADS = 10 * 32;  // 8 compute warps, MMA issuer, chunk loader
constexpr int RT_P01 = 2 * 512 * RT_NXMAX;  // bytes of P of two heads (hi | lo each)
constexpr float RT_NEG = -1.0e30f;   // logit of a padded key column

template <int D>
__host__ __device__ constexpr int rt_region0() { return (512 * D > RT_P01) ? 512 * D : RT_P01; }
template <int D>
__host__ __device__ constexpr int rt_smem() { return rt_region0<D>() + RT_P01 + RT_STAGES * RT_CHUNK + (5 * 256 + 2 * 128 + 128) * 4 + 256; }
// chunk order in `wcan`: D/16 S chunks (k-steps of W_S) | D/16 fc1 kbar chunks | nxp/4 fc1 P chunks
inline size_t rt_wcan_bytes(int D) { return (size_t)(2 * (D / 16) + RT_NXMAX / 4) * RT_CHUNK; }
// byte offset of the 16-byte entry (row n, 8 consecutive k starting at k8 * 8) inside a chunk part
__host__ __device__ __forceinline__ int rt_entry(int n, int k8) { return ((n >> 3) * 2 + (k8 & 1)) * 128 + (n & 7) * 16; }

struct RtFoldOut {
  float* mbar;           // [D]
  unsigned char* wcan;   // B chunks
  float* svec;           // [2][256]: s_r, s_b
  float* b1_eff;         // [256]
};

// 8 floats -> 16-byte hi and lo entries
__device__ __forceinline__ void rt_store8(unsigned char* dst, const float (&v)[8]) {
  uint32_t hi[4], lo[4];
#pragma unroll
  for (int e = 0; e < 4; ++e) split_bf16(v[2 * e], v[2 * e + 1], hi[e], lo[e]);
  *reinterpret_cast<uint4*>(dst) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
  *reinterpret_cast<uint4*>(dst + RT_PART) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}

// Fold bodies, 128 threads: fc1's kbar columns (W_1k') as chunks D/16 .. 2D/16-1, b_1', mbar.
template <int D>
__device__ __forceinline__ void rt_fold_fc1_block(int bid, const float* __restrict__ part, int n_part, int LH,
                                                  const ResidW& w, const RtFoldOut& o, bool mbar_ready) {
  constexpr int P = 3 * D + 1, IN = P + R_DC;
  constexpr int N_W1 = R_HID * (D / 8);
  __shared__ float mb[D];
  for (int d = threadIdx.x; d < D; d += 128) {
    if (mbar_ready) {   // reduced by the layer-major key pass (same order of additions)
      mb[d] = o.mbar[d];
    } else {
      const float acc = sum_parts(part, n_part, D, d);
      mb[d] = acc / (float)LH;
    }
  }
  __syncthreads();
  int idx = bid * 128 + threadIdx.x;
  if (bid == 0 && !mbar_ready)
    for (int d = threadIdx.x; d < D; d += 128) o.mbar[d] = mb[d];
  if (idx < N_W1) {
    const int n = idx / (D / 8), k8 = idx % (D / 8), k0 = k8 * 8;
    const float* row = w.fc1_w + (int64_t)n * IN;
    float v[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) v[e] = fmaf(row[2 * D + k0 + e], mb[k0 + e], row[k0 + e]);
    rt_store8(o.wcan + (size_t)(D / 16 + (k8 >> 1)) * RT_CHUNK + rt_entry(n, k8), v);
    return;
  }
  idx -= N_W1;
  const int unit = idx >> 5, lane = threadIdx.x & 31;
  if (unit < R_HID) {
    const float* row = w.fc1_w + (int64_t)unit * IN + D;
    float acc = 0.f;
#pragma unroll
    for (int d = lane; d < D; d += 32) acc = fmaf(__ldg(row + d), mb[d], acc);
    acc = warp_sum(acc);
    if (lane == 0) o.b1_eff[unit] = acc + w.fc1_b[unit];
  }
}
template <int D>
inline int rt_fold_fc1_grid() { return (R_HID * (D / 8) + R_HID * 32 + 127) / 128; }

// Fold body, 256 threads: block (part, cross-attention head h, 16 query keys k0 .. k0+15).  part 0 computes Kc_h of its
// keys (Eq. 6) and from it its rows of W_S (S chunks), s_r and s_b; part 1 computes Vc_h and its rows of U (fc1 P chunks).
// Keys >= n_xq are padding: zero rows, s_b = RT_NEG.  nxp = key columns per head (multiple of 16).  The weight slices
// are staged in shared memory with every load of a phase in flight at once: the body is a latency chain, not a stream.
template <int D>
__device__ __forceinline__ void rt_fold_xattn_block(int bid, const float* __restrict__ part, int n_part, int LH,
                                                    const float* __restrict__ kq, const int32_t* __restrict__ n_xq,
                                                    int nxp, const ResidW& w, const RtFoldOut& o, bool mbar_ready) {
  constexpr int P = 3 * D + 1, IN = P + R_DC;
  constexpr int KPT = 16 * D / 256;  // keys per thread in the W_S step
  __shared__ float mb[D];
  __shared__ float x[16][D];
  __shared__ float wbuf[8192];       // W_K_h / W_V_h as [D][32]; then W_Q rows of the head as [32][2D] or fc1's c columns [256][32]
  __shared__ float kv[16][R_DH + 1]; // Kc (scaled) or Vc of the block's keys
  __shared__ float red[8][R_DH];
  __shared__ float bqh[R_DH];
  const int tid = threadIdx.x;
  const int pt = bid & 1, h = (bid >> 1) & 3, k0 = (bid >> 3) * 16;
  const int nq = *n_xq;
  {  // stage W_K_h (part 0) or W_V_h (part 1): rows d of 32 consecutive floats
    const float* src = (pt == 0 ? w.wk_t : w.wv_t) + h * R_DH;
    float4 v[D / 32];
#pragma unroll
    for (int j = 0; j < D / 32; ++j) {
      const int d = (tid >> 3) + 32 * j;
      v[j] = __ldg(reinterpret_cast<const float4*>(src + d * R_DC) + (tid & 7));
    }
    for (int d = tid; d < D; d += 256) {
      if (mbar_ready) {
        mb[d] = o.mbar[d];
      } else {
        const float acc = sum_parts(part, n_part, D, d);
        mb[d] = acc / (float)LH;
      }
    }
    for (int i = tid; i < 16 * D; i += 256) {
      const int key = i / D, d = i % D;
      x[key][d] = (k0 + key < nq) ? kq[(int64_t)(k0 + key) * D + d] : 0.f;
    }
#pragma unroll
    for (int j = 0; j < D / 32; ++j) *reinterpret_cast<float4*>(&wbuf[((tid >> 3) + 32 * j) * 32 + (tid & 7) * 4]) = v[j];
  }
  __syncthreads();
  const float sc = 1.4426950408889634f * 0.17677669529663689f;  // log2(e) / sqrt(32)  (R10)
  float wreg[32];  // the next phase's weight slice, loaded while Kc / Vc are computed
  if (pt == 0) {
#pragma unroll
    for (int j = 0; j < 32; ++j) {  // W_Q rows h*32 + c: columns [0, D) and [2D, 3D), index e = tid + 256 j in [32][2D]
      const int e = tid + 256 * j, c = e / (2 * D), dd = e % (2 * D);
      wreg[j] = (e < 32 * 2 * D) ? __ldg(w.wq + (int64_t)(h * R_DH + c) * P + (dd < D ? dd : dd + D)) : 0.f;
    }
  } else {
#pragma unroll
    for (int j = 0; j < 32; ++j) {  // fc1 columns P + h*32 + c of every hidden unit: [256][32]
      const int n = (tid >> 5) + 8 * j, c = tid & 31;
      wreg[j] = __ldg(w.fc1_w + (int64_t)n * IN + P + h * R_DH + c);
    }
  }
  {  // Kc or Vc of 2 keys per thread
    const int c = tid & 31, ig = tid >> 5, oc = h * R_DH + c;
    float a0 = 0.f, a1 = 0.f;
#pragma unroll 8
    for (int d = 0; d < D; ++d) {
      const float wv = wbuf[d * 32 + c];
      a0 = fmaf(wv, x[2 * ig][d], a0);
      a1 = fmaf(wv, x[2 * ig + 1][d], a1);
    }
    const bool ok0 = k0 + 2 * ig < nq, ok1 = k0 + 2 * ig + 1 < nq;
    const float bias = pt == 0 ? w.bk[oc] : w.bv[oc], mul = pt == 0 ? sc : 1.f;
    kv[2 * ig][c] = ok0 ? (a0 + bias) * mul : 0.f;
    kv[2 * ig + 1][c] = ok1 ? (a1 + bias) * mul : 0.f;
    if (pt == 0) {  // partial sums of b_Q' over D/8 columns of W_Qm per thread
      const float* row = w.wq + (int64_t)oc * P + D;
      float acc = 0.f;
#pragma unroll
      for (int d = ig * (D / 8); d < (ig + 1) * (D / 8); ++d) acc = fmaf(__ldg(row + d), mb[d], acc);
      red[ig][c] = acc;
    }
  }
  __syncthreads();  // wbuf (W_K / W_V) is dead
  if (pt == 0) {
#pragma unroll
    for (int j = 0; j < 32; ++j)
      if (tid + 256 * j < 32 * 2 * D) wbuf[tid + 256 * j] = wreg[j];
    if (tid < R_DH) {
      float acc = w.bq[h * R_DH + tid];
#pragma unroll
      for (int g = 0; g < 8; ++g) acc += red[g][tid];
      bqh[tid] = acc;
    }
    __syncthreads();
    {  // W_S columns of this block: thread (d, group of KPT keys); W_Q'[c][d] = W_Qk[c][d] + W_Qkm[c][d] mbar[d]
      const int d = tid % D, kg = tid / D;
      float acc[KPT];
#pragma unroll
      for (int j = 0; j < KPT; ++j) acc[j] = 0.f;
      const float m = mb[d];
#pragma unroll 8
      for (int c = 0; c < R_DH; ++c) {
        const float wqp = fmaf(wbuf[c * 2 * D + D + d], m, wbuf[c * 2 * D + d]);
#pragma unroll
        for (int j = 0; j < KPT; ++j) acc[j] = fmaf(wqp, kv[kg * KPT + j][c], acc[j]);
      }
      __syncthreads();  // every thread has read wbuf: reuse it as the transposed W_S tile [16][D + 1]
#pragma unroll
      for (int j = 0; j < KPT; ++j) wbuf[(kg * KPT + j) * (D + 1) + d] = acc[j];
    }
    if (tid >= 224) {  // s_r (lanes 0-15 of the last warp) and s_b (lanes 16-31) of the block's keys
      const int t = tid - 224, i = t & 15;
      float acc = 0.f;
      if (t < 16) {
        for (int c = 0; c < R_DH; ++c) acc = fmaf(__ldg(w.wq + (int64_t)(h * R_DH + c) * P + 3 * D), kv[i][c], acc);
      } else {
        for (int c = 0; c < R_DH; ++c) acc = fmaf(bqh[c], kv[i][c], acc);
        if (k0 + i >= nq) acc = RT_NEG;
      }
      o.svec[(t < 16 ? 0 : 256) + h * nxp + k0 + i] = acc;
    }
    __syncthreads();
    if (tid < 16 * (D / 8)) {  // W_S entries: row n = (h, key), 8 consecutive d
      const int i = tid / (D / 8), k8 = tid % (D / 8), n = h * nxp + k0 + i;
      float v[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) v[e] = wbuf[i * (D + 1) + k8 * 8 + e];
      rt_store8(o.wcan + (size_t)(k8 >> 1) * RT_CHUNK + rt_entry(n, k8), v);
    }
  } else {
    // U rows (h, k0 .. k0+15) for the hidden units n = warp + 8 j held in wreg: thread (c = lane) multiplies its column
    // by Vc[:, c]; the sum over c is a warp reduction per (n, key) -- instead, transpose through shared memory:
#pragma unroll
    for (int j = 0; j < 32; ++j) wbuf[((tid >> 5) + 8 * j) * 32 + (tid & 31)] = wreg[j];
    __syncthreads();
    const int n = tid;
    float a0[8], a1[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a0[i] = 0.f; a1[i] = 0.f; }
#pragma unroll 8
    for (int c = 0; c < R_DH; ++c) {
      const float wv = wbuf[n * 32 + ((c + n) & 31)];  // rotated column order: conflict-free rows of 32 floats
      const int cc = (c + n) & 31;
#pragma unroll
      for (int i = 0; i < 8; ++i) { a0[i] = fmaf(wv, kv[i][cc], a0[i]); a1[i] = fmaf(wv, kv[8 + i][cc], a1[i]); }
    }
    unsigned char* ch = o.wcan + (size_t)(2 * (D / 16) + (h * nxp + k0) / 16) * RT_CHUNK;
    rt_store8(ch + rt_entry(n, 0), a0);
    rt_store8(ch + rt_entry(n, 1), a1);
  }
}
inline int rt_fold_xattn_grid(int nxp) { return 8 * (nxp / 16); }

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

#ifdef IKV_TRACE
__device__ long long g_rt_trace[2][64];
#define RT_T(w, i) do { if (blockIdx.x == 0) g_rt_trace[w][i] = clock64(); } while (0)
#else
#define RT_T(w, i) do { } while (0)
#endif

// ---------------------------------------------------------------------------------------------------------------
// k_tail_tc: the residual head of Eq. 4-6 over 128-token tiles, one persistent CTA per SM.
//   warps 0-7   tile loader (kbar rows -> A operand), per-head softmax, epilogue (GELU, fc2, s = rule + alpha z)
//   warp  8     MMA issuer (one thread)            warp 9   bulk-copy chunk loader (one thread)
// Per tile the compute warps run  fill(i) | epilogue(i-1) | softmax(i)  so that S(i) is multiplied under epilogue(i-1).
// (Measured and rejected: four extra warps streaming the tile's logits for rule_c inside this kernel -- with 212 KB of
// shared memory and 128 registers per thread a CTA keeps only 32 KB of loads in flight, 11 GB/s per SM, 110 k cycles per
// tile; the rule kernel with 196 KB in flight per SM stays a launch of its own.)
// ---------------------------------------------------------------------------------------------------------------
constexpr int RT_CWARPS = 8;
constexpr int RT_TAIL_THREADS = (RT_CWARPS + 2) * 32;

struct TailParams {
  const float* rule_c;       // [n_cand]  (Eq. 3)
  const float* kbar;         // [n_cand][D]
  const int32_t* n_cand;
  const int32_t* cand_pos;
  const int32_t* n_xq;
  const unsigned char* wcan;
  const float* svec;
  const float* b1_eff;
  int nxp;                   // key columns per head (multiple of 16, <= RT_NXMAX)
  int use_xattn;
  int early;                 // rule_c and kbar are complete when this grid starts (they come from the layer-major key
                             // pass, two kernels back): only the folded operands wait for the predecessor
  float* scores;             // by position
};

template <int D>
__host__ __device__ constexpr int rt_tail_smem() {
  return rt_region0<D>() + RT_P01 + RT_STAGES * RT_CHUNK + (5 * 256 + 2 * 128) * 4 + 256;
}

template <int D>
__global__ __launch_bounds__(RT_TAIL_THREADS, 1) void k_tail_tc(const TailParams p, const ResidW w) {
  constexpr int KS = D / 16;
  constexpr int A_PART = RT_M * D * 2;   // bytes of kbar hi (and of kbar lo)
  constexpr int A_SBO = (D / 8) * 128;   // byte distance between 8-row groups of the kbar rows
  if (threadIdx.x == 0) RT_T(0, 0);
  // Programmatic stream serialization.  p.early: the predecessor (k_post_key) only produces the folded operands, which
  // warp 9 loads after its own griddepcontrol.wait; set-up and the first tile's fill run under the predecessor.
  if (!p.early) pdl_wait();
  pdl_launch_dependents();
  if (threadIdx.x == 0) RT_T(0, 1);
  extern __shared__ __align__(128) unsigned char rt_smem_raw[];
  unsigned char* region0 = rt_smem_raw;                // kbar hi | lo; later P of heads 2, 3
  unsigned char* p01 = region0 + rt_region0<D>();      // P of heads 0, 1
  unsigned char* ring = p01 + RT_P01;                  // [RT_STAGES][RT_CHUNK]
  float* ep_b1 = reinterpret_cast<float*>(ring + RT_STAGES * RT_CHUNK);
  float* ep_wr = ep_b1 + 256;
  float* ep_w2 = ep_wr + 256;
  float* sv_r = ep_w2 + 256;
  float* sv_b = sv_r + 256;
  float* ep_z = sv_b + 256;                  // [2][128]
  uint64_t* bfull = reinterpret_cast<uint64_t*>(ep_z + 256);
  uint64_t* bempty = bfull + RT_STAGES;
  uint64_t* a_ready = bempty + RT_STAGES;   // kbar rows written (8 warps)
  uint64_t* s_full = a_ready + 1;           // S accumulator complete
  uint64_t* ak_free = s_full + 1;           // the MMAs reading the kbar rows have completed
  uint64_t* p_ready = ak_free + 1;          // [4] P of head h written (4 warps each)
  uint64_t* fc1_full = p_ready + 4;         // fc1 accumulator complete (and every operand buffer of the tile is free)
  uint64_t* tmem_free = fc1_full + 1;       // the epilogue has read the fc1 accumulator (8 warps)
  uint64_t* vec_ready = tmem_free + 1;      // b1', s_r, s_b (outputs of the fold) are in shared memory (warp 9)
  uint32_t* tmem_base_p = reinterpret_cast<uint32_t*>(vec_ready + 1);

  const int nc = *p.n_cand;
  const int n_tiles = (nc + RT_M - 1) / RT_M;
  if ((int)blockIdx.x >= n_tiles) return;
  const int nq = p.use_xattn ? *p.n_xq : 0;
  const bool xat = nq > 0;
  const int NXP = p.nxp;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int IN = 3 * D + 1 + R_DC;
  if (threadIdx.x == 0) {
    for (int s = 0; s < RT_STAGES; ++s) { mbar_init(&bfull[s], 1); mbar_init(&bempty[s], 1); }
    mbar_init(a_ready, RT_CWARPS);
    mbar_init(s_full, 1);
    mbar_init(ak_free, 1);
    for (int h = 0; h < 4; ++h) mbar_init(&p_ready[h], 4);
    mbar_init(fc1_full, 1);
    mbar_init(tmem_free, RT_CWARPS);
    mbar_init(vec_ready, 1);
    mbar_fence_init();
  }
  for (int n = threadIdx.x; n < R_HID; n += RT_TAIL_THREADS) {  // static weights: no dependency on the predecessor
    ep_wr[n] = __ldg(w.fc1_w + (int64_t)n * IN + 3 * D);
    ep_w2[n] = __ldg(w.fc2_w + n);
  }
  if (warp == 8) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_p)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_base_p;
  if (threadIdx.x == 0) RT_T(0, 2);
  const int HR = 512 * NXP;  // bytes of one head's P rows (hi | lo)
  // chunk schedule per tile (identical in the loader and the issuer): S chunks, fc1 kbar chunks, then the P chunks of
  // heads 0, 2, 1, 3 (warps 0-3 finish head 0 while warps 4-7 finish head 2).  Order in wcan: S | fc1 kbar | fc1 P by head.
  const int n_s = xat ? KS : 0, spp = NXP / 16;

  if (warp == 9) {
    // ------------------------------------------------------------------ chunk loader (one thread); first the folded
    // vectors, which like the chunks are outputs of the predecessor
    pdl_wait();
    for (int n = lane; n < R_HID; n += 32) {
      ep_b1[n] = p.b1_eff[n];
      sv_r[n] = xat ? p.svec[n] : 0.f;
      sv_b[n] = xat ? p.svec[256 + n] : 0.f;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(vec_ready);
    if (lane == 0) {
      const unsigned char* src_s = p.wcan;
      const unsigned char* src_k = p.wcan + (size_t)KS * RT_CHUNK;
      const unsigned char* src_p = p.wcan + (size_t)(2 * KS) * RT_CHUNK;
      int slot = 0;
      uint32_t ph = 1u;  // the first pass over the ring finds every slot free
      auto push = [&](const unsigned char* src, uint32_t pb) {
        mbar_wait(&bempty[slot], ph);
        mbar_arrive_expect_tx(&bfull[slot], 2 * pb);
        bulk_g2s(ring + slot * RT_CHUNK, src, pb, &bfull[slot]);
        bulk_g2s(ring + slot * RT_CHUNK + RT_PART, src + RT_PART, pb, &bfull[slot]);
        if (++slot == RT_STAGES) { slot = 0; ph ^= 1u; }
      };
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        for (int j = 0; j < n_s; ++j) push(src_s + (size_t)j * RT_CHUNK, (uint32_t)(128 * NXP));  // 4 NXP rows x 32 B
        for (int j = 0; j < KS; ++j) push(src_k + (size_t)j * RT_CHUNK, (uint32_t)RT_PART);
        if (xat) {
          const int order[4] = {0, 2, 1, 3};
          for (int o = 0; o < 4; ++o)
            for (int st = 0; st < spp; ++st) push(src_p + (size_t)(order[o] * spp + st) * RT_CHUNK, (uint32_t)RT_PART);
        }
      }
    }
    __syncwarp();
  } else if (warp == 8) {
    // ------------------------------------------------------------------ MMA issuer (one thread).  The descriptors are
    // kept as 64-bit values and advanced by additions: the issue loop is a serial instruction stream of one thread.
    if (lane == 0) {
      const uint32_t ibase = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 4) << 24);  // fp32 D, bf16 A/B, K-major, M=128
      const uint32_t idesc_h = ibase | ((256u >> 3) << 17);
      const uint32_t idesc_s = ibase | (((uint32_t)(4 * NXP) >> 3) << 17);
      const uint32_t r0 = smem_u32(region0), pp = smem_u32(p01), rg = smem_u32(ring);
      const uint64_t db0 = umma_desc(rg, 128, 256);
      const uint64_t da_k = umma_desc(r0, 128, (uint32_t)A_SBO);
      int slot = 0;
      uint32_t ph = 0u;
      uint64_t db = db0;
      // one chunk: hi*hi + lo*hi + hi*lo; a_lo - a_hi and b_lo - b_hi are constant offsets of the start-address field
      auto chunk = [&](uint64_t dah, uint32_t a_lo_off, uint32_t td, uint32_t idesc, uint32_t acc) {
        mbar_wait(&bfull[slot], ph);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        umma_bf16(td, dah, db, idesc, acc);
        umma_bf16(td, dah + (a_lo_off >> 4), db, idesc, 1u);
        umma_bf16(td, dah, db + (RT_PART >> 4), idesc, 1u);
        umma_commit(&bempty[slot]);
        db += (RT_CHUNK >> 4);
        if (++slot == RT_STAGES) { slot = 0; ph ^= 1u; db = db0; }
      };
      uint32_t par = 0u;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, par ^= 1u) {
        mbar_wait(a_ready, par);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        for (int s = 0; s < n_s; ++s) chunk(da_k + (uint64_t)(s * 16), (uint32_t)A_PART, tmem, idesc_s, s ? 1u : 0u);
        if (xat) umma_commit(s_full);
        if (tile != (int)blockIdx.x) {  // the previous tile's epilogue has read the fc1 accumulator
          mbar_wait(tmem_free, par ^ 1u);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        }
        for (int s = 0; s < KS; ++s) chunk(da_k + (uint64_t)(s * 16), (uint32_t)A_PART, tmem + 256u, idesc_h, s ? 1u : 0u);
        umma_commit(ak_free);
        if (xat) {
          const int order[4] = {0, 2, 1, 3};
          for (int o = 0; o < 4; ++o) {
            const int h = order[o];
            mbar_wait(&p_ready[h], par);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint64_t da_p =
                umma_desc(h < 2 ? pp + (uint32_t)(h * HR) : r0 + (uint32_t)((h - 2) * HR), 128, (uint32_t)(16 * NXP));
            for (int st = 0; st < spp; ++st) chunk(da_p + (uint64_t)(st * 16), (uint32_t)(HR / 2), tmem + 256u, idesc_h, 1u);
          }
        }
        umma_commit(fc1_full);
      }
    }
    __syncwarp();
  } else {
    // -------------------------------------------------------------------- warps 0-7
    constexpr int KB = D / 32, NU = 16 * KB / 8;  // kbar items per warp: 8 rows x 4 groups of 8 columns each
    const int qd = warp & 3, m = qd * 32 + lane, hp = warp >> 2, nh = warp >> 2;
    // epilogue of one tile: warp w reads TMEM lanes 32 (w % 4) .. + 31 (token rows) of accumulator half w / 4:
    // hid = acc + b1' + rule w_r -> erf-GELU -> fc2 dot; the two halves of a row are added through shared memory
    auto epilogue = [&](int tile, float rule) {
      const int tok = tile * RT_M + m;
      f32x2 z2 = pk2(0.f, 0.f);
      const f32x2 rule2 = pk2(rule, rule);
#pragma unroll 1
      for (int c0 = 0; c0 < 128; c0 += 16) {
        float v[16];
        tmem_ld16(tmem + ((uint32_t)(qd * 32) << 16) + (uint32_t)(256 + nh * 128 + c0), v);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 16; j += 4) {  // two hidden units per packed instruction; weights as 16-byte broadcasts
          const int n = nh * 128 + c0 + j;
          const float4 wr = *reinterpret_cast<const float4*>(&ep_wr[n]);
          const float4 b1 = *reinterpret_cast<const float4*>(&ep_b1[n]);
          const float4 w2 = *reinterpret_cast<const float4*>(&ep_w2[n]);
          const f32x2 ha = fma2(rule2, pk2(wr.x, wr.y), add2(pk2(v[j], v[j + 1]), pk2(b1.x, b1.y)));
          const f32x2 hb = fma2(rule2, pk2(wr.z, wr.w), add2(pk2(v[j + 2], v[j + 3]), pk2(b1.z, b1.w)));
          z2 = fma2(pk2(w2.x, w2.y), gelu_erf2(ha), z2);
          z2 = fma2(pk2(w2.z, w2.w), gelu_erf2(hb), z2);
        }
      }
      float z, zb;
      upk2(z2, z, zb);
      z += zb;
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(tmem_free);
      ep_z[nh * 128 + m] = z;
      bar_sync(1, RT_CWARPS * 32);
      if (nh == 0 && tok < nc) p.scores[p.cand_pos[tok]] = rule + w.alpha * ((ep_z[m] + ep_z[128 + m]) + w.fc2_b[0]);
      bar_sync(1, RT_CWARPS * 32);  // ep_z is free
    };
    int it = 0, prev_tile = -1;
    float rule = 0.f, prev_rule = 0.f;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
      const int t0 = tile * RT_M;
      const uint32_t par = (uint32_t)it & 1u;
      // kbar rows -> A operand (hi | lo): 128-byte global segments per row, 512 contiguous bytes of shared memory per warp
      // item; all loads are issued before the wait on the previous tile's MMAs and before the first use
      float4 x0[NU], x1[NU];
#pragma unroll
      for (int u = 0; u < NU; ++u) {
        const int unit = warp + 8 * u, rb = unit / KB, kb = unit % KB;
        const int row = rb * 8 + (lane & 7), k8 = kb * 4 + (lane >> 3);
        if (t0 + row < nc) {
          const float4* src = reinterpret_cast<const float4*>(p.kbar + (int64_t)(t0 + row) * D + k8 * 8);
          x0[u] = __ldg(src); x1[u] = __ldg(src + 1);
        } else {
          x0[u] = make_float4(0.f, 0.f, 0.f, 0.f); x1[u] = x0[u];
        }
      }
      if (it > 0) {  // the previous tile's MMAs are complete: its operand buffers are free, its accumulator is final
        mbar_wait(fc1_full, par ^ 1u);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      }
#pragma unroll
      for (int u = 0; u < NU; ++u) {
        const int unit = warp + 8 * u, rb = unit / KB, kb = unit % KB;
        const int k8 = kb * 4 + (lane >> 3);
        uint32_t hi[4], lo[4];
        split_bf16(x0[u].x, x0[u].y, hi[0], lo[0]); split_bf16(x0[u].z, x0[u].w, hi[1], lo[1]);
        split_bf16(x1[u].x, x1[u].y, hi[2], lo[2]); split_bf16(x1[u].z, x1[u].w, hi[3], lo[3]);
        unsigned char* dst = region0 + rb * A_SBO + k8 * 128 + (lane & 7) * 16;
        *reinterpret_cast<uint4*>(dst) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
        *reinterpret_cast<uint4*>(dst + A_PART) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // publish the rows to the async proxy (tcgen05.mma)
      __syncwarp();
      if (lane == 0) mbar_arrive(a_ready);
      if (threadIdx.x == 0 && it == 0) RT_T(0, 3);
      prev_rule = rule;
      rule = (t0 + m < nc) ? p.rule_c[t0 + m] : 0.f;
      if (it == 0) mbar_wait(vec_ready, 0u);  // b1', s_r, s_b
      if (it > 0) epilogue(prev_tile, prev_rule);   // S of this tile is multiplied meanwhile
      if (threadIdx.x == 0 && it == 1) RT_T(0, 12);
      if (xat) {
        // ---- per-head softmax of this thread's token row; warps 0-3 take heads 0, 1, warps 4-7 heads 2, 3
        mbar_wait(s_full, par);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (threadIdx.x == 0 && it == 0) RT_T(0, 4);
#pragma unroll 1
        for (int hh = 0; hh < 2; ++hh) {
          const int h = hp * 2 + hh;
          float x[RT_NXMAX];
#pragma unroll
          for (int c0 = 0; c0 < RT_NXMAX; c0 += 16)
            if (c0 < NXP) tmem_ld16(tmem + ((uint32_t)(qd * 32) << 16) + (uint32_t)(h * NXP + c0), &x[c0]);
          tmem_ld_wait();
          // two columns per packed fp32 instruction; s_r, s_b as 16-byte broadcasts
          const f32x2 rule2 = pk2(rule, rule);
          float mx = -CUDART_INF_F;
#pragma unroll
          for (int c = 0; c < RT_NXMAX; c += 4)
            if (c < NXP) {
              const float4 sr = *reinterpret_cast<const float4*>(&sv_r[h * NXP + c]);
              const float4 sb = *reinterpret_cast<const float4*>(&sv_b[h * NXP + c]);
              upk2(fma2(rule2, pk2(sr.x, sr.y), add2(pk2(x[c], x[c + 1]), pk2(sb.x, sb.y))), x[c], x[c + 1]);
              upk2(fma2(rule2, pk2(sr.z, sr.w), add2(pk2(x[c + 2], x[c + 3]), pk2(sb.z, sb.w))), x[c + 2], x[c + 3]);
              mx = fmaxf(fmaxf(mx, fmaxf(x[c], x[c + 1])), fmaxf(x[c + 2], x[c + 3]));
            }
          const f32x2 nmx2 = pk2(-mx, -mx);
          f32x2 l2 = pk2(0.f, 0.f);
#pragma unroll
          for (int c = 0; c < RT_NXMAX; c += 2)
            if (c < NXP) {
              float d0, d1;
              upk2(add2(pk2(x[c], x[c + 1]), nmx2), d0, d1);
              x[c] = ex2f(d0); x[c + 1] = ex2f(d1);
              l2 = add2(l2, pk2(x[c], x[c + 1]));
            }
          float l, lb;
          upk2(l2, l, lb);
          l += lb;
          const float inv = 1.f / l;
          const f32x2 inv2 = pk2(inv, inv), m1 = pk2(-1.f, -1.f);
          if (hp == 1 && hh == 0) mbar_wait(ak_free, par);  // heads 2, 3 overwrite the kbar rows
          unsigned char* base = (h < 2 ? p01 + h * HR : region0 + (h - 2) * HR) + (m >> 3) * (16 * NXP) + (m & 7) * 16;
#pragma unroll
          for (int g = 0; g < RT_NXMAX / 8; ++g)
            if (g * 8 < NXP) {
              uint32_t hi[4], lo[4];
#pragma unroll
              for (int e = 0; e < 4; ++e) {  // split_bf16 of the normalised pair, the subtraction packed
                const f32x2 pn = mul2(pk2(x[g * 8 + 2 * e], x[g * 8 + 2 * e + 1]), inv2);
                float a, b;
                upk2(pn, a, b);
                hi[e] = pack_bf16_rn(a, b);
                upk2(fma2(pk2(bf16lo(hi[e]), bf16hi(hi[e])), m1, pn), a, b);
                lo[e] = pack_bf16_rn(a, b);
              }
              *reinterpret_cast<uint4*>(base + g * 128) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
              *reinterpret_cast<uint4*>(base + g * 128 + HR / 2) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
          asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) mbar_arrive(&p_ready[h]);
          if (threadIdx.x == 0 && it == 0) RT_T(0, 5 + hh);
        }
      }
      prev_tile = tile;
    }
    mbar_wait(fc1_full, (uint32_t)(it - 1) & 1u);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (threadIdx.x == 0) RT_T(0, 9);
    epilogue(prev_tile, rule);
    if (threadIdx.x == 0) RT_T(0, 10);
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 8) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
  }
  if (threadIdx.x == 0) RT_T(0, 11);
}

}  // namespace ikv
