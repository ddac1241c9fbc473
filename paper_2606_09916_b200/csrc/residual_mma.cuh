// residual_mma.cuh -- residual head of Eq. 4-6 on the tensor pipe, fp32-grade.
// Topology per DESIGN.md R9-R12.  "FP32 residual head": every GEMM operand is split into a bf16 hi
// and a bf16 lo part and each product is taken as hi*hi + lo*hi + hi*lo with fp32 accumulation (mma.sync
// m16n8k16), which carries ~16 mantissa bits per operand; softmax, GELU and all vectors stay fp32.
//
// Folding of the constant inputs: phi_j = [kbar_j | mbar | kbar_j (.) mbar | rule_j] and mbar is the same for every
// token of the call, so   W phi_j + b = (W_k + W_km diag(mbar)) kbar_j + rule_j w_r + (b + W_m mbar).
// k_resid_fold builds the folded matrices of W_Q and fc1 once per call, directly in B-fragment order.
//
// One warp scores 16 candidates end to end in registers:
//   Q   = Wq' kbar + rule wq_r + bq'                          (16 x 128, K = D)
//   c_h = softmax(Q_h Kc_h^T / sqrt(32)) Vc_h,  h = 0..3       (online softmax over chunks of 64 query keys)
//   hid = W1k' kbar + W1c c + rule w1_r + b1'                 (16 x 256, K = D + 128), in 4 chunks of 64 units
//   z   = fc2_w . GELU_erf(hid) + fc2_b;   s = rule + alpha z
// Accumulator (C) fragments are turned into A fragments of the next product in registers.
#pragma once
#include "common.cuh"
#include "pipe.cuh"

namespace ikv {

constexpr int R_DC = 128;   // d_c
constexpr int R_HC = 4;     // H_c
constexpr int R_DH = 32;    // d_c / H_c
constexpr int R_HID = 256;  // hidden width
constexpr int R_WARPS = 4;  // 16-candidate tiles per CTA

// Device copy of the residual head.  Raw matrices are row-major [out][in] as loaded (R9).
struct ResidW {
  const float *wq, *bq;        // [128][3D+1], [128]
  const float *wk_t, *bk;      // [D][128] (transposed), [128]
  const float *wv_t, *bv;      // [D][128] (transposed), [128]
  const float *fc1_w, *fc1_b;  // [256][3D+1+128], [256]
  const float *fc2_w, *fc2_b;  // [256], [1]
  const uint4* w1c_frag;       // static: fc1 columns of c, [4 chunks][8 k-steps][8 n-tiles][32 lanes]
  float alpha;                 // already clipped to [-5,5]
};

__device__ __forceinline__ uint32_t pack_bf16_rn(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// (x, y) -> packed bf16 hi parts and packed bf16 lo parts (x = hi + lo up to ~2^-17 |x|)
__device__ __forceinline__ void split_bf16(float x, float y, uint32_t& hi, uint32_t& lo) {
  hi = pack_bf16_rn(x, y);
  lo = pack_bf16_rn(x - bf16lo(hi), y - bf16hi(hi));
}
// acc += A * B with A = (ah + al), B = (b.x,b.y hi | b.z,b.w lo), dropping lo*lo
__device__ __forceinline__ void mma3(float (&acc)[4], const uint32_t (&ah)[4], const uint32_t (&al)[4], const uint4& b) {
  mma_bf16_16816(acc, ah[0], ah[1], ah[2], ah[3], b.x, b.y);
  mma_bf16_16816(acc, al[0], al[1], al[2], al[3], b.x, b.y);
  mma_bf16_16816(acc, ah[0], ah[1], ah[2], ah[3], b.z, b.w);
}

// k index of the kbar A fragments: lane q loads kbar[row][16 s + 4 q .. + 3] as one float4, so mma k index kappa of
// k-step s stands for column 16 s + kperm(kappa).
__host__ __device__ __forceinline__ int kperm(int kappa) {
  return (kappa < 8) ? 4 * (kappa >> 1) + (kappa & 1) : 4 * ((kappa - 8) >> 1) + 2 + (kappa & 1);
}

// One B fragment (hi | lo) of lane (r, q) from a functor B(k_local 0..15, n_local 0..7).
template <typename F>
__device__ __forceinline__ uint4 make_bfrag(int lane, F B) {
  const int r = lane >> 2, q = lane & 3;
  const float v0 = B(2 * q, r), v1 = B(2 * q + 1, r), v2 = B(2 * q + 8, r), v3 = B(2 * q + 9, r);
  uint4 o;
  split_bf16(v0, v1, o.x, o.z);
  split_bf16(v2, v3, o.y, o.w);
  return o;
}

// mbar partial sums (Eq. 5 mbar): block b of >= D threads; part[b][d] = sum of rows 32 b .. 32 b + 31 of M.
__device__ __forceinline__ void mean_memory_part_block(int b, const float* __restrict__ M, int LH, int D,
                                                       float* __restrict__ part) {
  const int d = threadIdx.x, r0 = b * 32;
  if (d >= D) return;
  float acc = 0.f;
#pragma unroll 8
  for (int i = r0; i < min(LH, r0 + 32); ++i) acc += M[(int64_t)i * D + d];
  part[b * D + d] = acc;
}

// fc1' as the B operand of tcgen05.mma (kind::f16, K-major, no swizzle): chunks of 128 hidden units x 64 k, each as a hi
// and a lo bf16 part of W1C_PART bytes in the canonical layout (8 x 16-byte core matrices, 128 B contiguous; core
// matrix (n/8, k/8) at ((n/8) * 8 + k/8) * 128).  k < D: folded kbar columns (natural order); k >= D: the c columns.
constexpr int W1C_PART = 128 * 64 * 2;      // bytes of one part of one chunk
constexpr int W1C_CHUNK = 2 * W1C_PART;     // hi | lo
template <int D>
__host__ __device__ inline size_t w1_can_offset(int n, int k) {
  constexpr int NKC = D / 64 + 2;
  const int nh = n >> 7, nl = n & 127, kc = k >> 6, kl = k & 63;
  return (size_t)(nh * NKC + kc) * W1C_CHUNK + (size_t)((nl >> 3) * 8 + (kl >> 3)) * 128 + (nl & 7) * 16 + (kl & 7) * 2;
}

struct FoldOut {
  float* mbar;      // [D]
  uint4* wq_frag;   // [D/16][16][32]
  unsigned char* w1_can;  // fc1' for tcgen05: [2 N halves][D/64 + 2 K chunks][hi | lo][128 x 64 bf16, canonical K-major]
  float* bq_eff;    // [128]
  float* b1_eff;    // [256]
};

// Folds mbar into W_Q and fc1 (see the header of this file).  Blocks of 128 threads; resid_fold_grid() blocks cover
// D/16*16*32 W_Q fragment items, 256*D/8 canonical fc1 rows and 384 bias warps.
// sum over the partial rows part[b][d], b ascending (the order is part of the result); eight loads in flight
__device__ __forceinline__ float sum_parts(const float* __restrict__ part, int n_part, int D, int d) {
  float acc = 0.f;
  int b = 0;
  for (; b + 8 <= n_part; b += 8) {
    float v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = part[(b + j) * D + d];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc += v[j];
  }
  for (; b < n_part; ++b) acc += part[b * D + d];
  return acc;
}

template <int D>
__device__ __forceinline__ void resid_fold_block(int bid, const float* __restrict__ part, int n_part, int LH,
                                                 const ResidW& w, const FoldOut& o) {
  constexpr int KS = D / 16, P = 3 * D + 1, IN = P + R_DC;
  constexpr int N_WQ = KS * 16 * 32, N_W1 = R_HID * (D / 8), N_B = R_DC + R_HID;
  __shared__ float mb[D];
  for (int d = threadIdx.x; d < D; d += 128) {
    const float acc = sum_parts(part, n_part, D, d);
    mb[d] = acc / (float)LH;
  }
  __syncthreads();
  int idx = bid * 128 + threadIdx.x;
  if (bid == 0)
    for (int d = threadIdx.x; d < D; d += 128) o.mbar[d] = mb[d];
  if (idx < N_WQ) {
    const int lane = idx & 31, t = (idx >> 5) & 15, s = idx >> 9;
    o.wq_frag[idx] = make_bfrag(lane, [&](int kl, int nl) {
      const int n = t * 8 + nl, k = s * 16 + kperm(kl);
      const float* row = w.wq + (int64_t)n * P;
      return fmaf(row[2 * D + k], mb[k], row[k]);
    });
    return;
  }
  idx -= N_WQ;
  if (idx < N_W1) {
    // one 16-byte core-matrix row (8 consecutive k) of the folded fc1 kbar columns, hi and lo parts
    const int n = idx / (D / 8), kg = idx % (D / 8), k0 = kg * 8;
    const float* row = w.fc1_w + (int64_t)n * IN;
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int k = k0 + 2 * e;
      split_bf16(fmaf(row[2 * D + k], mb[k], row[k]), fmaf(row[2 * D + k + 1], mb[k + 1], row[k + 1]), hi[e], lo[e]);
    }
    unsigned char* dst = o.w1_can + w1_can_offset<D>(n, k0);
    *reinterpret_cast<uint4*>(dst) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(dst + W1C_PART) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    return;
  }
  idx -= N_W1;
  // folded biases: one warp per output unit (lanes stride the D columns of W_m, one round of coalesced loads)
  const int unit = idx >> 5, lane = threadIdx.x & 31;
  if (unit < N_B) {
    const bool isq = unit < R_DC;
    const int n = isq ? unit : unit - R_DC;
    const float* row = isq ? (w.wq + (int64_t)n * P + D) : (w.fc1_w + (int64_t)n * IN + D);
    float acc = 0.f;
#pragma unroll
    for (int d = lane; d < D; d += 32) acc = fmaf(__ldg(row + d), mb[d], acc);
    acc = warp_sum(acc);
    if (lane == 0) (isq ? o.bq_eff : o.b1_eff)[n] = acc + (isq ? w.bq[n] : w.fc1_b[n]);
  }
}
template <int D>
inline int resid_fold_grid() {
  return ((D / 16) * 16 * 32 + R_HID * (D / 8) + (R_DC + R_HID) * 32 + 127) / 128;
}

// Kc = W_K K^q + b_K, Vc = W_V K^q + b_V (Eq. 6): block `bid` = (16-key step v, cross-attention head hc), 128 threads
// = 32 channels of the head x 4 groups of 4 keys.  Written as B fragments:
//   kc_frag[((hc*2 + u)*nkt + t)*32 + lane] : S = Q_h Kc_h^T, k = head dim 16 u + kappa, n = key 8 t + r, scaled
//                                             by log2(e)/sqrt(32) so that the softmax runs on exp2
//   vc_frag[((hc*nks + v)*4 + nt)*32 + lane]: O = P Vc_h,     k = key 16 v + kappa, n = head dim 8 nt + r
// nkt = 2 nks = capacity in 8-key tiles.  Keys >= n_xq are zero.
__device__ __forceinline__ void resid_kv_frags_block(int bid, const float* __restrict__ kq,
                                                     const int32_t* __restrict__ n_xq, int D, const ResidW& w, int nks,
                                                     uint4* __restrict__ kc_frag, uint4* __restrict__ vc_frag) {
  __shared__ float x[16][128];
  __shared__ float kc[16][R_DH + 1], vc[16][R_DH + 1];
  const int nq = *n_xq, v = bid >> 2, hc = bid & 3, k0 = v * 16;
  if (k0 >= nq) return;
  for (int i = threadIdx.x; i < 16 * D; i += 128) {
    const int key = i / D, d = i % D;
    x[key][d] = (k0 + key < nq) ? kq[(int64_t)(k0 + key) * D + d] : 0.f;
  }
  __syncthreads();
  // thread (ch, dg): channel ch of the head, quarter dg of the D columns, all 16 keys; quarters summed through smem
  __shared__ float part[2][4][16][R_DH + 1];
  const int ch = threadIdx.x & 31, dg = threadIdx.x >> 5, o = hc * R_DH + ch;
  float ak[16], av[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) { ak[i] = 0.f; av[i] = 0.f; }
  const int dq = D / 4;
#pragma unroll 16
  for (int dd = 0; dd < dq; ++dd) {
    const int d = dg * dq + dd;
    const float wk = __ldg(w.wk_t + d * R_DC + o), wv = __ldg(w.wv_t + d * R_DC + o);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      ak[i] = fmaf(wk, x[i][d], ak[i]);
      av[i] = fmaf(wv, x[i][d], av[i]);
    }
  }
#pragma unroll
  for (int i = 0; i < 16; ++i) { part[0][dg][i][ch] = ak[i]; part[1][dg][i][ch] = av[i]; }
  __syncthreads();
  const float sc = 1.4426950408889634f * 0.17677669529663689f;  // log2(e) / sqrt(32)  (R10)
  const float bk = w.bk[o], bv = w.bv[o];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int key = dg * 4 + i;
    const bool ok = k0 + key < nq;
    const float sk = bk + ((part[0][0][key][ch] + part[0][1][key][ch]) + (part[0][2][key][ch] + part[0][3][key][ch]));
    const float sv = bv + ((part[1][0][key][ch] + part[1][1][key][ch]) + (part[1][2][key][ch] + part[1][3][key][ch]));
    kc[key][ch] = ok ? sk * sc : 0.f;
    vc[key][ch] = ok ? sv : 0.f;
  }
  __syncthreads();
  const int nkt = 2 * nks, lane = threadIdx.x & 31, a = threadIdx.x >> 5;
  {  // Kc: a = (u, tile-in-pair)
    const int u = a >> 1, tl = a & 1;
    kc_frag[((int64_t)(hc * 2 + u) * nkt + 2 * v + tl) * 32 + lane] =
        make_bfrag(lane, [&](int kl, int nl) { return kc[tl * 8 + nl][u * 16 + kl]; });
  }
  // Vc: a = nt
  vc_frag[((int64_t)(hc * nks + v) * 4 + a) * 32 + lane] =
      make_bfrag(lane, [&](int kl, int nl) { return vc[kl][a * 8 + nl]; });
}

struct ResidMmaParams {
  const float* rule_c;       // [n_cand]
  const float* kbar;         // [n_cand][D]
  const int32_t* n_cand;
  const int32_t* cand_pos;
  const int32_t* n_xq;
  const uint4 *wq_frag, *kc_frag, *vc_frag;
  const unsigned char* w1_can;  // fc1' chunks (tcgen05 B operand)
  const float *bq_eff, *b1_eff;
  int nks;                   // capacity of the key fragments in 16-key steps
  int use_xattn;
  float* scores;             // by position
};

__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// erf-GELU (exact GELU, not the tanh form) as  gelu(x) = max(x, 0) - |x| q(|x|),  q(a) = Phi(-a) =
// 0.5 erfc(a / sqrt 2) = 2^P(a)  with P a degree-7 polynomial fitted (weighted minimax over a in [0, 6], weight a q(a):
// the error of gelu itself) to log2(0.5 erfc(a / sqrt 2)); beyond a = 6, q < 1e-9 and a is clamped.  Against fp64 the
// fp32 Horner evaluation is within 7e-8 absolute over [-8, 8] (Abramowitz & Stegun 7.1.26, used before: 2.1e-7, and a
// reciprocal more).  One MUFU and 8 FMAs per element; the coefficients below are those of P(-n) for n = -|x|.
constexpr float GELU_A = 6.0f;
constexpr float GELU_C0 = -1.0f, GELU_C1 = 1.151126929e+00f, GELU_C2 = -4.590439269e-01f, GELU_C3 = 5.294857004e-02f,
                GELU_C4 = 7.670789278e-03f, GELU_C5 = 5.757889713e-04f, GELU_C6 = -1.279755249e-05f,
                GELU_C7 = -4.278683871e-06f;
__device__ __forceinline__ float gelu_erf(float x) {
  const float nax = -fabsf(x), n = fmaxf(nax, -GELU_A);
  float pl = fmaf(GELU_C7, n, GELU_C6);
  pl = fmaf(pl, n, GELU_C5);
  pl = fmaf(pl, n, GELU_C4);
  pl = fmaf(pl, n, GELU_C3);
  pl = fmaf(pl, n, GELU_C2);
  pl = fmaf(pl, n, GELU_C1);
  pl = fmaf(pl, n, GELU_C0);
  return fmaf(nax, ex2f(pl), fmaxf(x, 0.f));
}

// Two fp32 lanes per instruction (fma.rn.f32x2, sm_100): the epilogue and softmax loops of k_tail_tc are bound by
// the FMA pipe's issue rate, which a packed instruction uses once for two elements.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
// gelu of two values, same arithmetic as gelu_erf (bit-identical results)
__device__ __forceinline__ f32x2 gelu_erf2(f32x2 x) {
  float x0, x1;
  upk2(x, x0, x1);
  const float na0 = -fabsf(x0), na1 = -fabsf(x1);
  const f32x2 n = pk2(fmaxf(na0, -GELU_A), fmaxf(na1, -GELU_A));
  f32x2 pl = fma2(pk2(GELU_C7, GELU_C7), n, pk2(GELU_C6, GELU_C6));
  pl = fma2(pl, n, pk2(GELU_C5, GELU_C5));
  pl = fma2(pl, n, pk2(GELU_C4, GELU_C4));
  pl = fma2(pl, n, pk2(GELU_C3, GELU_C3));
  pl = fma2(pl, n, pk2(GELU_C2, GELU_C2));
  pl = fma2(pl, n, pk2(GELU_C1, GELU_C1));
  pl = fma2(pl, n, pk2(GELU_C0, GELU_C0));
  float p0, p1;
  upk2(pl, p0, p1);
  return fma2(pk2(na0, na1), pk2(ex2f(p0), ex2f(p1)), pk2(fmaxf(x0, 0.f), fmaxf(x1, 0.f)));
}

// ---- k_residual_mma: CTA = R_CWARPS consumer warps (one 16-candidate tile each) + 1 producer / MMA-issuer warp.
// Q projection and cross-attention run per warp in registers on mma.sync; their B fragments are laid out in global
// memory in consumption order and streamed by the producer as bulk copies (TMA unit) through a ring of RS_BYTES stages.
// fc1 -- the dense contraction of the head, (tokens x (D+128)) x ((D+128) x 256) -- runs on tcgen05: the consumer warps
// write their [kbar | c] rows, split into bf16 hi and lo parts, into shared memory in the canonical K-major layout (A
// operand, M = 128 rows per CTA of which 16 R_CWARPS are used), the producer streams the folded fc1 chunks (B operand,
// 128 hidden units x 64 k, hi | lo) into the dead ring and one thread issues hi*hi + lo*hi + hi*lo as tcgen05.mma
// kind::f16 into two 128-column accumulators in TMEM; warps 0-3 read them back with tcgen05.ld (one token row per
// thread) for the epilogue: + b1' + rule w_r, erf-GELU, fc2 dot, s = rule + alpha z.
// Ring stage sequence (identical in producer and consumers), nq > 0 only:
//   KS stages W_Q' k-step s (16 n-tiles); per head, per chunk of 64 query keys: 1 stage Kc, 1 stage Vc.
constexpr int R_CWARPS = 7;
constexpr int R_THREADS = (R_CWARPS + 2) * 32;  // + ring producer warp + fc1 loader / MMA issuer warp
constexpr int RS_BYTES = 8192;
constexpr int RS_STAGES = 4;
constexpr int R_TMEM_COLS = 256;
template <int D>
constexpr int resid_smem() {
  // ring | two fc1 chunk buffers | A hi | A lo (16 R_CWARPS rows each) | epilogue vectors (b1', w_r, fc2), z halves |
  // barriers + tmem base
  return RS_STAGES * RS_BYTES + 2 * W1C_CHUNK + 2 * (R_CWARPS * 16) * (D + R_DC) * 2 + 3 * R_HID * 4 + 2 * 128 * 4 + 256;
}

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  // shared-memory matrix descriptor, SWIZZLE_NONE: start address, leading (K) and stride (M/N) byte offsets between
  // core matrices, all >> 4; version 1 (sm_100)
  return (uint64_t)((saddr >> 4) & 0x3fff) | ((uint64_t)((lbo >> 4) & 0x3fff) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3fff) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int D>
__global__ __launch_bounds__(R_THREADS, 1) void k_residual_mma(const ResidMmaParams p, const ResidW w) {  // 9 warps
  constexpr int KS = D / 16;
  constexpr int KA = D + R_DC;                 // K of fc1 = row length of the A operand
  constexpr int A_PART = R_CWARPS * 16 * KA * 2;  // bytes of A hi (and of A lo); the MMA's rows 112..127 read past it
  constexpr int A_SBO = (KA / 8) * 128;        // byte distance between 8-row groups of A
  constexpr int KCK = D / 64;                  // 64-wide K chunks of the kbar columns
  constexpr int NKC = KCK + 2;                 // ... then the two c chunks
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  // A first: the MMA's unused rows 112..127 of a_lo then fall into the chunk buffers, inside the allocation
  extern __shared__ __align__(128) unsigned char a_hi[];
  unsigned char* a_lo = a_hi + A_PART;
  unsigned char* bbuf = a_lo + A_PART;                     // two fc1 chunk buffers
  unsigned char* ring = bbuf + 2 * W1C_CHUNK;              // [RS_STAGES][RS_BYTES]
  float* ep_b1 = reinterpret_cast<float*>(ring + RS_STAGES * RS_BYTES);  // [256] b1', then w_r, then fc2_w
  float* ep_wr = ep_b1 + R_HID;
  float* ep_w2 = ep_wr + R_HID;
  float* ep_z = ep_w2 + R_HID;                 // [2][128] fc2 partial dots of the two accumulator halves
  uint64_t* full = reinterpret_cast<uint64_t*>(ep_z + 2 * 128);
  uint64_t* empty = full + RS_STAGES;
  uint64_t* a_ready = empty + RS_STAGES;       // [2]: kbar columns of A written / c columns written (all consumer warps)
  uint64_t* bfull = a_ready + 2;               // [2] fc1 chunk landed
  uint64_t* bempty = bfull + 2;                // [2] its MMAs have completed
  uint64_t* tfull = bempty + 2;                // [2] accumulator half complete
  uint32_t* tmem_base_p = reinterpret_cast<uint32_t*>(tfull + 2);
  const int nc = *p.n_cand;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, r = lane >> 2, q = lane & 3;
  if (blockIdx.x * R_CWARPS * 16 >= nc) return;
  const int nq = p.use_xattn ? *p.n_xq : 0;
  const int nkt = 2 * p.nks;
  const int P = 3 * D + 1, IN = P + R_DC;
  if (threadIdx.x == 0) {
    for (int s = 0; s < RS_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], R_CWARPS); }
    mbar_init(&a_ready[0], R_CWARPS);
    mbar_init(&a_ready[1], R_CWARPS);
    for (int i = 0; i < 2; ++i) { mbar_init(&bfull[i], 1); mbar_init(&bempty[i], 1); mbar_init(&tfull[i], 1); }
    mbar_fence_init();
  }
  for (int n = threadIdx.x; n < R_HID; n += R_THREADS) {
    ep_b1[n] = p.b1_eff[n];
    ep_wr[n] = __ldg(w.fc1_w + (int64_t)n * IN + 3 * D);
    ep_w2[n] = __ldg(w.fc2_w + n);
  }
  if (warp == R_CWARPS + 1) {  // the MMA warp owns the tensor-memory allocation
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_p)), "n"(R_TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_base_p;

  if (warp == R_CWARPS + 1) {
    // ------------------------------------------------------------------ fc1 on tcgen05: chunk loader and MMA issuer.
    // The kbar columns of A are written at kernel start, so their chunks are multiplied while the consumer warps are
    // still in the Q projection and the cross attention; only the c chunks wait for them.
    if (lane == 0) {
      // instruction descriptor: D fp32, A and B bf16, both K-major, N = 128, M = 128
      const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
      const int n_k = 2 * KCK, n_chunks = n_k + (nq > 0 ? 4 : 0);
      auto chunk_id = [&](int i, int& nh, int& kc) {  // kbar chunks of both halves first, then the c chunks
        if (i < n_k) { nh = i / KCK; kc = i % KCK; } else { nh = (i - n_k) >> 1; kc = KCK + ((i - n_k) & 1); }
      };
      auto load_chunk = [&](int i) {
        int nh, kc;
        chunk_id(i, nh, kc);
        const int b = i & 1;
        mbar_arrive_expect_tx(&bfull[b], (uint32_t)W1C_CHUNK);
        bulk_g2s(bbuf + b * W1C_CHUNK, p.w1_can + (size_t)(nh * NKC + kc) * W1C_CHUNK, (uint32_t)W1C_CHUNK, &bfull[b]);
      };
      load_chunk(0);
      if (n_chunks > 1) load_chunk(1);
      mbar_wait(&a_ready[0], 0u);
      for (int i = 0; i < n_chunks; ++i) {
        int nh, kc;
        chunk_id(i, nh, kc);
        const int b = i & 1;
        if (i == n_k) mbar_wait(&a_ready[1], 0u);
        mbar_wait(&bfull[b], (uint32_t)(i >> 1) & 1u);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t bb = smem_u32(bbuf + b * W1C_CHUNK);
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
          const uint32_t a_off = (uint32_t)((kc * 8 + ks * 2) * 128);
          const uint64_t dah = umma_desc(smem_u32(a_hi) + a_off, 128, A_SBO);
          const uint64_t dal = umma_desc(smem_u32(a_lo) + a_off, 128, A_SBO);
          const uint64_t dbh = umma_desc(bb + ks * 256, 128, 1024);
          const uint64_t dbl = umma_desc(bb + W1C_PART + ks * 256, 128, 1024);
          const uint32_t td = tmem + (uint32_t)(nh * 128);
          umma_bf16(td, dah, dbh, idesc, (kc | ks) ? 1u : 0u);
          umma_bf16(td, dal, dbh, idesc, 1u);
          umma_bf16(td, dah, dbl, idesc, 1u);
        }
        umma_commit(&bempty[b]);
        if (kc == (nq > 0 ? NKC : KCK) - 1) umma_commit(&tfull[nh]);
        if (i + 2 < n_chunks) {
          mbar_wait(&bempty[b], (uint32_t)(i >> 1) & 1u);  // the MMAs reading this buffer are done
          load_chunk(i + 2);
        }
      }
    }
    __syncwarp();
    __syncthreads();  // z halves written
    __syncthreads();  // epilogue finished
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(R_TMEM_COLS));
    return;
  }

  if (warp == R_CWARPS) {
    // ------------------------------------------------------------------ ring producer (then joins the epilogue)
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      auto push = [&](const uint4* src0, uint32_t bytes0, const uint4* src1, uint32_t bytes1) {
        mbar_wait(&empty[s], ph ^ 1u);
        mbar_arrive_expect_tx(&full[s], bytes0 + bytes1);
        bulk_g2s(ring + s * RS_BYTES, src0, bytes0, &full[s]);
        if (bytes1) bulk_g2s(ring + s * RS_BYTES + bytes0, src1, bytes1, &full[s]);
        if (++s == RS_STAGES) { s = 0; ph ^= 1u; }
      };
      if (nq > 0) {
        for (int ks = 0; ks < KS; ++ks) push(p.wq_frag + ks * 16 * 32, 16 * 512, nullptr, 0);
        for (int hc = 0; hc < R_HC; ++hc)
          for (int kc0 = 0; kc0 < nq; kc0 += 64) {
            const int ntn = min(8, (nq - kc0 + 7) >> 3), nv = (ntn + 1) >> 1;
            push(p.kc_frag + ((int64_t)(hc * 2) * nkt + (kc0 >> 3)) * 32, ntn * 512,
                 p.kc_frag + ((int64_t)(hc * 2 + 1) * nkt + (kc0 >> 3)) * 32, ntn * 512);
            push(p.vc_frag + ((int64_t)(hc * p.nks + (kc0 >> 4)) * 4) * 32, nv * 4 * 512, nullptr, 0);
          }
      }
    }
    __syncwarp();
  } else {
  // -------------------------------------------------------------------- consumers
  const int t0 = (blockIdx.x * R_CWARPS + warp) * 16;
  const bool live = t0 < nc;  // warps past the end still walk the ring
  const int row0 = min(t0 + r, nc - 1), row1 = min(t0 + r + 8, nc - 1);
  const float rule0 = p.rule_c[row0], rule1 = p.rule_c[row1];
  const uint32_t ring_u32 = smem_u32(ring) + lane * 16;
  int rs = 0;
  uint32_t rph = 0;
  auto stage_wait = [&]() -> uint32_t {
    mbar_wait(&full[rs], rph);
    return ring_u32 + rs * RS_BYTES;
  };
  auto stage_done = [&]() {
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[rs]);
    if (++rs == RS_STAGES) { rs = 0; rph ^= 1u; }
  };

  // A fragments of kbar (hi | lo); k order per kperm()
  uint32_t akh[KS][4], akl[KS][4];
#pragma unroll
  for (int s = 0; s < KS; ++s) {
    const float4 x0 = __ldg(reinterpret_cast<const float4*>(p.kbar + (int64_t)row0 * D + s * 16 + 4 * q));
    const float4 x1 = __ldg(reinterpret_cast<const float4*>(p.kbar + (int64_t)row1 * D + s * 16 + 4 * q));
    split_bf16(x0.x, x0.y, akh[s][0], akl[s][0]);
    split_bf16(x1.x, x1.y, akh[s][1], akl[s][1]);
    split_bf16(x0.z, x0.w, akh[s][2], akl[s][2]);
    split_bf16(x1.z, x1.w, akh[s][3], akl[s][3]);
  }

  // the same values as rows of the fc1 A operand (canonical K-major layout, natural k order)
  const uint32_t a_row0 = (uint32_t)((warp * 2) * A_SBO + r * 16), a_row1 = a_row0 + (uint32_t)A_SBO;
#pragma unroll
  for (int s = 0; s < KS; ++s) {
    const uint32_t ko = (uint32_t)((2 * s + (q >> 1)) * 128 + (q & 1) * 8);
    *reinterpret_cast<uint2*>(a_hi + a_row0 + ko) = make_uint2(akh[s][0], akh[s][2]);
    *reinterpret_cast<uint2*>(a_hi + a_row1 + ko) = make_uint2(akh[s][1], akh[s][3]);
    *reinterpret_cast<uint2*>(a_lo + a_row0 + ko) = make_uint2(akl[s][0], akl[s][2]);
    *reinterpret_cast<uint2*>(a_lo + a_row1 + ko) = make_uint2(akl[s][1], akl[s][3]);
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // publish the rows to the async proxy (tcgen05.mma)
  __syncwarp();
  if (lane == 0) mbar_arrive(&a_ready[0]);

  if (nq > 0) {
    // ---- Q = Wq' kbar + rule wq_r + bq'
    float accq[16][4];
#pragma unroll
    for (int t = 0; t < 16; ++t) { accq[t][0] = accq[t][1] = accq[t][2] = accq[t][3] = 0.f; }
#pragma unroll
    for (int s = 0; s < KS; ++s) {
      const uint32_t sb = stage_wait();
#pragma unroll
      for (int t = 0; t < 16; ++t) mma3(accq[t], akh[s], akl[s], lds128(sb + t * 512));
      stage_done();
    }
#pragma unroll
    for (int t = 0; t < 16; ++t) {
      const int n = t * 8 + 2 * q;
      const float2 b = *reinterpret_cast<const float2*>(p.bq_eff + n);
      const float wr0 = __ldg(w.wq + (int64_t)n * P + 3 * D), wr1 = __ldg(w.wq + (int64_t)(n + 1) * P + 3 * D);
      accq[t][0] += fmaf(rule0, wr0, b.x); accq[t][1] += fmaf(rule0, wr1, b.y);
      accq[t][2] += fmaf(rule1, wr0, b.x); accq[t][3] += fmaf(rule1, wr1, b.y);
    }
    // ---- 4-head cross attention, online softmax in the exp2 domain over chunks of 64 query keys
#pragma unroll
    for (int hc = 0; hc < R_HC; ++hc) {
      uint32_t qh[2][4], ql[2][4];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int ta = hc * 4 + 2 * u, tb = ta + 1;
        split_bf16(accq[ta][0], accq[ta][1], qh[u][0], ql[u][0]);
        split_bf16(accq[ta][2], accq[ta][3], qh[u][1], ql[u][1]);
        split_bf16(accq[tb][0], accq[tb][1], qh[u][2], ql[u][2]);
        split_bf16(accq[tb][2], accq[tb][3], qh[u][3], ql[u][3]);
      }
      float m0 = -CUDART_INF_F, m1 = -CUDART_INF_F, l0 = 0.f, l1 = 0.f;
      float o[4][4];
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) { o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f; }
      for (int kc0 = 0; kc0 < nq; kc0 += 64) {
        const int ntn = min(8, (nq - kc0 + 7) >> 3);
        float sc[8][4];
        {
          const uint32_t sb = stage_wait();  // [u][ntn tiles]
#pragma unroll
          for (int t = 0; t < 8; ++t) {
            sc[t][0] = sc[t][1] = sc[t][2] = sc[t][3] = 0.f;
            if (t < ntn) {
#pragma unroll
              for (int u = 0; u < 2; ++u) mma3(sc[t], qh[u], ql[u], lds128(sb + (u * ntn + t) * 512));
            }
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const bool ok = t < ntn && (kc0 + t * 8 + 2 * q + e) < nq;
              if (!ok) { sc[t][e] = -CUDART_INF_F; sc[t][2 + e] = -CUDART_INF_F; }
            }
          }
          stage_done();
        }
        float x0 = -CUDART_INF_F, x1 = -CUDART_INF_F;
#pragma unroll
        for (int t = 0; t < 8; ++t) {
          x0 = fmaxf(x0, fmaxf(sc[t][0], sc[t][1]));
          x1 = fmaxf(x1, fmaxf(sc[t][2], sc[t][3]));
        }
        x0 = fmaxf(x0, __shfl_xor_sync(0xffffffffu, x0, 1)); x0 = fmaxf(x0, __shfl_xor_sync(0xffffffffu, x0, 2));
        x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, 1)); x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, 2));
        const float n0 = fmaxf(m0, x0), n1 = fmaxf(m1, x1);  // finite: every chunk holds at least one live key
        const float c0 = ex2f(m0 - n0), c1 = ex2f(m1 - n1);
        m0 = n0; m1 = n1;
        l0 *= c0; l1 *= c1;
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) { o[nt][0] *= c0; o[nt][1] *= c0; o[nt][2] *= c1; o[nt][3] *= c1; }
#pragma unroll
        for (int t = 0; t < 8; ++t) {
          sc[t][0] = ex2f(sc[t][0] - n0); sc[t][1] = ex2f(sc[t][1] - n0);
          sc[t][2] = ex2f(sc[t][2] - n1); sc[t][3] = ex2f(sc[t][3] - n1);
          l0 += sc[t][0] + sc[t][1];
          l1 += sc[t][2] + sc[t][3];
        }
        {
          const uint32_t sb = stage_wait();  // [nv key steps][4 tiles]
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            if (2 * v < ntn) {
              uint32_t ph[4], pl[4];
              split_bf16(sc[2 * v][0], sc[2 * v][1], ph[0], pl[0]);
              split_bf16(sc[2 * v][2], sc[2 * v][3], ph[1], pl[1]);
              split_bf16(sc[2 * v + 1][0], sc[2 * v + 1][1], ph[2], pl[2]);
              split_bf16(sc[2 * v + 1][2], sc[2 * v + 1][3], ph[3], pl[3]);
#pragma unroll
              for (int nt = 0; nt < 4; ++nt) mma3(o[nt], ph, pl, lds128(sb + (v * 4 + nt) * 512));
            }
          }
          stage_done();
        }
      }
      l0 += __shfl_xor_sync(0xffffffffu, l0, 1); l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
      l1 += __shfl_xor_sync(0xffffffffu, l1, 1); l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
      const float i0 = 1.f / l0, i1 = 1.f / l1;
      // c_h (Eq. 6) -> columns D + 32 hc .. of the fc1 A operand, hi and lo parts
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) {
        const uint32_t ko = (uint32_t)((D / 8 + hc * 4 + nt) * 128 + q * 4);
        uint32_t h0, l0b, h1, l1b;
        split_bf16(o[nt][0] * i0, o[nt][1] * i0, h0, l0b);
        split_bf16(o[nt][2] * i1, o[nt][3] * i1, h1, l1b);
        *reinterpret_cast<uint32_t*>(a_hi + a_row0 + ko) = h0;
        *reinterpret_cast<uint32_t*>(a_lo + a_row0 + ko) = l0b;
        *reinterpret_cast<uint32_t*>(a_hi + a_row1 + ko) = h1;
        *reinterpret_cast<uint32_t*>(a_lo + a_row1 + ko) = l1b;
      }
    }
  }

  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the c columns of A
  __syncwarp();
  if (lane == 0) mbar_arrive(&a_ready[1]);
  (void)live; (void)rule0; (void)rule1;
  }  // consumer warps

  // ---- epilogue, warps 0..7: warp w reads TMEM lanes 32 (w % 4) .. + 31 (token rows) of accumulator half w / 4:
  // hid = acc + b1' + rule w_r -> erf-GELU -> fc2 dot; the two halves of a row are added through shared memory
  {
    const int qd = warp & 3, nh = warp >> 2;
    const int m = qd * 32 + lane;
    const int tok = blockIdx.x * R_CWARPS * 16 + m;
    const bool valid = (m < R_CWARPS * 16) && (tok < nc);
    const float rule = valid ? p.rule_c[tok] : 0.f;
    float z = 0.f;
    mbar_wait(&tfull[nh], 0u);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
    for (int c0 = 0; c0 < 128; c0 += 16) {
      uint32_t v[16];
      const uint32_t taddr = tmem + ((uint32_t)(qd * 32) << 16) + (uint32_t)(nh * 128 + c0);
      asm volatile(
          "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
          : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
            "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
          : "r"(taddr));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int n = nh * 128 + c0 + j;
        z = fmaf(ep_w2[n], gelu_erf(__uint_as_float(v[j]) + fmaf(rule, ep_wr[n], ep_b1[n])), z);
      }
    }
    ep_z[nh * 128 + m] = z;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (nh == 0 && valid) p.scores[p.cand_pos[tok]] = rule + w.alpha * ((ep_z[m] + ep_z[128 + m]) + w.fc2_b[0]);
    __syncthreads();  // the MMA warp frees the tensor memory after this
  }
}

}  // namespace ikv
