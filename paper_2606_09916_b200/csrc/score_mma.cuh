// score_mma.cuh -- the bf16 key pass of the rule scorer (Eq. 3) and the mean key of Eq. 5
// as ONE persistent streaming kernel for sm_100a.
//
//   producer warp : per (16-token tile, layer) one 1-D bulk copy (TMA unit, UBLKCP) per token row
//                   [H_kv][D] bf16 (2 KB at Qwen3-8B shape) through the slot map into a ring of shared-memory
//                   stages, completion on an mbarrier (full[stage]); waits on empty[stage] before reuse.
//   consumer warps: warp w owns KV head(s) w, w+8, ...; the 16 x D key tile is the A operand of
//                   mma.sync.m16n8k16 (bf16 in, fp32 accumulate); the B operand holds the G memory rows of the
//                   group, each split into a bf16 hi and a bf16 lo part (two columns), so that
//                   hi + lo carries ~16 mantissa bits of M / sqrt(D) and keys are exact => fp32-grade logits.
//                   The contraction has only G (<= 8) useful columns: it is not a tcgen05 tile (R1);
//                   the tensor pipe is used here to keep the FMA pipe free, the kernel is HBM-bound.
//   Per (layer, head): logits -> scratch [L*Hq][ldc] (fp32), running (max, sum exp) per CTA in shared memory,
//   key bytes -> fp32 k_bar accumulators in registers (Eq. 5), reduced over the 8 head-warps per tile.
//   Tiles [0, ceil(n_cand/16)) are the candidates; the tiles after them are the live cross-attention positions
//   (K^q of Eq. 6, R7/R8) for which only the mean key is produced.
#pragma once
#include "common.cuh"
#include "pipe.cuh"

namespace ikv {

constexpr int KP_TOK = 16;       // tokens per stage = M of the mma
constexpr int KP_CWARPS = 8;     // consumer warps
constexpr int KP_THREADS = (KP_CWARPS + 1) * 32;
constexpr int KP_ROWPAD = 64;    // bytes added to each staged token row (bank spread for the 16-byte reads)

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  const uint32_t l = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(lo));
  const uint32_t h = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(hi));
  return l | (h << 16);
}

// B fragments of M / sqrt(D):  frag[((l*Hkv + kvh)*NT + nt)*(KS/2) + v][lane] (uint4), KS = D/16 k-steps,
// uint4 v = {b0, b1 of k-step 2v, b0, b1 of k-step 2v+1}.  k-order inside the tile follows the 16-byte key
// loads of the consumer: lane (r = lane/4, q = lane%4), load i covers d = 8(q+4i) .. +7;
// k-step s = 2i+j uses d = 8(q+4i) + 4j + {0,1} (b0) and + {2,3} (b1).  Column n = r:
//   G <= 4 (NT = 1): n = 2g -> hi(M[l, kvh*G+g]), n = 2g+1 -> lo;      G > 4 (NT = 2): tile 0 hi, tile 1 lo, n = g.
template <int D, int G>
__global__ void k_memory_frags(const float* __restrict__ M, int L, int Hkv, float inv_sqrt_d, uint4* __restrict__ frag) {
  constexpr int KS = D / 16, NT = (G <= 4) ? 1 : 2;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int total = L * Hkv * NT * (KS / 2) * 32;
  if (idx >= total) return;
  const int lane = idx & 31;
  int t = idx >> 5;
  const int v = t % (KS / 2); t /= (KS / 2);
  const int nt = t % NT; t /= NT;
  const int kvh = t % Hkv;
  const int l = t / Hkv;
  const int r = lane >> 2, q = lane & 3;
  int g, part;  // part 0 = hi, 1 = lo
  if (NT == 1) { g = r >> 1; part = r & 1; } else { g = r; part = nt; }
  uint32_t out[4];
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      float val[2];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        float x = 0.f;
        if (g < G) {
          const int d = 8 * (q + 4 * v) + 4 * j + 2 * b + e;
          const float m = M[((int64_t)l * Hkv * G + kvh * G + g) * D + d] * inv_sqrt_d;
          const float hi = __bfloat162float(__float2bfloat16_rn(m));
          x = part ? (m - hi) : hi;
        }
        val[e] = x;
      }
      out[j * 2 + b] = pack_bf16x2(val[0], val[1]);
    }
  frag[idx] = make_uint4(out[0], out[1], out[2], out[3]);
}

struct KeyPassParams {
  const bf16* k_pool;
  int64_t layer_stride;  // elements
  int L, Hkv;
  const uint4* frag;
  const int32_t* cand_slot;
  const int32_t* n_cand;
  const int32_t* xq_slot;  // may be NULL
  const int32_t* n_xq;     // may be NULL
  float* logits;           // [L*Hq][ldc]
  int64_t ldc;
  float2* partials;        // [L*Hq][gridDim.x]
  float* kbar;             // [n_cand][D]   (KBAR)
  float* kq;               // [n_xq][D]     (KBAR)
  int n_stage;
};

template <int D, int G, bool KBAR>
__global__ __launch_bounds__(KP_THREADS, 1) void k_key_pass(const KeyPassParams p) {
  constexpr int KS = D / 16, NI = D / 32, NT = (G <= 4) ? 1 : 2;
  constexpr int RSTR = D + 4;  // row stride (floats) of the k_bar reduction buffer
  const int L = p.L, Hkv = p.Hkv, Hq = Hkv * G;
  const int row_bytes = Hkv * D * 2;
  const int row_stride = row_bytes + KP_ROWPAD;
  const int stage_bytes = KP_TOK * row_stride;
  const int NS = p.n_stage;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* stage_base = smem_raw;                                     // [NS][16][row_stride]
  float2* stats = (float2*)(stage_base + (size_t)NS * stage_bytes);          // [L*Hq]
  uint64_t* full = (uint64_t*)(stats + (size_t)L * Hq);                      // [NS]
  uint64_t* empty = full + NS;                                               // [NS]
  float* red = (float*)(empty + NS);                                         // [KP_CWARPS][16][RSTR] if KBAR

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nc = *p.n_cand;
  const int nx = (KBAR && p.n_xq) ? *p.n_xq : 0;
  const int tiles_c = (nc + KP_TOK - 1) / KP_TOK;
  const int tiles = tiles_c + (nx + KP_TOK - 1) / KP_TOK;

  for (int i = threadIdx.x; i < L * Hq; i += KP_THREADS) stats[i] = make_float2(-CUDART_INF_F, 0.f);
  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], KP_CWARPS); }
    mbar_fence_init();
  }
  __syncthreads();

  if (warp == KP_CWARPS) {
    // ------------------------------------------------------------------ producer
    int it = 0;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
      const bool is_x = tile >= tiles_c;
      const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
      const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
      int64_t slot = 0;
      if (lane < nvalid) slot = is_x ? p.xq_slot[t0 + lane] : p.cand_slot[t0 + lane];
      const bf16* src = p.k_pool + slot * (int64_t)(Hkv * D);
      for (int l = 0; l < L; ++l, ++it) {
        const int s = it % NS;
        const uint32_t ph = (uint32_t)(it / NS) & 1u;
        if (lane == 0) {
          mbar_wait(&empty[s], ph ^ 1u);
          mbar_arrive_expect_tx(&full[s], (uint32_t)(nvalid * row_bytes));
        }
        __syncwarp();
        if (lane < nvalid)
          bulk_g2s(stage_base + (size_t)s * stage_bytes + lane * row_stride, src + (int64_t)l * p.layer_stride,
                   (uint32_t)row_bytes, &full[s]);
      }
    }
  } else {
    // ------------------------------------------------------------------ consumers
    const int r = lane >> 2, q = lane & 3;
    const uint32_t stage_u32 = smem_u32(stage_base);
    int it = 0;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
      const bool is_x = tile >= tiles_c;
      const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
      const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
      float kb[KBAR ? 2 : 1][KBAR ? NI : 1][8];
      if (KBAR) {
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
          for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int e = 0; e < 8; ++e) kb[a][i][e] = 0.f;
      }
      for (int l = 0; l < L; ++l, ++it) {
        const int s = it % NS;
        const uint32_t ph = (uint32_t)(it / NS) & 1u;
        mbar_wait(&full[s], ph);
        const uint32_t sb = stage_u32 + (uint32_t)(s * stage_bytes);
        for (int kvh = warp; kvh < Hkv; kvh += KP_CWARPS) {
          // B fragments of this (layer, head)
          const uint4* fp = p.frag + ((int64_t)(l * Hkv + kvh) * NT) * (KS / 2) * 32 + lane;
          uint4 bf[NT][KS / 2];
#pragma unroll
          for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int v = 0; v < KS / 2; ++v) bf[nt][v] = __ldg(fp + (nt * (KS / 2) + v) * 32);
          uint4 ka[NI], kc[NI];
          const uint32_t a_lo = sb + (uint32_t)(r * row_stride + kvh * D * 2 + q * 16);
          const uint32_t a_hi = a_lo + (uint32_t)(8 * row_stride);
#pragma unroll
          for (int i = 0; i < NI; ++i) {
            ka[i] = lds128(a_lo + i * 64);
            kc[i] = lds128(a_hi + i * 64);
          }
          float c[NT][4];
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) { c[nt][0] = c[nt][1] = c[nt][2] = c[nt][3] = 0.f; }
#pragma unroll
          for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              mma_bf16_16816(c[nt], ka[i].x, kc[i].x, ka[i].y, kc[i].y, bf[nt][i].x, bf[nt][i].y);
              mma_bf16_16816(c[nt], ka[i].z, kc[i].z, ka[i].w, kc[i].w, bf[nt][i].z, bf[nt][i].w);
            }
          if (KBAR) {
#pragma unroll
            for (int i = 0; i < NI; ++i) {
              const uint32_t ua[4] = {ka[i].x, ka[i].y, ka[i].z, ka[i].w};
              const uint32_t uc[4] = {kc[i].x, kc[i].y, kc[i].z, kc[i].w};
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                kb[0][i][2 * e] += bf16lo(ua[e]);
                kb[0][i][2 * e + 1] += bf16hi(ua[e]);
                kb[1][i][2 * e] += bf16lo(uc[e]);
                kb[1][i][2 * e + 1] += bf16hi(uc[e]);
              }
            }
          }
          if (!is_x) {
            // logits of this thread: NH heads x 2 tokens (r, r+8)
            constexpr int NH = (NT == 1) ? 1 : 2;
            float x[NH][2];
            int g0;
            if (NT == 1) {
              g0 = q;
              x[0][0] = c[0][0] + c[0][1];
              x[0][1] = c[0][2] + c[0][3];
            } else {
              g0 = 2 * q;
              x[0][0] = c[0][0] + c[NT - 1][0];
              x[NH - 1][0] = c[0][1] + c[NT - 1][1];
              x[0][1] = c[0][2] + c[NT - 1][2];
              x[NH - 1][1] = c[0][3] + c[NT - 1][3];
            }
            const bool v0 = r < nvalid, v1 = (r + 8) < nvalid;
#pragma unroll
            for (int hh = 0; hh < NH; ++hh) {
              const int g = g0 + hh;
              const bool gv = g < G;
              const int lh = l * Hq + kvh * G + (gv ? g : 0);
              float* lrow = p.logits + (int64_t)lh * p.ldc + t0;
              if (gv && v0) lrow[r] = x[hh][0];
              if (gv && v1) lrow[r + 8] = x[hh][1];
              float mx = fmaxf(v0 ? x[hh][0] : -CUDART_INF_F, v1 ? x[hh][1] : -CUDART_INF_F);
              mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
              mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
              mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
              float se = (v0 ? __expf(x[hh][0] - mx) : 0.f) + (v1 ? __expf(x[hh][1] - mx) : 0.f);
              se += __shfl_xor_sync(0xffffffffu, se, 4);
              se += __shfl_xor_sync(0xffffffffu, se, 8);
              se += __shfl_xor_sync(0xffffffffu, se, 16);
              if (r == 0 && gv) {
                const float2 st = stats[lh];
                const float mn = fmaxf(st.x, mx);
                stats[lh] = make_float2(mn, st.y * __expf(st.x - mn) + se * __expf(mx - mn));
              }
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
      }
      if (KBAR) {
        // reduce the per-head-warp partial sums of this tile and write the mean key
        const int nw = min(KP_CWARPS, Hkv);
        if (warp < nw) {
          float* dst = red + ((size_t)warp * KP_TOK) * RSTR;
#pragma unroll
          for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int i = 0; i < NI; ++i) {
              float4* d4 = reinterpret_cast<float4*>(dst + (size_t)(r + 8 * a) * RSTR + 8 * (q + 4 * i));
              d4[0] = make_float4(kb[a][i][0], kb[a][i][1], kb[a][i][2], kb[a][i][3]);
              d4[1] = make_float4(kb[a][i][4], kb[a][i][5], kb[a][i][6], kb[a][i][7]);
            }
        }
        bar_sync(1, KP_CWARPS * 32);
        const float inv = 1.f / (float)(L * Hkv);
        float* outp = is_x ? p.kq : p.kbar;
        for (int o = threadIdx.x; o < nvalid * D; o += KP_CWARPS * 32) {
          const int tok = o / D, d = o % D;
          float acc = 0.f;
          for (int w = 0; w < nw; ++w) acc += red[((size_t)w * KP_TOK + tok) * RSTR + d];
          outp[(int64_t)(t0 + tok) * D + d] = acc * inv;
        }
        bar_sync(1, KP_CWARPS * 32);
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < L * Hq; i += KP_THREADS) p.partials[(int64_t)i * gridDim.x + blockIdx.x] = stats[i];
}

// shared memory of k_key_pass; returns 0 if not even two stages fit
inline size_t key_pass_smem(int L, int Hq, int Hkv, int D, bool kbar, int max_smem, int* n_stage) {
  const size_t stage = (size_t)KP_TOK * (Hkv * D * 2 + KP_ROWPAD);
  const size_t fixed = (size_t)L * Hq * 8 + 2 * 8 * 8 + (kbar ? (size_t)KP_CWARPS * KP_TOK * (D + 4) * 4 : 0) + 128;
  if (fixed + 2 * stage > (size_t)max_smem) { *n_stage = 0; return 0; }
  int ns = (int)(((size_t)max_smem - fixed) / stage);
  if (ns > 8) ns = 8;
  *n_stage = ns;
  return fixed + (size_t)ns * stage;
}

// ---------------------------------------------------------------------------------------------
// a3  rule_c = sum_{l,h} exp(x[l,h,c] - lse[l,h])   (Eq. 3).  One CTA of 256 threads per 64 candidates:
// thread (cq = tid % 16 -> 4 candidates, lg = tid / 16 -> rows lg, lg+16, ...), 16-byte loads.
// ---------------------------------------------------------------------------------------------
__global__ __launch_bounds__(256) void k_score_rule4(const float* __restrict__ logits, int64_t ldc, int LH,
                                                     const float* __restrict__ lse,
                                                     const int32_t* __restrict__ n_cand_p,
                                                     const int32_t* __restrict__ cand_pos, float* __restrict__ rule_c,
                                                     float* __restrict__ scores, int scatter_scores,
                                                     float* __restrict__ rule_out) {
  __shared__ float4 part[16][16];
  const int nc = *n_cand_p;
  const int c0 = blockIdx.x * 64;
  if (c0 >= nc) return;
  const int cq = threadIdx.x & 15, lg = threadIdx.x >> 4;
  const int c = c0 + cq * 4;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  if (c < nc) {  // rows are padded to a multiple of 4 (ldc % 4 == 0); lanes past n_cand read scratch, never stored
#pragma unroll 6
    for (int lh = lg; lh < LH; lh += 16) {
      const float4 v = *reinterpret_cast<const float4*>(logits + (int64_t)lh * ldc + c);
      const float e = __ldg(lse + lh);
      acc.x += __expf(v.x - e); acc.y += __expf(v.y - e); acc.z += __expf(v.z - e); acc.w += __expf(v.w - e);
    }
  }
  part[lg][cq] = acc;
  __syncthreads();
  if (threadIdx.x < 64) {
    const int cc = c0 + threadIdx.x;
    if (cc < nc) {
      const float* pf = reinterpret_cast<const float*>(&part[0][0]);
      float rsum = 0.f;
#pragma unroll
      for (int g = 0; g < 16; ++g) rsum += pf[g * 64 + threadIdx.x];
      rule_c[cc] = rsum;
      const int pos = cand_pos[cc];
      if (scatter_scores) scores[pos] = rsum;
      if (rule_out) rule_out[pos] = rsum;
    }
  }
}

}  // namespace ikv
