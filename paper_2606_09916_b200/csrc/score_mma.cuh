// score_mma.cuh -- the bf16 key pass of the rule scorer (Eq. 3) and the mean key of Eq. 5
// as ONE persistent streaming kernel for sm_100a (one CTA per SM, three warp roles).
//
//   producer warp  : per (32-token tile, layer) one 1-D bulk copy (TMA unit, UBLKCP) per token row
//                    [H_kv][D] bf16 (2 KB at Qwen3-8B shape) through the slot map into a ring of shared-memory
//                    stages, completion on an mbarrier (full[stage]); waits on empty[stage] before reuse.
//   logit warps    : warp w owns KV head(s) w, w+8, ...; the two 16 x D key tiles of the stage are the A operands of
//                    mma.sync.m16n8k16 (bf16 in, fp32 accumulate); the B operand holds the G memory rows of the
//                    group, each split into a bf16 hi and a bf16 lo part (two columns), so that hi + lo carries
//                    ~16 mantissa bits of M / sqrt(D) and keys are exact => fp32-grade logits.  The B fragments are
//                    prefetched one whole stage ahead.  The contraction has only G (<= 8) useful columns: it is
//                    not a tcgen05 tile (R1); the tensor pipe keeps the FMA pipe free, the kernel is
//                    HBM-bound.  Logits -> scratch [L*Hq][ldc] (fp32); running (max, sum exp) per (l,h) per CTA.
//   mean-key warps : warp dq owns one quarter of D; every lane sums its 16-byte chunks over all KV heads and layers
//                    in fp32 registers (Eq. 5) and writes k_bar once per tile -- no cross-warp reduction.
//   Tiles [0, ceil(n_cand/32)) are the candidates; the tiles after them are the live cross-attention positions
//   (K^q of Eq. 6, R7/R8) for which only the mean key is produced.
#pragma once
#include "common.cuh"
#include "pipe.cuh"

namespace ikv {

constexpr int KP_TOK = 32;       // tokens per stage = two m16 tiles of the mma
constexpr int KP_LWARPS = 8;     // logit warps
constexpr int KP_KWARPS = 4;     // mean-key warps
// G <= 4: a producer warp of its own (13 warps, 128 registers per thread).  G > 4 with mean keys: the two-tile B
// fragments need ~170 registers in the logit warps, more than a 13-warp CTA leaves.  Round 1 let the first mean-key
// warp also produce (12 warps; -DIKV_KP_MERGED=1 still builds it); now the CTA has four whole warpgroups and the logit
// warps take registers from the others with setmaxnreg (configs[2]: 2.00 -> 1.96 ms).
#ifndef IKV_KP_MERGED
#define IKV_KP_MERGED 0
#endif
__host__ __device__ constexpr bool kp_merged(int G, bool kbar) { return IKV_KP_MERGED && kbar && G > 4; }
// G > 4 with mean keys, not merged: four whole warpgroups (logit | logit | mean-key | producer + three idle warps), so
// that setmaxnreg can move registers from the last two to the logit warps (KP_REG_*)
__host__ __device__ constexpr bool kp_regsplit(int G, bool kbar) { return !IKV_KP_MERGED && kbar && G > 4; }
__host__ __device__ constexpr int kp_threads(int G, bool kbar) {
  return kp_regsplit(G, kbar) ? 512 : (KP_LWARPS + KP_KWARPS + (kp_merged(G, kbar) ? 0 : 1)) * 32;
}
constexpr int KP_REG_LOGIT = 184, KP_REG_OTHER = 72;   // 256 x 184 + 256 x 72 = 65,536 registers
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
__device__ __forceinline__ void memory_frags_item(int idx, const float* __restrict__ M, int L, int Hkv, float inv_sqrt_d,
                                                  uint4* __restrict__ frag) {
  constexpr int KS = D / 16, NT = (G <= 4) ? 1 : 2;
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
  int l2_hints;            // bit 0: keys evict_first, bit 1: logits evict_last
};

// Warp roles of k_key_pass: warps [0, KP_LWARPS) logit warps, [KP_LWARPS, KP_LWARPS + KP_KWARPS) mean-key warps
// (KBAR only; warp (dq, th) owns the d-quarter dq of the token part th).  Producer: a warp of its own, or the first
// mean-key warp (kp_merged).
template <int D, int G, bool KBAR>
__global__ __launch_bounds__(kp_threads(G, KBAR), 1) void k_key_pass(const KeyPassParams p) {
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  constexpr int KS = D / 16, NI = D / 32, NT = (G <= 4) ? 1 : 2;
  constexpr bool MERGED = kp_merged(G, KBAR);
  constexpr int KP_THREADS = kp_threads(G, KBAR);
  const int L = p.L, Hkv = p.Hkv, Hq = Hkv * G;
  const int row_bytes = Hkv * D * 2;
  const int row_stride = row_bytes + KP_ROWPAD;
  const int stage_bytes = KP_TOK * row_stride;
  const int NS = p.n_stage;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* stage_base = smem_raw;                                     // [NS][KP_TOK][row_stride]
  float2* stats = (float2*)(stage_base + (size_t)NS * stage_bytes);          // [L*Hq]
  uint64_t* full = (uint64_t*)(stats + (size_t)L * Hq);                      // [NS]
  uint64_t* empty = full + NS;                                               // [NS]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nc = *p.n_cand;
  const int nx = (KBAR && p.n_xq) ? *p.n_xq : 0;
  const int tiles_c = (nc + KP_TOK - 1) / KP_TOK;
  const int tiles = tiles_c + (nx + KP_TOK - 1) / KP_TOK;

  for (int i = threadIdx.x; i < L * Hq; i += KP_THREADS) stats[i] = make_float2(-CUDART_INF_F, 0.f);
  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], KP_LWARPS + (KBAR ? KP_KWARPS : 0)); }
    mbar_fence_init();
  }
  __syncthreads();

  const uint64_t pol_keys = l2_policy_evict_first();  // keys are read exactly once per pass
  const uint64_t pol_logits = l2_policy_evict_last();  // the rule kernel re-reads the logits scratch
  if constexpr (kp_regsplit(G, KBAR)) {
    if (warp < KP_LWARPS) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(KP_REG_LOGIT));
    else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(KP_REG_OTHER));
  }
  if (!MERGED && warp == KP_LWARPS + KP_KWARPS) {
    // ------------------------------------------------------------------ producer (a warp of its own)
    int s = 0;
    uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
      const bool is_x = tile >= tiles_c;
      const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
      const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
      int64_t slot = 0;
      if (lane < nvalid) slot = is_x ? p.xq_slot[t0 + lane] : p.cand_slot[t0 + lane];
      const bf16* src = p.k_pool + slot * (int64_t)(Hkv * D);
      for (int l = 0; l < L; ++l) {
        if (lane == 0) {
          mbar_wait(&empty[s], ph ^ 1u);
          mbar_arrive_expect_tx(&full[s], (uint32_t)(nvalid * row_bytes));
        }
        __syncwarp();
        if (lane < nvalid) {
          if (p.l2_hints & 1)
            bulk_g2s_hint(stage_base + (size_t)s * stage_bytes + lane * row_stride, src + (int64_t)l * p.layer_stride,
                          (uint32_t)row_bytes, &full[s], pol_keys);
          else
            bulk_g2s(stage_base + (size_t)s * stage_bytes + lane * row_stride, src + (int64_t)l * p.layer_stride,
                     (uint32_t)row_bytes, &full[s]);
        }
        if (++s == NS) { s = 0; ph ^= 1u; }
      }
    }
  } else if (warp < KP_LWARPS) {
    // ------------------------------------------------------------------ logit warps
    const int r = lane >> 2, q = lane & 3;
    const uint32_t stage_u32 = smem_u32(stage_base);
    const int nhw = (Hkv - warp + KP_LWARPS - 1) / KP_LWARPS;  // heads of this warp (may be 0)
    constexpr int HP = (NT == 1) ? 2 : 1;                      // heads per prefetch chunk
    const int nchunk = (nhw + HP - 1) / HP;
    uint4 bf[HP][NT][KS / 2], bn[HP][NT][KS / 2];
    auto load_chunk = [&](uint4 (&dst)[HP][NT][KS / 2], int l, int ck) {
#pragma unroll
      for (int h = 0; h < HP; ++h) {
        const int hi = ck * HP + h;
        if (hi < nhw) {
          const uint4* fp = p.frag + ((int64_t)(l * Hkv + warp + hi * KP_LWARPS) * NT) * (KS / 2) * 32 + lane;
#pragma unroll
          for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int v = 0; v < KS / 2; ++v) dst[h][nt][v] = __ldg(fp + (nt * (KS / 2) + v) * 32);
        }
      }
    };
    if (nhw > 0) load_chunk(bn, 0, 0);
    int s = 0;
    uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
      const bool is_x = tile >= tiles_c;
      const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
      const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
      for (int l = 0; l < L; ++l) {
        mbar_wait(&full[s], ph);
        if (!is_x) {
          const uint32_t sb = stage_u32 + (uint32_t)(s * stage_bytes);
          for (int ck = 0; ck < nchunk; ++ck) {
#pragma unroll
            for (int h = 0; h < HP; ++h)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int v = 0; v < KS / 2; ++v) bf[h][nt][v] = bn[h][nt][v];
            {  // prefetch the fragments of this warp's next chunk: one whole stage ahead when Hkv <= 8
              int nk = ck + 1, nl = l;
              if (nk == nchunk) { nk = 0; nl = (l + 1 == L) ? 0 : l + 1; }
              load_chunk(bn, nl, nk);
            }
#pragma unroll
            for (int h = 0; h < HP; ++h) {
            const int hi = ck * HP + h;
            if (hi >= nhw) break;
            const int kvh = warp + hi * KP_LWARPS;
            float c[2][NT][4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
              uint4 ka[NI], kc[NI];
              const uint32_t a_lo = sb + (uint32_t)((mt * 16 + r) * row_stride + kvh * D * 2 + q * 16);
              const uint32_t a_hi = a_lo + (uint32_t)(8 * row_stride);
#pragma unroll
              for (int i = 0; i < NI; ++i) {
                ka[i] = lds128(a_lo + i * 64);
                kc[i] = lds128(a_hi + i * 64);
              }
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) { c[mt][nt][0] = c[mt][nt][1] = c[mt][nt][2] = c[mt][nt][3] = 0.f; }
#pragma unroll
              for (int i = 0; i < NI; ++i)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                  mma_bf16_16816(c[mt][nt], ka[i].x, kc[i].x, ka[i].y, kc[i].y, bf[h][nt][i].x, bf[h][nt][i].y);
                  mma_bf16_16816(c[mt][nt], ka[i].z, kc[i].z, ka[i].w, kc[i].w, bf[h][nt][i].z, bf[h][nt][i].w);
                }
            }
            // logits of this thread: NH heads x 4 tokens (r, r+8, r+16, r+24)
            constexpr int NH = (NT == 1) ? 1 : 2;
            float x[NH][4];
            int g0;
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
              if (NT == 1) {
                x[0][2 * mt] = c[mt][0][0] + c[mt][0][1];
                x[0][2 * mt + 1] = c[mt][0][2] + c[mt][0][3];
              } else {
                x[0][2 * mt] = c[mt][0][0] + c[mt][NT - 1][0];
                x[NH - 1][2 * mt] = c[mt][0][1] + c[mt][NT - 1][1];
                x[0][2 * mt + 1] = c[mt][0][2] + c[mt][NT - 1][2];
                x[NH - 1][2 * mt + 1] = c[mt][0][3] + c[mt][NT - 1][3];
              }
            }
            g0 = (NT == 1) ? q : 2 * q;
            bool tv[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) tv[e] = (r + 8 * e) < nvalid;
#pragma unroll
            for (int hh = 0; hh < NH; ++hh) {
              const int g = g0 + hh;
              const bool gv = g < G;
              const int lh = l * Hq + kvh * G + (gv ? g : 0);
              float* lrow = p.logits + (int64_t)lh * p.ldc + t0 + r;
              float mx = -CUDART_INF_F;
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                if (gv && tv[e]) {
                  if (p.l2_hints & 2) st_f32_hint(lrow + 8 * e, x[hh][e], pol_logits);
                  else lrow[8 * e] = x[hh][e];
                }
                mx = fmaxf(mx, tv[e] ? x[hh][e] : -CUDART_INF_F);
              }
              mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
              mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
              mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
              float se = 0.f;
#pragma unroll
              for (int e = 0; e < 4; ++e) se += tv[e] ? __expf(x[hh][e] - mx) : 0.f;
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
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
        if (++s == NS) { s = 0; ph ^= 1u; }
      }
    }
  } else if (KBAR && warp < KP_LWARPS + KP_KWARPS) {
    // ------------------------------------------------------------------ mean-key warps (Eq. 5).  MERGED: the first one
    // also produces: it tops the ring up (non-blocking test of the slot's empty barrier) before every stage it consumes,
    // and blocks on a slot only when nothing it issued is left for it to consume.
    constexpr int CH = D / 32;                 // 16-byte chunks per token in a d-quarter
    constexpr int TPL = 32 / CH;               // tokens per warp load
    constexpr int ROWS = KP_TOK / (KP_KWARPS / 4);
    constexpr int NG = ROWS / TPL;             // token groups per warp
    const int kw = warp - KP_LWARPS, dq = kw & 3, th = kw >> 2;
    const bool prod = MERGED && (kw == 0);
    const int tl = lane / CH, ch = lane % CH;
    const uint32_t stage_u32 = smem_u32(stage_base);
    const uint32_t lane_off = (uint32_t)((th * ROWS + tl) * row_stride + dq * (D / 4) * 2 + ch * 16);
    const float inv = 1.f / (float)(L * Hkv);
    // producer state
    const int my_tiles = (tiles > (int)blockIdx.x) ? (tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int total_stages = my_tiles * L;
    int issued = 0, consumed = 0, p_tile = blockIdx.x, p_l = 0, p_s = 0;
    uint32_t p_ph = 0;
    auto slot_of_tile = [&](int tile) -> int64_t {
      if (tile >= tiles) return 0;
      const bool tx = tile >= tiles_c;
      const int t0 = (tx ? tile - tiles_c : tile) * KP_TOK;
      const int nv = min(KP_TOK, (tx ? nx : nc) - t0);
      return (lane < nv) ? (int64_t)(tx ? p.xq_slot[t0 + lane] : p.cand_slot[t0 + lane]) : 0;
    };
    int64_t p_slot = 0, p_slot_next = 0;
    if (prod) { p_slot = slot_of_tile(p_tile); p_slot_next = slot_of_tile(p_tile + gridDim.x); }
    auto try_issue = [&](bool block) -> bool {
      if (issued >= total_stages || issued - consumed >= NS) return false;
      uint32_t ok = 1u;
      if (lane == 0) {
        if (block) mbar_wait(&empty[p_s], p_ph ^ 1u);
        else ok = mbar_test_wait(&empty[p_s], p_ph ^ 1u) ? 1u : 0u;
      }
      ok = __shfl_sync(0xffffffffu, ok, 0);
      if (!ok) return false;
      const bool tx = p_tile >= tiles_c;
      const int t0 = (tx ? p_tile - tiles_c : p_tile) * KP_TOK;
      const int nv = min(KP_TOK, (tx ? nx : nc) - t0);
      if (lane == 0) mbar_arrive_expect_tx(&full[p_s], (uint32_t)(nv * row_bytes));
      __syncwarp();
      if (lane < nv) {
        if (p.l2_hints & 1)
          bulk_g2s_hint(stage_base + (size_t)p_s * stage_bytes + lane * row_stride,
                        p.k_pool + p_slot * (int64_t)(Hkv * D) + (int64_t)p_l * p.layer_stride, (uint32_t)row_bytes,
                        &full[p_s], pol_keys);
        else
          bulk_g2s(stage_base + (size_t)p_s * stage_bytes + lane * row_stride,
                   p.k_pool + p_slot * (int64_t)(Hkv * D) + (int64_t)p_l * p.layer_stride, (uint32_t)row_bytes,
                   &full[p_s]);
      }
      if (++p_l == L) {
        p_l = 0;
        p_tile += gridDim.x;
        p_slot = p_slot_next;
        p_slot_next = slot_of_tile(p_tile + gridDim.x);
      }
      if (++p_s == NS) { p_s = 0; p_ph ^= 1u; }
      ++issued;
      return true;
    };
    int s = 0;
    uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
      const bool is_x = tile >= tiles_c;
      const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
      const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
      float kb[NG][8];
#pragma unroll
      for (int gI = 0; gI < NG; ++gI)
#pragma unroll
        for (int e = 0; e < 8; ++e) kb[gI][e] = 0.f;
      for (int l = 0; l < L; ++l) {
        if (prod) {
          while (try_issue(false)) {
          }
          if (issued == consumed) try_issue(true);
        }
        mbar_wait(&full[s], ph);
        const uint32_t sb = stage_u32 + (uint32_t)(s * stage_bytes) + lane_off;
#pragma unroll 4
        for (int kvh = 0; kvh < Hkv; ++kvh) {
#pragma unroll
          for (int gI = 0; gI < NG; ++gI) {
            const uint4 u = lds128(sb + (uint32_t)(gI * TPL * row_stride + kvh * D * 2));
            kb[gI][0] += bf16lo(u.x); kb[gI][1] += bf16hi(u.x);
            kb[gI][2] += bf16lo(u.y); kb[gI][3] += bf16hi(u.y);
            kb[gI][4] += bf16lo(u.z); kb[gI][5] += bf16hi(u.z);
            kb[gI][6] += bf16lo(u.w); kb[gI][7] += bf16hi(u.w);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
        if (++s == NS) { s = 0; ph ^= 1u; }
        ++consumed;
      }
      float* outp = is_x ? p.kq : p.kbar;
#pragma unroll
      for (int gI = 0; gI < NG; ++gI) {
        const int tok = th * ROWS + gI * TPL + tl;
        if (tok < nvalid) {
          float4* d4 = reinterpret_cast<float4*>(outp + (int64_t)(t0 + tok) * D + dq * (D / 4) + ch * 8);
          d4[0] = make_float4(kb[gI][0] * inv, kb[gI][1] * inv, kb[gI][2] * inv, kb[gI][3] * inv);
          d4[1] = make_float4(kb[gI][4] * inv, kb[gI][5] * inv, kb[gI][6] * inv, kb[gI][7] * inv);
        }
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < L * Hq; i += KP_THREADS) p.partials[(int64_t)i * gridDim.x + blockIdx.x] = stats[i];
}

// shared memory of k_key_pass; returns 0 if not even two stages fit
inline size_t key_pass_smem(int L, int Hq, int Hkv, int D, bool kbar, int max_smem, int* n_stage) {
  (void)kbar;
  const size_t stage = (size_t)KP_TOK * (Hkv * D * 2 + KP_ROWPAD);
  const size_t fixed = (size_t)L * Hq * 8 + 2 * 8 * 8 + 128;
  if (fixed + 2 * stage > (size_t)max_smem) { *n_stage = 0; return 0; }
  int ns = (int)(((size_t)max_smem - fixed) / stage);
  if (ns > 8) ns = 8;
  *n_stage = ns;
  return fixed + (size_t)ns * stage;
}

// ---------------------------------------------------------------------------------------------
// a3  rule_c = sum_{l,h} exp(x[l,h,c] - lse[l,h])   (Eq. 3).  One block of 256 threads per 64 candidates (launched
// from k_rule_fused, fused_small.cuh):
// thread (cq = tid % 16 -> 4 candidates, lg = tid / 16 -> rows lg, lg+16, ...), 16-byte loads.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void score_rule4_block(int bid, int n_blocks, const float* __restrict__ logits, int64_t ldc,
                                                  int LH, const float* __restrict__ lse,
                                                  const int32_t* __restrict__ n_cand_p,
                                                  const int32_t* __restrict__ cand_pos, float* __restrict__ rule_c,
                                                  float* __restrict__ scores, int scatter_scores,
                                                  float* __restrict__ rule_out, int l2_hints) {
  __shared__ float4 part[16][16];
  const uint64_t pol = l2_policy_evict_first();  // the logits are dead once read
  const int nc = *n_cand_p;
  // newest tiles first: the key pass wrote the logits in tile order, so the tail of the scratch is still in L2
  const int c0 = (n_blocks - 1 - bid) * 64;
  if (c0 >= nc) return;
  const int cq = threadIdx.x & 15, lg = threadIdx.x >> 4;
  const int c = c0 + cq * 4;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  if (c < nc) {  // rows are padded to a multiple of 4 (ldc % 4 == 0); lanes past n_cand read scratch, never stored
#pragma unroll 12
    for (int lh = lg; lh < LH; lh += 16) {
      const float* lp = logits + (int64_t)lh * ldc + c;
      const float4 v = (l2_hints & 4) ? ld_f32x4_hint(lp, pol) : *reinterpret_cast<const float4*>(lp);
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
