// score_lm.cuh -- the bf16 key pass of the rule scorer (Eq. 3) and the mean key of Eq. 5
// in LAYER-MAJOR order with deferred normalisation: no logits scratch, no separate lse / rule launches.
//
// Eq. 3 normalises every (layer, head) row over ALL candidates, so a token's contribution exp(x - lse[l,h]) cannot be
// summed over (l,h) before the whole row has been seen.  k_key_pass (score_mma.cuh) therefore writes the fp32 logits
// (L*H_q*4 B per token, 6 % of the key bytes) and two more launches read them back.  Here every persistent CTA (one per
// SM) owns a fixed set of 32-token tiles and walks layer by layer over them; the logits of the last two layers and the
// running rule sum of every (token, head) it owns stay ON CHIP, in tensor memory used as a per-thread scratchpad
// (tcgen05.ld / tcgen05.st, 512 columns x 128 lanes per SM), and so do the mean-key accumulators:
//   per layer l, per CTA : (max, sum exp) of its tokens per head -> global partials[l*Hq+h][cta]; counter[l] += 1
//   stats warp           : waits for counter[l] = all CTAs, reduces the partials -> lse[l, :] in shared memory
//   logit warps, layer l : rule_acc += exp(x_{l-2} - lse[l-2]) for the tile in flight, then shift x_{l-1}, x_l
// The two-layer deferral gives the grid a whole layer (~11 us at Qwen3-8B shape) of slack, so no CTA ever waits for the
// slowest one on the critical path; only the last two layers are finished after the stream has ended.  All sums are taken
// in a fixed order: scores are bit-identical from run to run.
//
// Capacity: 12 columns per tile and logit warp, 32 per tile for the mean key -> at most LM_MT_KBAR = 9 tiles (288 tokens)
// per CTA with mean keys, LM_MT = 21 without; G <= 4 and H_kv <= 8.  Other calls take k_key_pass.
#pragma once
#include "common.cuh"
#include "pipe.cuh"
#include "score_mma.cuh"

namespace ikv {

constexpr int LM_MT_KBAR = 9;   // tiles per CTA, learnable calls (56 TMEM columns per tile)
constexpr int LM_MT = 21;       // tiles per CTA, rule-only calls (24 TMEM columns per tile)
constexpr int LM_SWARPS = 3;    // stats warps: each reduces a third of the CTAs' partials of every layer
__host__ __device__ constexpr int lm_threads(bool kbar) { return (KP_LWARPS + (kbar ? KP_KWARPS : 0) + 1 + LM_SWARPS) * 32; }

struct KeyPassLmParams {
  const bf16* k_pool;
  int64_t layer_stride;  // elements
  int L, Hkv;
  const uint4* frag;
  const int32_t* cand_slot;
  const int32_t* cand_pos;
  const int32_t* n_cand;
  const int32_t* xq_slot;  // may be NULL
  const int32_t* n_xq;     // may be NULL
  float2* partials;        // [L][gridDim.x][Hq]
  int32_t* layer_cnt;      // [L], zero at launch
  float* rule_c;           // [n_cand]
  float* scores;           // by position, written when scatter_scores
  float* rule_out;         // optional, by position
  int scatter_scores;
  float* kbar;             // [n_cand][D]   (KBAR)
  float* kq;               // [n_xq][D]     (KBAR)
  int n_stage;
  int l2_hints;
  unsigned long long* tstamp;  // profiling: {min start, max end} of the launch in %globaltimer ns, or NULL
  const float* mpart;      // partial sums of the memory rows (k_mem_prep), [n_mpart][D]; with mbar_out != NULL one
  int n_mpart, LH;         // statistics warp of CTA 0 reduces them to mbar (Eq. 5) while the keys stream, in the order
  float* mbar_out;         // the fold blocks would use (b ascending): they then start with one load instead of a chain
};

__device__ __forceinline__ void tmem_ld4(uint32_t taddr, float (&v)[4]) {
  uint32_t r[4];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 4; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const float (&v)[4]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(__float_as_uint(v[0])),
               "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,"
      "%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]),
        "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]),
        "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,"
      "%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
      "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
      "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
      "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
      "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15])),
      "r"(__float_as_uint(v[16])), "r"(__float_as_uint(v[17])), "r"(__float_as_uint(v[18])), "r"(__float_as_uint(v[19])),
      "r"(__float_as_uint(v[20])), "r"(__float_as_uint(v[21])), "r"(__float_as_uint(v[22])), "r"(__float_as_uint(v[23])),
      "r"(__float_as_uint(v[24])), "r"(__float_as_uint(v[25])), "r"(__float_as_uint(v[26])), "r"(__float_as_uint(v[27])),
      "r"(__float_as_uint(v[28])), "r"(__float_as_uint(v[29])), "r"(__float_as_uint(v[30])), "r"(__float_as_uint(v[31]))
      : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

#ifdef IKV_TRACE
#define LM_GUARD(tag, cond)                                                                                   \
  do {                                                                                                        \
    long long _n = 0;                                                                                         \
    while (!(cond)) {                                                                                         \
      __nanosleep(64);                                                                                        \
      if (++_n > 4000000LL) {                                                                                 \
        printf("LM hang: %s cta %d warp %d lane %d\n", tag, (int)blockIdx.x, (int)(threadIdx.x >> 5), (int)(threadIdx.x & 31)); \
        __trap();                                                                                             \
      }                                                                                                       \
    }                                                                                                         \
  } while (0)
#else
#define LM_GUARD(tag, cond) do { while (!(cond)) __nanosleep(64); } while (0)
#endif

#ifdef IKV_TRACE
__device__ long long g_lm_wait[160][4];
#endif
__device__ __forceinline__ int ld_acquire_i32(const int32_t* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// Warp roles: warps [0, 8) logit warps (warp = KV head), [8, 12) mean-key warps (KBAR), then producer, then stats warp.
template <int D, int G, bool KBAR>
__global__ __launch_bounds__(lm_threads(KBAR), 1) void k_key_pass_lm(const KeyPassLmParams p) {
  static_assert(G <= 4, "layer-major key pass: G <= 4");
  pdl_wait();  // launched with programmatic stream serialization: nothing is read before the predecessor is complete
  pdl_launch_dependents();
  if (p.tstamp && threadIdx.x == 0) {  // kernel time without host events between the launches (they cost the overlap)
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    atomicMin(p.tstamp, t);
  }
  constexpr int KS = D / 16, NI = D / 32;
  constexpr int THREADS = lm_threads(KBAR);
  constexpr int MT = KBAR ? LM_MT_KBAR : LM_MT;
  constexpr int W_PROD = KP_LWARPS + (KBAR ? KP_KWARPS : 0), W_STATS = W_PROD + 1;
  constexpr int KB_COL0 = 2 * 12 * MT;  // first TMEM column of the mean-key accumulators
  const int L = p.L, Hkv = p.Hkv, Hq = Hkv * G;
  const int row_bytes = Hkv * D * 2;
  const int row_stride = row_bytes + KP_ROWPAD;
  const int stage_bytes = KP_TOK * row_stride;
  const int NS = p.n_stage;

  extern __shared__ __align__(128) unsigned char lm_smem[];
  unsigned char* stage_base = lm_smem;                                       // [NS][KP_TOK][row_stride]
  int32_t* slot_s = (int32_t*)(stage_base + (size_t)NS * stage_bytes);       // [MT][32] slots of the CTA's tiles
  float* lse_s = (float*)(slot_s + MT * 32);                                 // [4][Hq] ring over layers
  float2* part_s = (float2*)(lse_s + 4 * ((Hq + 1) & ~1));                   // [4][Hq] this CTA's (max, sum exp), ring
  float2* stat_s = part_s + 4 * ((Hq + 1) & ~1);                             // [LM_SWARPS][Hq] merges of the stats warps
  uint64_t* full = (uint64_t*)(stat_s + LM_SWARPS * ((Hq + 1) & ~1));        // [NS]
  uint64_t* empty = full + NS;                                               // [NS]
  uint64_t* pub_bar = empty + NS;                                            // [4] the logit warps have written part_s[l & 3]
  volatile int* lse_flag = (volatile int*)(pub_bar + 4);                     // [4]: l + 1 once lse[l] is in slot l & 3
  uint32_t* tmem_base_p = (uint32_t*)(lse_flag + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nc = *p.n_cand;
  const int nx = (KBAR && p.n_xq) ? *p.n_xq : 0;
  const int tiles_c = (nc + KP_TOK - 1) / KP_TOK;
  const int tiles = tiles_c + (nx + KP_TOK - 1) / KP_TOK;
  const int my_tiles = (tiles > (int)blockIdx.x) ? (tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
  const int n_lwarps = Hkv < KP_LWARPS ? Hkv : KP_LWARPS;  // logit warps with a KV head

  for (int i = threadIdx.x; i < my_tiles * 32; i += THREADS) {
    const int tile = blockIdx.x + (i >> 5) * gridDim.x, k = i & 31;
    const bool tx = tile >= tiles_c;
    const int t = (tx ? tile - tiles_c : tile) * KP_TOK + k;
    slot_s[i] = (t < (tx ? nx : nc)) ? (tx ? p.xq_slot[t] : p.cand_slot[t]) : 0;
  }
  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], n_lwarps + (KBAR ? KP_KWARPS : 0)); }
    for (int i = 0; i < 4; ++i) { mbar_init(&pub_bar[i], n_lwarps); lse_flag[i] = 0; }
    mbar_fence_init();
  }
  if (warp == W_STATS) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_p)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_base_p;
  const uint64_t pol_keys = l2_policy_evict_first();  // keys are read exactly once per pass

  if (warp == W_PROD) {
    // ------------------------------------------------------------------ producer: layer by layer over the CTA's tiles
    int s = 0;
    uint32_t ph = 0;
    for (int l = 0; l < L; ++l) {
      const bf16* lay = p.k_pool + (int64_t)l * p.layer_stride;
      for (int i = 0; i < my_tiles; ++i) {
        const int tile = blockIdx.x + i * gridDim.x;
        const bool is_x = tile >= tiles_c;
        const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
        const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
        const int64_t slot = slot_s[i * 32 + lane];
        if (lane == 0) {
          mbar_wait(&empty[s], ph ^ 1u);
          mbar_arrive_expect_tx(&full[s], (uint32_t)(nvalid * row_bytes));
        }
        __syncwarp();
        if (lane < nvalid) {
          unsigned char* dst = stage_base + (size_t)s * stage_bytes + lane * row_stride;
          const bf16* src = lay + slot * (int64_t)(Hkv * D);
          if (p.l2_hints & 1) bulk_g2s_hint(dst, src, (uint32_t)row_bytes, &full[s], pol_keys);
          else bulk_g2s(dst, src, (uint32_t)row_bytes, &full[s]);
        }
        if (++s == NS) { s = 0; ph ^= 1u; }
      }
    }
  } else if (warp >= W_STATS) {
    // ------------------------------------------------------------------ stats warps: lse[l, :] once every CTA has
    // published its (max, sum exp) partials of layer l.  Lane = head: the partials of one CTA are contiguous, every lane
    // merges its head's partials in CTA order (fixed order: deterministic).
    const int target = (int)gridDim.x;
    const int n_cta = gridDim.x;
    const int hq2 = (Hq + 1) & ~1;
    const int sw = warp - W_STATS;
    const int per = (n_cta + LM_SWARPS - 1) / LM_SWARPS, j_lo = sw * per, j_hi = min(n_cta, j_lo + per);
    if (KBAR && blockIdx.x == 0 && sw == LM_SWARPS - 1 && p.mbar_out) {
      for (int d = lane; d < D; d += 32) {
        float acc = 0.f;
        int b = 0;
        for (; b + 8 <= p.n_mpart; b += 8) {
          float v[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) v[j] = p.mpart[(b + j) * D + d];
#pragma unroll
          for (int j = 0; j < 8; ++j) acc += v[j];
        }
        for (; b < p.n_mpart; ++b) acc += p.mpart[b * D + d];
        p.mbar_out[d] = acc / (float)p.LH;
      }
    }
    for (int l = 0; l < L; ++l) {
      if (sw == 0) {
        // publish this CTA's partials of layer l (the logit warps only write shared memory: the fence and the atomic
        // stay off their critical path)
        mbar_wait(&pub_bar[l & 3], (uint32_t)(l >> 2) & 1u);
        for (int h = lane; h < Hq; h += 32)
          p.partials[((int64_t)l * n_cta + blockIdx.x) * Hq + h] = part_s[(l & 3) * hq2 + h];
        __threadfence();
        __syncwarp();
        if (lane == 0) atomicAdd(p.layer_cnt + l, 1);
      }
      if (my_tiles == 0) continue;  // a CTA without tiles needs no lse
      if (lane == 0) {
        LM_GUARD("layer counter", ld_acquire_i32(p.layer_cnt + l) >= target);
      }
      __syncwarp();
      for (int h0 = 0; h0 < Hq; h0 += 32) {
        const int h = min(h0 + lane, Hq - 1);
        const float2* pp = p.partials + (int64_t)l * n_cta * Hq + h;
        float m = -CUDART_INF_F, s = 0.f;
        for (int j0 = j_lo; j0 < j_hi; j0 += 25) {
          float2 v[25];
#pragma unroll
          for (int j = 0; j < 25; ++j)
            v[j] = (j0 + j < j_hi) ? __ldcg(pp + (int64_t)(j0 + j) * Hq) : make_float2(-CUDART_INF_F, 0.f);
#pragma unroll
          for (int j = 0; j < 25; ++j)
            if (v[j].y > 0.f) {
              const float mn = fmaxf(m, v[j].x);
              s = s * __expf(m - mn) + v[j].y * __expf(v[j].x - mn);
              m = mn;
            }
        }
        if (h0 + lane < Hq) stat_s[sw * hq2 + h0 + lane] = make_float2(m, s);
      }
      bar_sync(3, LM_SWARPS * 32);  // the three partial merges are in shared memory
      if (sw == 0) {
        float* out = lse_s + (l & 3) * hq2;
        for (int h = lane; h < Hq; h += 32) {
          float m = -CUDART_INF_F, s = 0.f;
#pragma unroll
          for (int k = 0; k < LM_SWARPS; ++k) {
            const float2 v = stat_s[k * hq2 + h];
            if (v.y > 0.f) {
              const float mn = fmaxf(m, v.x);
              s = s * __expf(m - mn) + v.y * __expf(v.x - mn);
              m = mn;
            }
          }
          out[h] = m + logf(s);
        }
        __syncwarp();
        __threadfence_block();
        if (lane == 0) lse_flag[l & 3] = l + 1;
      }
      bar_sync(3, LM_SWARPS * 32);  // stat_s is rewritten for the next layer
    }
  } else if (warp < KP_LWARPS) {
    // ------------------------------------------------------------------ logit warps
    const int r = lane >> 2, q = lane & 3;
    const int kvh = warp;
    const bool active = warp < n_lwarps;
    const bool gv = q < G;
    const uint32_t stage_u32 = smem_u32(stage_base);
    const uint32_t tcol = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 12 * MT);
    const int lh_stride = (Hq + 1) & ~1;
    if (active) {
      uint4 bf[KS / 2], bn[KS / 2];
      auto load_frag = [&](uint4 (&dst)[KS / 2], int l) {
        const uint4* fp = p.frag + ((int64_t)(l * Hkv + kvh)) * (KS / 2) * 32 + lane;
#pragma unroll
        for (int v = 0; v < KS / 2; ++v) dst[v] = __ldg(fp + v * 32);
      };
      load_frag(bn, 0);
      int s = 0;
      uint32_t ph = 0;
#ifdef IKV_TRACE
      if (warp == 0 && lane == 0) { g_lm_wait[blockIdx.x][0] = 0; g_lm_wait[blockIdx.x][1] = 0; g_lm_wait[blockIdx.x][2] = clock64(); }
#endif
      for (int l = 0; l < L; ++l) {
#pragma unroll
        for (int v = 0; v < KS / 2; ++v) bf[v] = bn[v];
        if (l + 1 < L) load_frag(bn, l + 1);
        float m_run = -CUDART_INF_F, s_run = 0.f;  // (max, sum exp) of this thread's tokens of head q in layer l
        float lse2 = 0.f;
        if (l >= 2 && my_tiles > 0) {  // a CTA without tiles only publishes its (empty) partials
#ifdef IKV_TRACE
          const long long tw0 = clock64();
#endif
          LM_GUARD("lse of layer l-2", lse_flag[(l - 2) & 3] == l - 1);
#ifdef IKV_TRACE
          if (warp == 0 && lane == 0) { g_lm_wait[blockIdx.x][0] += clock64() - tw0; g_lm_wait[blockIdx.x][1] += 1; }
#endif
          lse2 = lse_s[((l - 2) & 3) * lh_stride + kvh * G + (gv ? q : 0)];
        }
        for (int i = 0; i < my_tiles; ++i) {
          const int tile = blockIdx.x + i * gridDim.x;
          const bool is_x = tile >= tiles_c;
          mbar_wait(&full[s], ph);
          if (!is_x) {
            const int t0 = tile * KP_TOK;
            const int nvalid = min(KP_TOK, nc - t0);
            const uint32_t sb = stage_u32 + (uint32_t)(s * stage_bytes);
            float c[2][4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
              uint4 ka[NI], kc[NI];
              const uint32_t a_lo = sb + (uint32_t)((mt * 16 + r) * row_stride + kvh * D * 2 + q * 16);
              const uint32_t a_hi = a_lo + (uint32_t)(8 * row_stride);
#pragma unroll
              for (int k = 0; k < NI; ++k) {
                ka[k] = lds128(a_lo + k * 64);
                kc[k] = lds128(a_hi + k * 64);
              }
              c[mt][0] = c[mt][1] = c[mt][2] = c[mt][3] = 0.f;
#pragma unroll
              for (int k = 0; k < NI; ++k) {
                mma_bf16_16816(c[mt], ka[k].x, kc[k].x, ka[k].y, kc[k].y, bf[k].x, bf[k].y);
                mma_bf16_16816(c[mt], ka[k].z, kc[k].z, ka[k].w, kc[k].w, bf[k].z, bf[k].w);
              }
            }
            // this thread: head q, tokens r, r+8, r+16, r+24 (hi and lo columns of the memory row summed)
            float x[4];
            x[0] = c[0][0] + c[0][1]; x[1] = c[0][2] + c[0][3];
            x[2] = c[1][0] + c[1][1]; x[3] = c[1][2] + c[1][3];
            float mx = m_run;
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (r + 8 * e < nvalid) mx = fmaxf(mx, x[e]);
            if (mx > m_run) { s_run *= __expf(m_run - mx); m_run = mx; }  // m_run = -inf: s_run is 0 and stays 0
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (r + 8 * e < nvalid) s_run += __expf(x[e] - m_run);
            // tensor-memory scratch of the tile: [rule_acc | x of layer l-1 | x of layer l-2], 4 tokens each
            const uint32_t ta = tcol + (uint32_t)(12 * i);
            float racc[4] = {0.f, 0.f, 0.f, 0.f}, xa[4] = {0.f, 0.f, 0.f, 0.f}, xb[4] = {0.f, 0.f, 0.f, 0.f};
            if (l >= 1) {
              tmem_ld4(ta, racc);
              tmem_ld4(ta + 4, xa);
              tmem_ld4(ta + 8, xb);
              tmem_wait_ld();
            }
            if (l >= 2) {
#pragma unroll
              for (int e = 0; e < 4; ++e) racc[e] += __expf(xb[e] - lse2);
            }
            tmem_st4(ta, racc);
            tmem_st4(ta + 4, x);
            tmem_st4(ta + 8, xa);
            tmem_wait_st();
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(&empty[s]);
          if (++s == NS) { s = 0; ph ^= 1u; }
        }
        // publish (max, sum exp) of head q over this CTA's tokens: merge the 8 lanes (r = 0..7) that share the head
#pragma unroll
        for (int ofs = 4; ofs < 32; ofs <<= 1) {
          const float mo = __shfl_xor_sync(0xffffffffu, m_run, ofs), so = __shfl_xor_sync(0xffffffffu, s_run, ofs);
          const float mn = fmaxf(m_run, mo);
          const float a = (m_run == -CUDART_INF_F) ? 0.f : s_run * __expf(m_run - mn);
          const float b = (mo == -CUDART_INF_F) ? 0.f : so * __expf(mo - mn);
          m_run = mn; s_run = a + b;
        }
        if (r == 0 && gv) part_s[(l & 3) * lh_stride + kvh * G + q] = make_float2(m_run, s_run);
        __syncwarp();
        if (lane == 0) mbar_arrive(&pub_bar[l & 3]);  // a stats warp publishes the row (fence + atomic off this path)
      }
#ifdef IKV_TRACE
      if (warp == 0 && lane == 0) g_lm_wait[blockIdx.x][3] = clock64() - g_lm_wait[blockIdx.x][2];
#endif
      // ---- the last two layers, once every CTA has finished: then the per-token sum over heads and KV heads
      if (my_tiles > 0) {
        LM_GUARD("lse of the last layer", lse_flag[(L - 1) & 3] == L);
        if (L >= 2) LM_GUARD("lse of layer L-2", lse_flag[(L - 2) & 3] == L - 1);
        const float lse_a = lse_s[((L - 1) & 3) * lh_stride + kvh * G + (gv ? q : 0)];
        const float lse_b = (L >= 2) ? lse_s[((L - 2) & 3) * lh_stride + kvh * G + (gv ? q : 0)] : 0.f;
        float* red = reinterpret_cast<float*>(stage_base);  // [MT][8 warps][32 tokens]: the ring is drained
        // every consumer warp is past its last stage before the ring is reused: named barrier over logit + mean-key warps
        bar_sync(1, (KP_LWARPS + (KBAR ? KP_KWARPS : 0)) * 32);
        for (int i = 0; i < my_tiles; ++i) {
          const int tile = blockIdx.x + i * gridDim.x;
          if (tile >= tiles_c) break;
          const uint32_t ta = tcol + (uint32_t)(12 * i);
          float racc[4], xa[4], xb[4];
          tmem_ld4(ta, racc);
          tmem_ld4(ta + 4, xa);
          tmem_ld4(ta + 8, xb);
          tmem_wait_ld();
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            float v = racc[e] + __expf(xa[e] - lse_a);
            if (L >= 2) v += __expf(xb[e] - lse_b);
            v = gv ? v : 0.f;
            v += __shfl_xor_sync(0xffffffffu, v, 1);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            if (q == 0) red[(i * KP_LWARPS + warp) * 32 + r + 8 * e] = v;
          }
        }
      } else {
        bar_sync(1, (KP_LWARPS + (KBAR ? KP_KWARPS : 0)) * 32);
      }
    } else {
      // a logit warp without a KV head (H_kv < 8) only takes part in the barriers
      bar_sync(1, (KP_LWARPS + (KBAR ? KP_KWARPS : 0)) * 32);
    }
    bar_sync(2, KP_LWARPS * 32);  // red[] is complete
    if (my_tiles > 0) {
      const float* red = reinterpret_cast<const float*>(stage_base);
      for (int i = warp; i < my_tiles; i += KP_LWARPS) {  // warp w sums tile w, w+8, ...: lane = token
        const int tile = blockIdx.x + i * gridDim.x;
        if (tile >= tiles_c) break;
        const int tok = tile * KP_TOK + lane;
        float v = 0.f;
        for (int w = 0; w < n_lwarps; ++w) v += red[(i * KP_LWARPS + w) * 32 + lane];
        if (tok < nc) {
          p.rule_c[tok] = v;
          const int pos = p.cand_pos[tok];
          if (p.scatter_scores) p.scores[pos] = v;
          if (p.rule_out) p.rule_out[pos] = v;
        }
      }
    }
  } else if (KBAR && warp < KP_LWARPS + KP_KWARPS) {
    // ------------------------------------------------------------------ mean-key warps (Eq. 5): warp dq owns one quarter
    // of D.  The sum over the KV heads is a contraction with a stacked identity matrix: for every pair of KV heads the
    // 4-byte piece j of the lane's 16-byte chunk (rows r, r+8) of head kvh is the k < 8 half of an mma.sync.m16n8k16
    // A tile and the same piece of head kvh + 1 the k >= 8 half; B = [I8; I8] adds the two heads into the fp32
    // accumulators -- products with 1.0 are exact, and one HMMA replaces 32 unpack + 32 add instructions.  The tile's
    // accumulators live in tensor memory between the layers.
    // Thread (r, q) ends up with d = 8 q .. 8 q + 7 of the quarter for the tokens 16 mt + r and 16 mt + r + 8.
    constexpr int CW = D / 32;                 // 16-byte chunks of a d-quarter (lanes q < CW hold data)
    const int dq = warp - KP_LWARPS;
    const int r = lane >> 2, q = lane & 3;
    const uint32_t stage_u32 = smem_u32(stage_base);
    const uint32_t lane_off = (uint32_t)(r * row_stride + dq * (D / 4) * 2 + (q % CW) * 16);
    const uint32_t tcol = tmem + ((uint32_t)(dq * 32) << 16) + (uint32_t)KB_COL0;
    const float inv = 1.f / (float)(L * Hkv);
    // B = [I8; I8]: b0 holds rows k = 2q, 2q+1 and b1 rows k = 2q+8, 2q+9 of column n = r -- the same pattern
    const uint32_t one_sel = (r == 2 * q) ? 0x00003f80u : ((r == 2 * q + 1) ? 0x3f800000u : 0u);
    int s = 0;
    uint32_t ph = 0;
    for (int l = 0; l < L; ++l) {
      for (int i = 0; i < my_tiles; ++i) {
        float c[2][2][2][4];  // [m-tile][piece j = 2 ks + t of the chunk][row r: d 2j, 2j+1 | row r+8: d 2j, 2j+1]
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
          for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int t = 0; t < 2; ++t) c[a][b][t][0] = c[a][b][t][1] = c[a][b][t][2] = c[a][b][t][3] = 0.f;
        mbar_wait(&full[s], ph);
        const uint32_t sb = stage_u32 + (uint32_t)(s * stage_bytes) + lane_off;
        // two KV heads per HMMA: k = 0..7 of the A tile come from head kvh, k = 8..15 from head kvh + 1, B = [I8; I8]
#pragma unroll 2
        for (int kvh = 0; kvh + 1 < Hkv; kvh += 2) {
#pragma unroll
          for (int mt = 0; mt < 2; ++mt) {
            const uint4 ka = lds128(sb + (uint32_t)(mt * 16 * row_stride + kvh * D * 2));
            const uint4 kc = lds128(sb + (uint32_t)((mt * 16 + 8) * row_stride + kvh * D * 2));
            const uint4 kd = lds128(sb + (uint32_t)(mt * 16 * row_stride + (kvh + 1) * D * 2));
            const uint4 ke = lds128(sb + (uint32_t)((mt * 16 + 8) * row_stride + (kvh + 1) * D * 2));
            mma_bf16_16816(c[mt][0][0], ka.x, kc.x, kd.x, ke.x, one_sel, one_sel);
            mma_bf16_16816(c[mt][0][1], ka.y, kc.y, kd.y, ke.y, one_sel, one_sel);
            mma_bf16_16816(c[mt][1][0], ka.z, kc.z, kd.z, ke.z, one_sel, one_sel);
            mma_bf16_16816(c[mt][1][1], ka.w, kc.w, kd.w, ke.w, one_sel, one_sel);
          }
        }
        if (Hkv & 1) {
          const int kvh = Hkv - 1;
#pragma unroll
          for (int mt = 0; mt < 2; ++mt) {
            const uint4 ka = lds128(sb + (uint32_t)(mt * 16 * row_stride + kvh * D * 2));
            const uint4 kc = lds128(sb + (uint32_t)((mt * 16 + 8) * row_stride + kvh * D * 2));
            mma_bf16_16816(c[mt][0][0], ka.x, kc.x, 0u, 0u, one_sel, 0u);
            mma_bf16_16816(c[mt][0][1], ka.y, kc.y, 0u, 0u, one_sel, 0u);
            mma_bf16_16816(c[mt][1][0], ka.z, kc.z, 0u, 0u, one_sel, 0u);
            mma_bf16_16816(c[mt][1][1], ka.w, kc.w, 0u, 0u, one_sel, 0u);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
        if (++s == NS) { s = 0; ph ^= 1u; }
        // kb[(mt * 2 + row) * 8 + e]: token 16 mt + r + 8 row, d = 8 q + e;  e = 4 ks + 2 t + {0, 1}
        float kb[32];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
          for (int ks = 0; ks < 2; ++ks)
#pragma unroll
            for (int t = 0; t < 2; ++t) {
              kb[(mt * 2 + 0) * 8 + 4 * ks + 2 * t + 0] = c[mt][ks][t][0];
              kb[(mt * 2 + 0) * 8 + 4 * ks + 2 * t + 1] = c[mt][ks][t][1];
              kb[(mt * 2 + 1) * 8 + 4 * ks + 2 * t + 0] = c[mt][ks][t][2];
              kb[(mt * 2 + 1) * 8 + 4 * ks + 2 * t + 1] = c[mt][ks][t][3];
            }
        const uint32_t ta = tcol + (uint32_t)(32 * i);
        if (l >= 1) {
          float acc[32];
          tmem_ld32(ta, acc);
          tmem_wait_ld();
#pragma unroll
          for (int e = 0; e < 32; ++e) kb[e] += acc[e];
        }
        tmem_st32(ta, kb);
        tmem_wait_st();
      }
    }
    bar_sync(1, (KP_LWARPS + KP_KWARPS) * 32);  // pairs with the logit warps' barrier before the ring is reused
    for (int i = 0; i < my_tiles; ++i) {
      const int tile = blockIdx.x + i * gridDim.x;
      const bool is_x = tile >= tiles_c;
      const int t0 = (is_x ? tile - tiles_c : tile) * KP_TOK;
      const int nvalid = min(KP_TOK, (is_x ? nx : nc) - t0);
      float kb[32];
      tmem_ld32(tcol + (uint32_t)(32 * i), kb);
      tmem_wait_ld();
      float* outp = is_x ? p.kq : p.kbar;
      if (q < CW) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int tok = (j >> 1) * 16 + r + 8 * (j & 1);
          if (tok < nvalid) {
            float4* d4 = reinterpret_cast<float4*>(outp + (int64_t)(t0 + tok) * D + dq * (D / 4) + q * 8);
            d4[0] = make_float4(kb[j * 8 + 0] * inv, kb[j * 8 + 1] * inv, kb[j * 8 + 2] * inv, kb[j * 8 + 3] * inv);
            d4[1] = make_float4(kb[j * 8 + 4] * inv, kb[j * 8 + 5] * inv, kb[j * 8 + 6] * inv, kb[j * 8 + 7] * inv);
          }
        }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == W_STATS) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
  }
  if (p.tstamp && threadIdx.x == 0) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    atomicMax(p.tstamp + 1, t);
  }
}

// shared memory of k_key_pass_lm; returns 0 if not even two stages fit
inline size_t key_pass_lm_smem(int Hq, int Hkv, int D, bool kbar, int max_smem, int* n_stage) {
  const size_t stage = (size_t)KP_TOK * (Hkv * D * 2 + KP_ROWPAD);
  const size_t fixed = (size_t)(kbar ? LM_MT_KBAR : LM_MT) * 32 * 4 + 4 * (size_t)((Hq + 1) & ~1) * (4 + 8) + LM_SWARPS * (size_t)((Hq + 1) & ~1) * 8 + 2 * 8 * 8 + 4 * 8 + 64 + 128;
  if (fixed + 2 * stage > (size_t)max_smem) { *n_stage = 0; return 0; }
  int ns = (int)(((size_t)max_smem - fixed) / stage);
  if (ns > 8) ns = 8;
  *n_stage = ns;
  return fixed + (size_t)ns * stage;
}

}  // namespace ikv
