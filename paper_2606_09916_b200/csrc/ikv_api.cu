// ikv_api.cu -- C-ABI of libikv (include/ikv.h): host-side session/scratch manager and kernel launches.
// Everything on the hot path runs in the kernels of score.cuh / residual.cuh / select.cuh / decode.cuh.
#include <cuda.h>
#include <limits.h>
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>

#include <type_traits>

#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/ikv.h"
#include "common.cuh"
#include "decode.cuh"
#include "decode_mma.cuh"
#include "residual_mma.cuh"
#include "residual_tc.cuh"
#include "score.cuh"
#include "score_mma.cuh"
#include "score_lm.cuh"
#include "score_rows_tc.cuh"
#include "prefill_mma.cuh"
#include "prefill_tc.cuh"
#include "loss.cuh"
#include "select.cuh"
#include "select_cluster.cuh"
#include "fused_small.cuh"

using namespace ikv;

namespace {

struct Session {
  uint64_t id = 0;
  float* d_mem = nullptr;   // M_t      [L][Hq][D]
  float* d_qenc = nullptr;  // normalize(Enc(q_t)) of the latest update
  uint64_t tick = 0;
  bool has_update = false;
  // compact survivor list for decode
  int32_t* live_slots = nullptr;
  int32_t* d_n_live = nullptr;
  int live_cap = 0;
  int covered = 0;            // positions [0, covered) are represented by the list
  int live_ub = 0;            // host upper bound of the list length
  const int32_t* map_ptr = nullptr;
  uint32_t map_epoch = 0;     // ikv_request.map_epoch at the last select / rescan
  bool list_fresh = false;    // live_slots was rewritten by the last library launch on this session: the next decode
                              // launch is made WITHOUT programmatic serialization (full stream order), see R27
};

template <typename T>
struct DevBuf {
  T* p = nullptr;
  size_t n = 0;
};

}  // namespace

// Scratch of ikv_decode_attn_static: [0, 256) a zero word (the empty survivor list's length) | split partials.  In host
// code this name is a host-side stand-in, never a device address: ikv_create resolves it with cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[IKV_STATIC_SCRATCH_BYTES];

// Scratch of one score pass (a1-a5 of one request).  The context derives from it: its own copy is the set in use; a
// batched ikv_score gives every lane a set of its own and swaps it in around that lane's launches (the kernels take
// the pointers by value).
struct Scratch {
  uint4* frag = nullptr;     // B fragments of M / sqrt(D) for the bf16 key pass
  int32_t* lm_cnt = nullptr; // per-layer arrival counters of k_key_pass_lm
  int64_t cap_tokens = 0;    // token-sized buffers (ensure_scratch)
  int32_t *cand_pos = nullptr, *cand_slot = nullptr, *d_ncand = nullptr;
  float* logits = nullptr;
  float2* partials = nullptr;
  float *lse = nullptr, *rule_c = nullptr, *kbar = nullptr, *mbar = nullptr;
  int32_t *xq_slot = nullptr, *d_nxq = nullptr;
  float* kq = nullptr;
  uint4 *kc_frag = nullptr, *vc_frag = nullptr;  // B fragments of Kc / Vc (Eq. 6)
  int64_t xq_cap = 0;
  // folded residual operands of the current call (residual_mma.cuh)
  float *mpart = nullptr, *bq_eff = nullptr, *b1_eff = nullptr;
  uint4* wq_frag = nullptr;
  unsigned char* w1_can = nullptr;  // fc1' chunks for tcgen05 (residual_mma.cuh)
  unsigned char* rt_wcan = nullptr; // operand chunks of k_residual_tc (residual_tc.cuh)
  float* rt_svec = nullptr;         // s_r | s_b
  uint8_t* keepflag = nullptr;      // select fallback (maps > CL_MAX_N)
  int32_t* tmp_slot = nullptr;
};
constexpr int IKV_MAX_LANES = 8;

struct ikv_ctx : Scratch {
  ikv_config cfg;
  int G = 1;
  int64_t layer_stride = 0;  // elements
  std::unordered_map<uint64_t, Session> sessions;
  uint64_t tick = 0;
  std::string err;
  int n_sm = 148;
  int max_smem = 48 * 1024;  // opt-in dynamic shared memory per CTA
  bool use_pdl = true;       // programmatic dependent launch between decode kernels (IKV_CFG_NO_PDL disables)
  bool pdl_prune = true;     // ... and along the kernels of the prune pass (IKV_CFG_NO_PDL_PRUNE disables)
  bool attr_done[2][2][9] = {};
  int dbg_l2 = 7;            // IKV_TUNE_L2_HINTS
  int use_lm = 1;            // IKV_TUNE_LAYER_MAJOR

  // lanes of a batched ikv_score: the small kernels of request r run on stream r % n_lanes with that lane's scratch,
  // the key passes in request order on the caller's stream (lane 0 uses the context's own set)
  int n_lanes = 4;           // IKV_TUNE_BATCH_LANES
  int lanes_ready = 0;
  Scratch lane_set[IKV_MAX_LANES];
  cudaStream_t lane_stream[IKV_MAX_LANES] = {};
  cudaEvent_t lane_ev[IKV_MAX_LANES][3] = {};  // small -> key, key -> small, join
  cudaEvent_t fork_ev = nullptr;

  unsigned char* static_scratch = nullptr;  // device address of g_static_scratch on this context's device
  std::string static_scratch_err;           // why it could not be resolved

  bool pf_attr_done[2][9] = {};
  bool pt_attr_done[2][2][2][9] = {};
  CUtensorMap tm_k, tm_v;    // the pools as 2-D tensors [L n_slots H_kv][D], box 64 x 1, SWIZZLE_128B (TMA gather4)
  bool tm_ok = false;
  int prefill_tiled = 1;     // IKV_TUNE_PREFILL_TILED: 0 = ikv_prefill_attn row by row through the decode kernels
  // multi-row scorer on tcgen05 (score_rows_tc.cuh)
  int rows_tc = 1;           // IKV_TUNE_ROWS_TC
  unsigned char* rows_bank = nullptr;
  float2* rows_partials = nullptr;
  size_t rows_partials_cap = 0;
  bool rows_attr_done = false;

  uint32_t* kept_bits = nullptr;
  int32_t* firstpos = nullptr;
  float* part_o = nullptr;
  float2* part_ml = nullptr;
  int64_t part_cap = 0;  // in (req*Hq*split) units
  // ikv_prune_host staging
  int32_t *st_map = nullptr, *st_freed = nullptr, *st_counts = nullptr;
  uint8_t* st_valid = nullptr;
  float *st_scores = nullptr, *st_qrows = nullptr;
  int64_t st_cap = 0, st_qcap = 0;
  unsigned char* st_out = nullptr;   // device: [counts 16 B][slot map cap*4][freed cap*4][valid cap], one D2H copy
  unsigned char* st_host = nullptr;  // pinned host mirror of st_out

  // kernel-level profiling (ikv_profile_*)
  int prof_on = 0;           // 0 off, 1 the two dominant kernels, 2 every kernel of the path
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_ev[IKV_PROF_SLOTS];
  std::vector<cudaEvent_t> ev_pool;   // events are created once and reused (ikv_profile_read returns them here)
  // level 1 times the layer-major key pass by in-kernel %globaltimer stamps ({min start, max end} per launch): host
  // events between programmatically launched kernels would take their overlap away and inflate the pass being timed
  unsigned long long* ts_ring = nullptr;
  int ts_used = 0;
  static constexpr int TS_SLOTS = 4096;

  // residual head (transposed on the device)
  bool has_resid = false;
  bool resid_attr_done = false;
  int tail_smem_set = 0;     // dynamic shared memory k_tail_tc was last configured for
  int resid_tc = 1;          // IKV_TUNE_RESID_TC: 0 = always the unfolded kernel
  float* resid_blob = nullptr;
  ResidW rw{};
};

namespace {

#define IKV_FAIL(ctx, code, ...)                         \
  do {                                                   \
    char _b[512];                                        \
    snprintf(_b, sizeof _b, __VA_ARGS__);                \
    (ctx)->err = _b;                                     \
    return (code);                                       \
  } while (0)

#define CU(ctx, call)                                                                              \
  do {                                                                                             \
    cudaError_t _e = (call);                                                                       \
    if (_e != cudaSuccess) {                                                                       \
      const bool oom = (_e == cudaErrorMemoryAllocation);                                          \
      IKV_FAIL(ctx, oom ? IKV_ERR_OOM : IKV_ERR_CUDA, "%s failed: %s (%s:%d)", #call,              \
               cudaGetErrorString(_e), __FILE__, __LINE__);                                        \
    }                                                                                              \
  } while (0)

#define LAUNCH_CHECK(ctx)                                                                          \
  do {                                                                                             \
    cudaError_t _e = cudaGetLastError();                                                           \
    if (_e != cudaSuccess)                                                                         \
      IKV_FAIL(ctx, IKV_ERR_CUDA, "kernel launch failed: %s (%s:%d)", cudaGetErrorString(_e),      \
               __FILE__, __LINE__);                                                                \
  } while (0)

struct ProfScope {  // brackets a launch with events when profiling is on and the stream is not capturing
  ikv_ctx* c; int which; cudaStream_t st; cudaEvent_t a = nullptr, b = nullptr;
  ProfScope(ikv_ctx* c_, int which_, cudaStream_t st_) : c(c_), which(which_), st(st_) {
    if (!c->prof_on || which >= IKV_PROF_SLOTS || (c->prof_on < 2 && which > IKV_PROF_DECODE)) return;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    cudaStreamIsCapturing(st, &cs);
    if (cs != cudaStreamCaptureStatusNone) return;
    a = take();
    b = take();
    cudaEventRecord(a, st);
  }
  cudaEvent_t take() {
    if (!c->ev_pool.empty()) { cudaEvent_t e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
  }
  ~ProfScope() {
    if (!a) return;
    cudaEventRecord(b, st);
    c->prof_ev[which].emplace_back(a, b);
  }
};

template <typename T>
ikv_status grow(ikv_ctx* ctx, T** p, size_t count) {
  if (*p) CU(ctx, cudaFree(*p));
  *p = nullptr;
  CU(ctx, cudaMalloc((void**)p, count * sizeof(T)));
  return IKV_OK;
}

#define TRY(expr)                      \
  do {                                 \
    ikv_status _s = (expr);            \
    if (_s != IKV_OK) return _s;       \
  } while (0)

// Launch with the programmatic-stream-serialization attribute (PDL): the kernel may start while its predecessor in
// the stream drains; it orders itself with griddepcontrol.wait.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*fn)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                       Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, fn, KArgs(args)...);
}

// Test support (ikv_test_late_writer): a producer that triggers its dependents FIRST, idles, and only then writes.
__global__ void k_late_writer(uint4* dst, const uint4* src, int64_t n16, int64_t delay_ns) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  unsigned long long t0, t1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  do { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); } while ((long long)(t1 - t0) < delay_ns);
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n16; i += (int64_t)gridDim.x * blockDim.x)
    dst[i] = src[i];
}

// scores[pos_c] = (first ? 0 : scores[pos_c]) + w * rule_c[c]   (multi-row scorer: weighted sum over the rows)
__global__ void k_axpy_scatter(const float* __restrict__ rule_c, const int32_t* __restrict__ cand_pos,
                               const int32_t* __restrict__ n_cand, float w, int first, float* __restrict__ scores) {
  pdl_wait();
  pdl_launch_dependents();
  const int nc = *n_cand;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
    const int pos = cand_pos[c];
    scores[pos] = (first ? 0.f : scores[pos]) + w * rule_c[c];
  }
}
// StreamingLLM (sink + recent window; R30): position scores of the candidates
__global__ void k_streaming_scores(const int32_t* __restrict__ cand_pos, const int32_t* __restrict__ n_cand, int n_sink,
                                   float* __restrict__ scores) {
  const int nc = *n_cand;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
    const int pos = cand_pos[c];
    scores[pos] = pos < n_sink ? 1073741824.f : (float)pos;
  }
}
// SnapKV max-pool smoothing over the logical positions, candidates only ("kernel 7 ... max-pool"; R29).
// scores holds finite values exactly at the candidates (+-INF fillers elsewhere, R6).  Two launches: pooled -> tmp -> back.
__global__ void k_maxpool_cand(const float* __restrict__ scores, const int32_t* __restrict__ cand_pos,
                               const int32_t* __restrict__ n_cand, int N, int half, float* __restrict__ tmp) {
  const int nc = *n_cand;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
    const int pos = cand_pos[c];
    float m = scores[pos];
    for (int i = max(0, pos - half); i <= min(N - 1, pos + half); ++i) {
      const float v = scores[i];
      if (isfinite(v) && v > m) m = v;
    }
    tmp[c] = m;
  }
}
// H2O "ratio mode with a recent-window floor" (R31): the n_recent most recent candidates are kept
// first (score 1e30 + position).  One block: |F| is counted from the +INF fillers.
__global__ __launch_bounds__(1024) void k_h2o_boost(const int32_t* __restrict__ cand_pos, const int32_t* __restrict__ n_cand,
                                                    int N, int C, float ratio, int floor_, float* __restrict__ scores) {
  __shared__ int warp_tot[32];
  int nf = 0;
  for (int j = threadIdx.x; j < N; j += 1024) nf += (scores[j] == CUDART_INF_F) ? 1 : 0;
  int tot;
  block_excl_scan_1024(nf, warp_tot, &tot);
  const int cstar = max(0, C - tot);
  int n_recent = (int)floorf(ratio * (float)cstar + 0.5f);
  n_recent = min(cstar, max(floor_, n_recent));
  const int nc = *n_cand;
  __syncthreads();
  for (int c = max(0, nc - n_recent) + threadIdx.x; c < nc; c += 1024) {
    const int pos = cand_pos[c];
    scores[pos] = 1.0e30f + (float)pos;
  }
}
// KV-read counters of a prefill chunk: raw += sum (pos_i + 1), eff += sum #live positions <= pos_i.
// n_live (may be NULL) = number of live positions in [0, covered), covered <= q_pos0: only the gap is scanned.
__global__ __launch_bounds__(1024) void k_prefill_reads(const int32_t* __restrict__ S, int32_t dead, int q_pos0, int n_q,
                                                        unsigned long long* __restrict__ reads,
                                                        const int32_t* __restrict__ n_live, int covered) {
  __shared__ int warp_tot[32];
  // live positions in [0, q_pos0) are common to every row; then an inclusive count along the chunk
  int base = n_live ? *n_live : 0;
  for (int j0 = n_live ? covered : 0; j0 < q_pos0; j0 += 1024) {
    const int j = j0 + threadIdx.x;
    int tot;
    block_excl_scan_1024((j < q_pos0 && S[j] != dead) ? 1 : 0, warp_tot, &tot);
    base += tot;
  }
  unsigned long long eff = 0;
  int run = base;
  for (int i0 = 0; i0 < n_q; i0 += 1024) {
    const int i = i0 + threadIdx.x, j = q_pos0 + i;
    const int lv = (i < n_q && S[j] != dead) ? 1 : 0;
    int tot;
    const int ex = block_excl_scan_1024(lv, warp_tot, &tot);
    if (i < n_q) eff += (unsigned long long)(run + ex + lv);
    run += tot;
  }
  // block sum of eff
  __shared__ unsigned long long acc;
  if (threadIdx.x == 0) acc = 0;
  __syncthreads();
  atomicAdd(&acc, eff);
  __syncthreads();
  if (threadIdx.x == 0) {
    atomicAdd(&reads[0], (unsigned long long)n_q * (unsigned long long)(q_pos0 + 1) +
                             (unsigned long long)n_q * (unsigned long long)(n_q - 1) / 2);
    atomicAdd(&reads[1], acc);
  }
}

__global__ void k_fill_i32(int32_t* p, int64_t n, int32_t v) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    p[i] = v;
}

template <typename T>
__global__ void k_init_dead(T* k_pool, T* v_pool, int64_t layer_stride, int L, int row /* Hkv*D */, int64_t slot) {
  const int l = blockIdx.x;
  for (int i = threadIdx.x; i < row; i += blockDim.x) {
    k_pool[(int64_t)l * layer_stride + slot * row + i] = (T)(-1.0e4f);
    v_pool[(int64_t)l * layer_stride + slot * row + i] = (T)0.f;
  }
}

int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

// The buffers of a scratch set whose size depends on the model shape only.
bool scratch_alloc_fixed(Scratch& s, const ikv_config& cfg) {
  const int LH = cfg.n_layers * cfg.n_q_heads, KS = cfg.head_dim / 16;
  bool ok = cudaMalloc((void**)&s.d_ncand, 4) == cudaSuccess && cudaMalloc((void**)&s.d_nxq, 4) == cudaSuccess;
  ok = ok && cudaMemset(s.d_nxq, 0, 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.lse, (size_t)LH * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.lm_cnt, (size_t)cfg.n_layers * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.mbar, (size_t)cfg.head_dim * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.mpart, (size_t)((LH + 31) / 32) * cfg.head_dim * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.bq_eff, R_DC * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.b1_eff, R_HID * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.wq_frag, (size_t)KS * 16 * 32 * sizeof(uint4)) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.w1_can, (size_t)2 * (cfg.head_dim / 64 + 2) * W1C_CHUNK) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.rt_wcan, rt_wcan_bytes(cfg.head_dim)) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&s.rt_svec, 512 * 4) == cudaSuccess;
  // B fragments: [L][Hkv][NT<=2][D/32][32 lanes] uint4
  ok = ok && cudaMalloc((void**)&s.frag, (size_t)cfg.n_layers * cfg.n_kv_heads * 2 * (cfg.head_dim / 32) * 32 *
                                             sizeof(uint4)) == cudaSuccess;
  return ok;
}

void scratch_free(Scratch& s) {
  void* bufs[] = {s.frag, s.lm_cnt, s.cand_pos, s.cand_slot, s.d_ncand, s.logits, s.partials, s.lse, s.rule_c, s.kbar,
                  s.mbar, s.xq_slot, s.d_nxq, s.kq, s.kc_frag, s.vc_frag, s.mpart, s.bq_eff, s.b1_eff, s.wq_frag,
                  s.w1_can, s.rt_wcan, s.rt_svec, s.keepflag, s.tmp_slot};
  for (void* b : bufs) cudaFree(b);
  s = Scratch{};
}

ikv_status ensure_scratch(ikv_ctx* c, int64_t tokens) {
  if (tokens <= c->cap_tokens) return IKV_OK;
  const int L = c->cfg.n_layers, Hq = c->cfg.n_q_heads, D = c->cfg.head_dim;
  const int64_t cap = round_up(tokens, 1024);
  const int64_t n_tiles = cap / SCORE_TILE;
  c->cap_tokens = 0;  // a failed growth must not leave the old capacity standing over freed buffers
  TRY(grow(c, &c->cand_pos, cap));
  TRY(grow(c, &c->cand_slot, cap));
  TRY(grow(c, &c->logits, (size_t)L * Hq * cap));
  TRY(grow(c, &c->partials, (size_t)L * Hq * (n_tiles > c->n_sm ? n_tiles : c->n_sm)));
  TRY(grow(c, &c->rule_c, cap));
  TRY(grow(c, &c->kbar, (size_t)cap * D));
  TRY(grow(c, &c->keepflag, cap));
  TRY(grow(c, &c->tmp_slot, cap));
  c->cap_tokens = cap;
  return IKV_OK;
}

ikv_status ensure_xq(ikv_ctx* c, int64_t n) {
  if (n <= c->xq_cap) return IKV_OK;
  const int64_t cap = round_up(n, 256);
  c->xq_cap = 0;
  TRY(grow(c, &c->xq_slot, cap));
  TRY(grow(c, &c->kq, (size_t)cap * c->cfg.head_dim));
  TRY(grow(c, &c->kc_frag, (size_t)cap * 32));  // 4 heads x 2 k-steps x cap/8 tiles x 32 lanes
  TRY(grow(c, &c->vc_frag, (size_t)cap * 32));  // 4 heads x cap/16 steps x 4 tiles x 32 lanes
  c->xq_cap = cap;
  return IKV_OK;
}

ikv_status ensure_parts(ikv_ctx* c, int64_t units) {
  if (units <= c->part_cap) return IKV_OK;
  c->part_cap = 0;
  TRY(grow(c, &c->part_o, (size_t)units * c->cfg.head_dim));
  TRY(grow(c, &c->part_ml, (size_t)units));
  c->part_cap = units;
  return IKV_OK;
}

ikv_status ensure_staging(ikv_ctx* c, int64_t tokens, int64_t qelems) {
  if (tokens > c->st_cap) {
    const int64_t cap = round_up(tokens, 1024);
    const size_t bytes = 16 + (size_t)cap * 9;
    c->st_cap = 0;
    if (c->st_out) CU(c, cudaFree(c->st_out));
    if (c->st_host) CU(c, cudaFreeHost(c->st_host));
    c->st_out = nullptr; c->st_host = nullptr;
    CU(c, cudaMalloc((void**)&c->st_out, bytes));
    CU(c, cudaMallocHost((void**)&c->st_host, bytes));
    c->st_counts = reinterpret_cast<int32_t*>(c->st_out);
    c->st_map = reinterpret_cast<int32_t*>(c->st_out + 16);
    c->st_freed = c->st_map + cap;
    c->st_valid = reinterpret_cast<uint8_t*>(c->st_freed + cap);
    TRY(grow(c, &c->st_scores, cap));
    c->st_cap = cap;
  }
  if (qelems > c->st_qcap) {
    c->st_qcap = 0;
    TRY(grow(c, &c->st_qrows, qelems));
    c->st_qcap = qelems;
  }
  return IKV_OK;
}

ikv_status session_live_reserve(ikv_ctx* c, Session& s, int n) {
  if (n <= s.live_cap) return IKV_OK;
  const int cap = (int)round_up((int64_t)n + n / 4 + 1024, 1024);
  s.live_cap = 0;
  TRY(grow(c, &s.live_slots, cap));
  s.live_cap = cap;
  s.covered = 0;
  s.map_ptr = nullptr;
  return IKV_OK;
}

void session_free(Session& s) {
  cudaFree(s.d_mem);
  cudaFree(s.d_qenc);
  cudaFree(s.live_slots);
  cudaFree(s.d_n_live);
}

// M_0 = 0 (R3).  The zero fills are enqueued on `st`, the stream the session's first use is enqueued on; with
// `sync` (ikv_session_open, which has no stream) the host waits for them, so that they are ordered before work on any
// stream, including non-blocking ones.
ikv_status session_create(ikv_ctx* c, uint64_t id, Session** out, cudaStream_t st, bool sync) {
  auto it = c->sessions.find(id);
  if (it == c->sessions.end()) {
    if ((int)c->sessions.size() >= c->cfg.max_sessions) {  // LRU eviction
      auto victim = c->sessions.begin();
      for (auto jt = c->sessions.begin(); jt != c->sessions.end(); ++jt)
        if (jt->second.tick < victim->second.tick) victim = jt;
      session_free(victim->second);
      c->sessions.erase(victim);
    }
    Session s;
    s.id = id;
    const size_t n = (size_t)c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim;
    CU(c, cudaMalloc((void**)&s.d_mem, n * sizeof(float)));
    CU(c, cudaMalloc((void**)&s.d_qenc, n * sizeof(float)));
    CU(c, cudaMalloc((void**)&s.d_n_live, sizeof(int32_t)));
    it = c->sessions.emplace(id, s).first;
  }
  Session& s = it->second;
  const size_t n = (size_t)c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim;
  CU(c, cudaMemsetAsync(s.d_mem, 0, n * sizeof(float), st));  // M_0 = 0 (R3)
  CU(c, cudaMemsetAsync(s.d_qenc, 0, n * sizeof(float), st));
  CU(c, cudaMemsetAsync(s.d_n_live, 0, sizeof(int32_t), st));
  if (sync) CU(c, cudaStreamSynchronize(st));
  s.has_update = false;
  s.list_fresh = false;
  s.covered = 0;
  s.map_ptr = nullptr;
  s.tick = ++c->tick;
  *out = &s;
  return IKV_OK;
}

Session* session_find(ikv_ctx* c, uint64_t id) {
  auto it = c->sessions.find(id);
  if (it == c->sessions.end()) return nullptr;
  it->second.tick = ++c->tick;
  return &it->second;
}

ikv_status check_request(ikv_ctx* c, const ikv_request& r) {
  if (r.seq_len < 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "seq_len < 0");
  if (r.seq_len > 0 && !r.slot_map) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "slot_map is NULL");
  if (!(0 <= r.prefix_len && r.prefix_len <= r.q_start && r.q_start <= r.q_end && r.q_end <= r.seq_len))
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "need 0 <= prefix_len <= q_start <= q_end <= seq_len (got %d %d %d %d)",
             r.prefix_len, r.q_start, r.q_end, r.seq_len);
  if (r.budget < 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "budget < 0");
  if (r.radix_protected_len < 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "radix_protected_len < 0");
  if (r.n_xattn_pos < 0 || (r.n_xattn_pos > 0 && !r.xattn_pos))
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "bad xattn_pos / n_xattn_pos");
  return IKV_OK;
}

// ---- typed launch helpers -------------------------------------------------------------------------------
template <typename T, int D, int G>
ikv_status launch_logits(ikv_ctx* c, const Session& s, const float* M, int N, bool kbar, cudaStream_t st) {
  const int L = c->cfg.n_layers, Hkv = c->cfg.n_kv_heads, Hq = c->cfg.n_q_heads;
  const int n_tiles = (N + SCORE_TILE - 1) / SCORE_TILE;
  const int64_t ldc = c->cap_tokens;
  const size_t smem = (size_t)Hq * (SCORE_TILE + 1) * 4 + SCORE_TILE * 4 + (kbar ? (size_t)SCORE_TILE * D * 4 : 0);
  const float isd = 1.0f / sqrtf((float)D);
  ProfScope prof(c, 0, st);
  if (kbar) {
    auto fn = k_score_logits<T, D, G, true>;
    if (smem > 48 * 1024) CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    fn<<<n_tiles, 256, smem, st>>>((const T*)c->cfg.k_pool, c->layer_stride, L, Hkv, M, c->cand_slot, c->d_ncand,
                                   c->cfg.dead_slot, c->logits, ldc, c->partials, n_tiles, c->kbar, isd);
  } else {
    auto fn = k_score_logits<T, D, G, false>;
    if (smem > 48 * 1024) CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    fn<<<n_tiles, 256, smem, st>>>((const T*)c->cfg.k_pool, c->layer_stride, L, Hkv, M, c->cand_slot, c->d_ncand,
                                   c->cfg.dead_slot, c->logits, ldc, c->partials, n_tiles, nullptr, isd);
  }
  LAUNCH_CHECK(c);
  (void)s;
  return IKV_OK;
}

template <typename T, int D>
ikv_status dispatch_logits_g(ikv_ctx* c, const Session& s, const float* M, int N, bool kbar, cudaStream_t st) {
  switch (c->G) {
    case 1: return launch_logits<T, D, 1>(c, s, M, N, kbar, st);
    case 2: return launch_logits<T, D, 2>(c, s, M, N, kbar, st);
    case 4: return launch_logits<T, D, 4>(c, s, M, N, kbar, st);
    case 5: return launch_logits<T, D, 5>(c, s, M, N, kbar, st);
    case 8: return launch_logits<T, D, 8>(c, s, M, N, kbar, st);
  }
  IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "GQA group size %d not supported (1,2,4,5,8)", c->G);
}

ikv_status dispatch_logits(ikv_ctx* c, const Session& s, const float* M, int N, bool kbar, cudaStream_t st) {
  // plain-FMA kernel: fp32 pools only (the bf16 pools take k_key_pass)
  if (c->cfg.head_dim == 128) return dispatch_logits_g<float, 128>(c, s, M, N, kbar, st);
  return dispatch_logits_g<float, 64>(c, s, M, N, kbar, st);
}

template <typename T, int D, int G>
ikv_status launch_decode(ikv_ctx* c, int layer, const DecBatch& batch, int n_req, int n_split, const void* q,
                         void* out, float sm_scale, cudaStream_t st, bool pdl_split) {
  const int Hkv = c->cfg.n_kv_heads, Hq = c->cfg.n_q_heads;
  const T* kl = (const T*)c->cfg.k_pool + (int64_t)layer * c->layer_stride;
  const T* vl = (const T*)c->cfg.v_pool + (int64_t)layer * c->layer_stride;
  if constexpr (std::is_same<T, bf16>::value) {
    // tensor-pipe split kernel behind a bulk-copy ring (decode_mma.cuh).  At most half an SM's shared memory per
    // CTA: the CTAs of two consecutive layer calls co-reside (PDL), so the next call's K/V stream starts while this
    // call drains.
    const int n_hg = (Hkv + DM_CWARPS - 1) / DM_CWARPS;
    int nhalf = 0;
    const size_t smem = decode_mma_smem(Hkv < DM_CWARPS ? Hkv : DM_CWARPS, D, (c->max_smem + 1024) / 2 - 1024, &nhalf);
    if (nhalf < 2) IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "decode: a half-stage of %d heads x %d does not fit", Hkv, D);
    DecMmaParams p;
    p.k_layer = kl; p.v_layer = vl; p.Hkv = Hkv; p.dead = c->cfg.dead_slot; p.q = (const bf16*)q; p.sm_scale = sm_scale;
    p.part_o = c->part_o; p.part_ml = c->part_ml; p.n_split = n_split; p.n_stage = nhalf;
    auto fn = k_decode_mma<D, G>;
    if (!c->attr_done[0][D == 128][G]) {
      CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      c->attr_done[0][D == 128][G] = true;
    }
    {
      ProfScope prof(c, 1, st);
      CU(c, launch_pdl(fn, dim3(n_split, n_req, n_hg), dim3(DM_THREADS), smem, st, pdl_split, p, batch));
    }
  } else {
    constexpr int VEC = Elem<T>::VEC;
    constexpr int NGRP = 4 * (32 / (D / VEC));
    const size_t smem = (size_t)NGRP * G * (D + 2) * 4;
    auto fn = k_decode_split<T, D, G>;
    if (smem > 48 * 1024) CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ProfScope prof(c, 1, st);
    fn<<<dim3(n_split, Hkv, n_req), 128, smem, st>>>(kl, vl, Hkv, c->cfg.dead_slot, batch, (const T*)q, sm_scale,
                                                     c->part_o, c->part_ml, n_split);
    LAUNCH_CHECK(c);
  }
  ProfScope prof(c, IKV_PROF_DECODE_MERGE, st);
  CU(c, launch_pdl(k_decode_merge4<T, D>, dim3(Hq, n_req), dim3(DMG_THREADS), 0, st, c->use_pdl, (const float*)c->part_o,
                   (const float2*)c->part_ml, n_split, batch, (T*)out));
  return IKV_OK;
}

template <typename T, int D>
ikv_status dispatch_decode_g(ikv_ctx* c, int layer, const DecBatch& b, int n_req, int n_split, const void* q,
                             void* out, float sc, cudaStream_t st, bool pdl) {
  switch (c->G) {
    case 1: return launch_decode<T, D, 1>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
    case 2: return launch_decode<T, D, 2>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
    case 4: return launch_decode<T, D, 4>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
    case 5: return launch_decode<T, D, 5>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
    case 8: return launch_decode<T, D, 8>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
  }
  IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "GQA group size %d not supported (1,2,4,5,8)", c->G);
}

ikv_status dispatch_decode(ikv_ctx* c, int layer, const DecBatch& b, int n_req, int n_split, const void* q,
                           void* out, float sc, cudaStream_t st, bool pdl) {
  const bool bf = c->cfg.kv_dtype == IKV_BF16;
  if (c->cfg.head_dim == 128) return bf ? dispatch_decode_g<bf16, 128>(c, layer, b, n_req, n_split, q, out, sc, st, pdl)
                                        : dispatch_decode_g<float, 128>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
  return bf ? dispatch_decode_g<bf16, 64>(c, layer, b, n_req, n_split, q, out, sc, st, pdl)
            : dispatch_decode_g<float, 64>(c, layer, b, n_req, n_split, q, out, sc, st, pdl);
}

// bf16 key pass on the tensor pipe.  Layer-major with deferred normalisation (score_lm.cuh) when the call fits its
// on-chip capacity: *lm_done = true, rule_c / scores / k_bar are final.  Otherwise k_key_pass (score_mma.cuh): logits
// scratch + partials, *n_part = number of partial (max, sum) columns.
struct LmOut { float* scores; float* rule_out; int scatter; };
// lane != nullptr (batched ikv_score): the key pass goes on lane->kst, after the work enqueued on st so far, and st
// continues after it.
struct KeyLane { cudaStream_t kst; cudaEvent_t to_key, from_key; };

template <int D, int G>
ikv_status launch_key_pass(ikv_ctx* c, const float* M, bool kbar, bool with_xq, int n_mpart, int* n_part, int N, int n_x,
                           const LmOut& lo, bool* lm_done, cudaStream_t st, const KeyLane* lane) {
  const int L = c->cfg.n_layers, Hkv = c->cfg.n_kv_heads, Hq = c->cfg.n_q_heads;
  const int n_fb = mem_prep_frag_blocks<D, G>(L, Hkv);
  const int grid = c->n_sm;
  bool lm = false;
  if constexpr (G <= 4) {
    const int tiles_ub = (N + KP_TOK - 1) / KP_TOK + ((with_xq ? n_x : 0) + KP_TOK - 1) / KP_TOK;
    // every layer costs the grid one statistics round trip (~4 us): below three tiles per CTA the logits-scratch
    // kernel is faster (IKV_TUNE_LAYER_MAJOR = 2 takes the layer-major kernel whenever the call fits its capacity)
    // In a batch (lane != nullptr) the rule kernel of the logits-scratch path runs on the lane's stream under the next
    // request's key pass, and the layer-major kernel's per-layer round trips are not hidden by anything: measured on
    // configs[4] 13.7 -> 13.4 ms (24 layers), 6.35 -> 5.85 ms (8 layers).
    lm = c->use_lm && Hkv <= KP_LWARPS && (tiles_ub + grid - 1) / grid <= (kbar ? LM_MT_KBAR : LM_MT) &&
         (c->use_lm >= 2 || (tiles_ub >= 3 * grid && !lane));
  }
  {
    ProfScope prof(c, IKV_PROF_MEM_PREP, st);
    CU(c, launch_pdl(k_mem_prep<D, G>, dim3(n_fb + n_mpart), dim3(128), 0, st, c->pdl_prune, M, L, Hkv,
                     1.0f / sqrtf((float)D), c->frag, n_fb, L * Hq, c->mpart, lm ? c->lm_cnt : (int32_t*)nullptr));
  }
  *lm_done = lm;
  cudaStream_t ks = st;
  if (lane) {
    ks = lane->kst;
    CU(c, cudaEventRecord(lane->to_key, st));
    CU(c, cudaStreamWaitEvent(ks, lane->to_key, 0));
  }
  auto rejoin = [&]() -> ikv_status {
    if (lane) {
      CU(c, cudaEventRecord(lane->from_key, ks));
      CU(c, cudaStreamWaitEvent(st, lane->from_key, 0));
    }
    return IKV_OK;
  };
  if constexpr (G <= 4) {
    if (lm) {
      int ns = 0;
      const size_t smem = key_pass_lm_smem(Hq, Hkv, D, kbar, c->max_smem, &ns);
      if (ns < 2) IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "key pass: a stage of %d bytes does not fit shared memory", Hkv * D * 2 * KP_TOK);
      KeyPassLmParams p;
      p.k_pool = (const bf16*)c->cfg.k_pool; p.layer_stride = c->layer_stride; p.L = L; p.Hkv = Hkv; p.frag = c->frag;
      p.cand_slot = c->cand_slot; p.cand_pos = c->cand_pos; p.n_cand = c->d_ncand;
      p.xq_slot = with_xq ? c->xq_slot : nullptr; p.n_xq = with_xq ? c->d_nxq : nullptr;
      p.partials = c->partials; p.layer_cnt = c->lm_cnt; p.rule_c = c->rule_c;
      p.scores = lo.scores; p.rule_out = lo.rule_out; p.scatter_scores = lo.scatter;
      p.kbar = c->kbar; p.kq = c->kq; p.n_stage = ns; p.l2_hints = c->dbg_l2;
      p.tstamp = nullptr;
      p.mpart = c->mpart; p.n_mpart = n_mpart; p.LH = L * Hq; p.mbar_out = (kbar && n_mpart > 0) ? c->mbar : nullptr;
      if (c->prof_on == 1 && c->ts_ring && c->ts_used < ikv_ctx::TS_SLOTS) p.tstamp = c->ts_ring + 2 * (c->ts_used++);
      ProfScope prof(c, c->prof_on == 1 ? IKV_PROF_SLOTS : IKV_PROF_KEY_PASS, ks);  // level 1: stamps instead of events
      if (kbar) {
        auto fn = k_key_pass_lm<D, G, true>;
        CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CU(c, launch_pdl(fn, dim3(grid), dim3(lm_threads(true)), smem, ks, c->pdl_prune, p));
      } else {
        auto fn = k_key_pass_lm<D, G, false>;
        CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CU(c, launch_pdl(fn, dim3(grid), dim3(lm_threads(false)), smem, ks, c->pdl_prune, p));
      }
      *n_part = grid;
      return rejoin();
    }
  }
  int ns = 0;
  const size_t smem = key_pass_smem(L, Hq, Hkv, D, kbar, c->max_smem, &ns);
  if (ns < 2) IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "key pass: L*Hq = %d and row of %d bytes do not fit shared memory", L * Hq,
                       Hkv * D * 2);
  KeyPassParams p;
  p.k_pool = (const bf16*)c->cfg.k_pool; p.layer_stride = c->layer_stride; p.L = L; p.Hkv = Hkv; p.frag = c->frag;
  p.cand_slot = c->cand_slot; p.n_cand = c->d_ncand;
  p.xq_slot = with_xq ? c->xq_slot : nullptr; p.n_xq = with_xq ? c->d_nxq : nullptr;
  p.logits = c->logits; p.ldc = c->cap_tokens; p.partials = c->partials; p.kbar = c->kbar; p.kq = c->kq;
  p.n_stage = ns;
  p.l2_hints = c->dbg_l2;
  {
    ProfScope prof(c, 0, ks);
    if (kbar) {
      auto fn = k_key_pass<D, G, true>;
      CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      CU(c, launch_pdl(fn, dim3(grid), dim3(kp_threads(G, true)), smem, ks, c->pdl_prune, p));
    } else {
      auto fn = k_key_pass<D, G, false>;
      CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      CU(c, launch_pdl(fn, dim3(grid), dim3(kp_threads(G, false)), smem, ks, c->pdl_prune, p));
    }
    LAUNCH_CHECK(c);
  }
  *n_part = grid;
  return rejoin();
}

template <int D>
ikv_status dispatch_key_pass_g(ikv_ctx* c, const float* M, bool kbar, bool xq, int n_mpart, int* n_part, int N, int n_x,
                               const LmOut& lo, bool* lm_done, cudaStream_t st, const KeyLane* lane) {
  switch (c->G) {
    case 1: return launch_key_pass<D, 1>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane);
    case 2: return launch_key_pass<D, 2>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane);
    case 4: return launch_key_pass<D, 4>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane);
    case 5: return launch_key_pass<D, 5>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane);
    case 8: return launch_key_pass<D, 8>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane);
  }
  IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "GQA group size %d not supported (1,2,4,5,8)", c->G);
}

ikv_status dispatch_key_pass(ikv_ctx* c, const float* M, bool kbar, bool xq, int n_mpart, int* n_part, int N, int n_x,
                             const LmOut& lo, bool* lm_done, cudaStream_t st, const KeyLane* lane) {
  return c->cfg.head_dim == 128 ? dispatch_key_pass_g<128>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane)
                                : dispatch_key_pass_g<64>(c, M, kbar, xq, n_mpart, n_part, N, n_x, lo, lm_done, st, lane);
}

// Swaps lane k's scratch set with the context's own for the lifetime of the object (lane 0 is the context's own).
struct LaneSwap {
  ikv_ctx* c; int k;
  LaneSwap(ikv_ctx* c_, int k_) : c(c_), k(k_) { if (k > 0) std::swap(static_cast<Scratch&>(*c), c->lane_set[k]); }
  ~LaneSwap() { if (k > 0) std::swap(static_cast<Scratch&>(*c), c->lane_set[k]); }
};

ikv_status lanes_prepare(ikv_ctx* c, int K) {
  if (!c->fork_ev) CU(c, cudaEventCreateWithFlags(&c->fork_ev, cudaEventDisableTiming));
  for (int k = c->lanes_ready; k < K; ++k) {
    if (!c->lane_stream[k]) CU(c, cudaStreamCreateWithFlags(&c->lane_stream[k], cudaStreamNonBlocking));
    for (cudaEvent_t& e : c->lane_ev[k])
      if (!e) CU(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    if (k > 0 && !c->lane_set[k].frag) {
      if (!scratch_alloc_fixed(c->lane_set[k], c->cfg)) {
        scratch_free(c->lane_set[k]);
        IKV_FAIL(c, IKV_ERR_OOM, "ikv_score: scratch of lane %d: %s", k, cudaGetErrorString(cudaGetLastError()));
      }
      CU(c, cudaDeviceSynchronize());  // the memset of d_nxq is on the legacy stream
    }
    c->lanes_ready = k + 1;
  }
  return IKV_OK;
}

// a1: fillers, candidate list and (n_x > 0) the compaction of the live cross-attention positions as a second cluster of
// the same launch.
ikv_status launch_partition(ikv_ctx* c, const ikv_request& r, int n_x, float* scores, float* rule_out, cudaStream_t st) {
  const int N = r.seq_len;
  const int grid = CL_CTAS * (n_x > 0 ? 2 : 1);
  ProfScope prof(c, IKV_PROF_PARTITION, st);
#define IKV_PART_ARGS r.slot_map, N, c->cfg.dead_slot, r.prefix_len, r.q_start, r.q_end, scores, rule_out, \
                      c->cand_pos, c->cand_slot, c->d_ncand
#define IKV_X_ARGS r.xattn_pos, n_x, c->xq_slot, c->d_nxq
#define IKV_PART_LAUNCH(MAXI) \
  CU(c, launch_pdl(k_partition_cl<MAXI>, dim3(grid), dim3(1024), 0, st, c->pdl_prune, IKV_PART_ARGS, IKV_X_ARGS))
  if (N <= CL_CTAS * 1024 * 4) IKV_PART_LAUNCH(4);
  else if (N <= CL_CTAS * 1024 * 8) IKV_PART_LAUNCH(8);
  else if (N <= CL_MAX_N) IKV_PART_LAUNCH(16);
  else {
    k_partition<<<1, 1024, 0, st>>>(IKV_PART_ARGS);
    if (n_x > 0)
      k_xattn_compact<<<1, 1024, 0, st>>>(r.slot_map, N, c->cfg.dead_slot, r.xattn_pos, n_x, r.q_start, c->xq_slot,
                                          c->d_nxq);
  }
#undef IKV_PART_LAUNCH
#undef IKV_PART_ARGS
#undef IKV_X_ARGS
  LAUNCH_CHECK(c);
  return IKV_OK;
}

// M_ovr: score against these rows [L][Hq][D] instead of the session's memory (multi-row scorer); part: run the partition
// (a1) first; scatter: write the rule score into `scores` (otherwise it stays in the compact rule_c[] scratch).
ikv_status score_one(ikv_ctx* c, const ikv_request& r, int mode, float* scores, float* rule_out, cudaStream_t st,
                     const float* M_ovr = nullptr, bool part = true, bool scatter = true, const KeyLane* lane = nullptr) {
  const int N = r.seq_len;
  if (N == 0) return IKV_OK;
  const int base_mode = mode & 0xff;
  Session* s = session_find(c, r.session_id);
  if (!s) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session %llu does not exist", (unsigned long long)r.session_id);
  const int L = c->cfg.n_layers, Hq = c->cfg.n_q_heads, Hkv = c->cfg.n_kv_heads, D = c->cfg.head_dim;
  const bool learn = (base_mode == IKV_MODE_LEARNABLE) && !(mode & IKV_FLAG_NO_RESIDUAL);
  if (base_mode == IKV_MODE_LEARNABLE && !c->has_resid)
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "IKV_MODE_LEARNABLE needs ikv_residual_load first");
  TRY(ensure_scratch(c, N));
  const float* M = M_ovr ? M_ovr : ((base_mode == IKV_MODE_QUERY) ? s->d_qenc : s->d_mem);

  const bool fast = c->cfg.kv_dtype == IKV_BF16;  // tensor-pipe key pass; fp32 pools take the plain FMA kernel
  const bool use_x = learn && !(mode & IKV_FLAG_NO_XATTN);
  const int n_x = use_x ? (r.xattn_pos ? r.n_xattn_pos : (r.q_end - r.q_start)) : 0;
  if (learn) TRY(ensure_xq(c, n_x > 0 ? n_x : 1));
  // at most RT_NXMAX query positions: folded cross attention, the whole head on tcgen05 (residual_tc.cuh)
  const bool tc = learn && c->resid_tc && n_x <= RT_NXMAX;
  const int nxp = tc ? (n_x > 0 ? (n_x + 15) / 16 * 16 : 16) : 0;
  if (part) TRY(launch_partition(c, r, n_x, scores, rule_out, st));
  const int LH = L * Hq, n_mpart = learn ? (LH + 31) / 32 : 0;  // mbar partial sums ride along with the fragments
  int n_part = (N + SCORE_TILE - 1) / SCORE_TILE;
  bool lm_done = false;  // the layer-major key pass has already produced rule_c (and the scores of a rule-only call)
  if (fast) {
    LmOut lo{scores, rule_out, (learn || !scatter) ? 0 : 1};
    TRY(dispatch_key_pass(c, M, learn, n_x > 0, n_mpart, &n_part, N, n_x, lo, &lm_done, st, lane));
  } else {
    if (n_mpart > 0) {
      if (D == 128) k_mem_prep<128, 1><<<n_mpart, 128, 0, st>>>(M, L, Hkv, 0.f, nullptr, 0, LH, c->mpart, nullptr);
      else k_mem_prep<64, 1><<<n_mpart, 128, 0, st>>>(M, L, Hkv, 0.f, nullptr, 0, LH, c->mpart, nullptr);
      LAUNCH_CHECK(c);
    }
    TRY(dispatch_logits(c, *s, M, N, learn, st));
    if (n_x > 0) {
      k_mean_key_list<float><<<n_x, D, 0, st>>>((const float*)c->cfg.k_pool, c->layer_stride, L, Hkv, D, c->xq_slot,
                                                c->d_nxq, c->kq);
      LAUNCH_CHECK(c);
    }
  }
  PostKeyParams pk;
  pk.partials = c->partials; pk.n_part = n_part; pk.lse = c->lse; pk.n_lse = LH;
  pk.mpart = c->mpart; pk.n_mpart = n_mpart; pk.LH = LH;
  pk.fold.mbar = c->mbar; pk.fold.wq_frag = c->wq_frag; pk.fold.w1_can = c->w1_can;
  pk.fold.bq_eff = c->bq_eff; pk.fold.b1_eff = c->b1_eff;
  pk.kq = c->kq; pk.n_xq = c->d_nxq; pk.nks = (int)(c->xq_cap / 16); pk.kc_frag = c->kc_frag; pk.vc_frag = c->vc_frag;
  pk.n_fold = 0; pk.n_kv = 0; pk.tc = tc ? 1 : 0; pk.nxp = nxp;
  pk.rt.mbar = c->mbar; pk.rt.wcan = c->rt_wcan; pk.rt.svec = c->rt_svec; pk.rt.b1_eff = c->b1_eff;
  if (lm_done) pk.n_lse = 0;   // no lse rows to reduce, no logits to read back
  pk.mbar_ready = (lm_done && learn) ? 1 : 0;
  if (lm_done && !learn) return IKV_OK;
  if (tc) {
    // launch 1: lse rows and the folded operands of the residual head (they need the mean keys of the query positions,
    // i.e. the finished key pass).  launch 2: rule_c (Eq. 3).  launch 3: k_tail_tc, the residual head (Eq. 4-6), one
    // persistent CTA per SM.
    pk.n_fold = D == 128 ? rt_fold_fc1_grid<128>() : rt_fold_fc1_grid<64>();
    pk.n_kv = n_x > 0 ? rt_fold_xattn_grid(nxp) : 0;
    {
      ProfScope prof(c, IKV_PROF_POST_KEY, st);
      CU(c, launch_pdl(D == 128 ? k_post_key<128, true> : k_post_key<64, true>,
                       dim3((pk.n_lse + 3) / 4 + pk.n_fold + pk.n_kv), dim3(256), 0, st, c->pdl_prune, pk, c->rw));
    }
    RuleParams rp;
    rp.logits = c->logits; rp.ldc = c->cap_tokens; rp.LH = LH; rp.lse = c->lse; rp.n_cand = c->d_ncand;
    rp.cand_pos = c->cand_pos; rp.rule_c = c->rule_c; rp.scores = scores; rp.scatter_scores = 0;
    rp.rule_out = rule_out; rp.n_rule = (N + 63) / 64; rp.l2_hints = c->dbg_l2;
    pk.n_fold = 0; pk.n_kv = 0;
    if (!lm_done) {
      ProfScope prof(c, IKV_PROF_RULE, st);
      CU(c, launch_pdl(D == 128 ? k_rule_fused<128> : k_rule_fused<64>, dim3(rp.n_rule), dim3(256), 0, st, c->pdl_prune,
                       rp, pk, c->rw));
    }
    TailParams tp;
    tp.rule_c = c->rule_c; tp.kbar = c->kbar; tp.n_cand = c->d_ncand; tp.cand_pos = c->cand_pos; tp.n_xq = c->d_nxq;
    tp.wcan = c->rt_wcan; tp.svec = c->rt_svec; tp.b1_eff = c->b1_eff; tp.nxp = nxp;
    tp.use_xattn = (use_x && n_x > 0) ? 1 : 0; tp.scores = scores;
    tp.early = lm_done ? 1 : 0;  // rule_c and kbar then come from the key pass, complete before k_post_key started
    const int smem = D == 128 ? rt_tail_smem<128>() : rt_tail_smem<64>();
    if (c->tail_smem_set != smem) {
      CU(c, cudaFuncSetAttribute(k_tail_tc<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, rt_tail_smem<128>()));
      CU(c, cudaFuncSetAttribute(k_tail_tc<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, rt_tail_smem<64>()));
      c->tail_smem_set = smem;
    }
    const int n_tiles = (N + RT_M - 1) / RT_M;
    ProfScope prof(c, IKV_PROF_RESIDUAL, st);
    CU(c, launch_pdl(D == 128 ? k_tail_tc<128> : k_tail_tc<64>, dim3(n_tiles < c->n_sm ? n_tiles : c->n_sm),
                     dim3(RT_TAIL_THREADS), smem, st, c->pdl_prune, tp, c->rw));
    return IKV_OK;
  }
  {
    // launch 1: lse rows.  launch 2: rule_c (Eq. 3) and, for a learnable call on the unfolded kernel, the folded residual
    // operands and the Kc / Vc fragments, whose latency-bound bodies hide under the rule blocks' stream of the logits.
    if (!lm_done) {
      ProfScope prof(c, IKV_PROF_POST_KEY, st);
      CU(c, launch_pdl(D == 128 ? k_post_key<128, false> : k_post_key<64, false>, dim3((LH + 3) / 4), dim3(128), 0, st,
                       c->pdl_prune, pk, c->rw));
    }
    pk.n_fold = learn ? (D == 128 ? resid_fold_grid<128>() : resid_fold_grid<64>()) : 0;
    pk.n_kv = (learn && n_x > 0) ? 4 * ((n_x + 15) / 16) : 0;
    RuleParams rp;
    rp.logits = c->logits; rp.ldc = c->cap_tokens; rp.LH = LH; rp.lse = c->lse; rp.n_cand = c->d_ncand;
    rp.cand_pos = c->cand_pos; rp.rule_c = c->rule_c; rp.scores = scores; rp.scatter_scores = (learn || !scatter) ? 0 : 1;
    rp.rule_out = rule_out; rp.n_rule = lm_done ? 0 : (N + 63) / 64; rp.l2_hints = c->dbg_l2;
    const int grid = rp.n_rule + pk.n_fold + pk.n_kv;
    ProfScope prof(c, IKV_PROF_RULE, st);
    CU(c, launch_pdl(D == 128 ? k_rule_fused<128> : k_rule_fused<64>, dim3(grid), dim3(256), 0, st, c->pdl_prune, rp, pk,
                     c->rw));
  }
  if (learn) {
    ResidMmaParams rp;
    rp.rule_c = c->rule_c; rp.kbar = c->kbar; rp.n_cand = c->d_ncand; rp.cand_pos = c->cand_pos; rp.n_xq = c->d_nxq;
    rp.wq_frag = c->wq_frag; rp.w1_can = c->w1_can; rp.kc_frag = c->kc_frag; rp.vc_frag = c->vc_frag;
    rp.bq_eff = c->bq_eff; rp.b1_eff = c->b1_eff; rp.nks = (int)(c->xq_cap / 16);
    rp.use_xattn = (use_x && n_x > 0) ? 1 : 0;
    rp.scores = scores;
    const int nblk = (N + R_CWARPS * 16 - 1) / (R_CWARPS * 16);
    if (!c->resid_attr_done) {
      CU(c, cudaFuncSetAttribute(k_residual_mma<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, resid_smem<128>()));
      CU(c, cudaFuncSetAttribute(k_residual_mma<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, resid_smem<64>()));
      c->resid_attr_done = true;
    }
    ProfScope prof(c, IKV_PROF_RESIDUAL, st);
    CU(c, launch_pdl(D == 128 ? k_residual_mma<128> : k_residual_mma<64>, dim3(nblk), dim3(R_THREADS),
                     D == 128 ? resid_smem<128>() : resid_smem<64>(), st, c->pdl_prune, rp, c->rw));
  }
  return IKV_OK;
}

template <int D, int G>
ikv_status launch_prefill(ikv_ctx* c, const PrefillParams& p, bf16* out, cudaStream_t st) {
  auto fn = k_prefill_mma<D, G>;
  if (!c->pf_attr_done[D == 128][G]) {
    CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, pf_smem<D>()));
    c->pf_attr_done[D == 128][G] = true;
  }
  fn<<<dim3(p.n_split, p.Hkv, (p.n_q + PF_BR - 1) / PF_BR), 64 * G, pf_smem<D>(), st>>>(p);
  LAUNCH_CHECK(c);
  k_prefill_merge<D><<<dim3(p.Hkv * G, p.n_q), D, 0, st>>>(p.part_o, p.part_ml, p.n_split, out);
  LAUNCH_CHECK(c);
  return IKV_OK;
}
template <int D, int G, bool TG, int MT = 1>
ikv_status launch_prefill_tc(ikv_ctx* c, const PrefillParams& p, bf16* out, cudaStream_t st) {
  auto fn = k_prefill_tc<D, G, TG, MT>;
  if (!c->pt_attr_done[MT - 1][TG][D == 128][G]) {
    CU(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, pt_smem<D, TG, MT>()));
    c->pt_attr_done[MT - 1][TG][D == 128][G] = true;
  }
  constexpr int BR = MT * 128 / G;
  PrefillParams pk = p;
  pk.out_direct = p.n_split == 1 ? out : nullptr;   // a single split writes the output itself
  fn<<<dim3(p.n_split, p.Hkv, (p.n_q + BR - 1) / BR), pt_threads<TG, MT>(), pt_smem<D, TG, MT>(), st>>>(pk, c->tm_k, c->tm_v);
  LAUNCH_CHECK(c);
  if (pk.out_direct) return IKV_OK;
  CU(c, launch_pdl(k_prefill_merge<D>, dim3(p.Hkv * G, p.n_q), dim3(D), 0, st, c->use_pdl, (const float*)p.part_o,
                   (const float2*)p.part_ml, p.n_split, out));
  return IKV_OK;
}
template <int D>
ikv_status dispatch_prefill(ikv_ctx* c, const PrefillParams& p, bf16* out, cudaStream_t st) {
  if (p.m_tiles == 2) {   // two 128-row tiles per CTA share each gathered K/V tile
    switch (c->G) {
      case 1: return launch_prefill_tc<D, 1, true, 2>(c, p, out, st);
      case 2: return launch_prefill_tc<D, 2, true, 2>(c, p, out, st);
      case 4: return launch_prefill_tc<D, 4, true, 2>(c, p, out, st);
      case 8: return launch_prefill_tc<D, 8, true, 2>(c, p, out, st);
    }
  }
  if ((c->prefill_tiled == 1 || c->prefill_tiled >= 4) && c->tm_ok) {   // tcgen05 where 128 / G rows x G heads make a 128-row tile; TMA gather4
    switch (c->G) {
      case 1: return launch_prefill_tc<D, 1, true>(c, p, out, st);
      case 2: return launch_prefill_tc<D, 2, true>(c, p, out, st);
      case 4: return launch_prefill_tc<D, 4, true>(c, p, out, st);
      case 8: return launch_prefill_tc<D, 8, true>(c, p, out, st);
    }
  }
  if (c->prefill_tiled == 1 || c->prefill_tiled >= 3) {   // the same with cp.async producers (no tensor map)
    switch (c->G) {
      case 1: return launch_prefill_tc<D, 1, false>(c, p, out, st);
      case 2: return launch_prefill_tc<D, 2, false>(c, p, out, st);
      case 4: return launch_prefill_tc<D, 4, false>(c, p, out, st);
      case 8: return launch_prefill_tc<D, 8, false>(c, p, out, st);
    }
  }
  switch (c->G) {
    case 1: return launch_prefill<D, 1>(c, p, out, st);
    case 2: return launch_prefill<D, 2>(c, p, out, st);
    case 4: return launch_prefill<D, 4>(c, p, out, st);
    case 5: return launch_prefill<D, 5>(c, p, out, st);
    case 8: return launch_prefill<D, 8>(c, p, out, st);
  }
  IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "GQA group size %d not supported (1,2,4,5,8)", c->G);
}

// The tiled kernel (prefill_mma.cuh).  The session's survivor list is made to cover a prefix [0, covered) with
// covered <= q_pos0 (rebuilt for [0, q_pos0) when it is stale, reaches into the chunk, or lags it by more than 4,096
// positions); the rest of the positions come from the slot map.  Chunks of more than 1,024 rows go in groups of 1,024
// (bounds the partials).
ikv_status prefill_tiled(ikv_ctx* c, int layer, const ikv_request& r, int q_pos0, int n_q, const bf16* q, bf16* out,
                         float sm_scale, cudaStream_t st) {
  Session* s = session_find(c, r.session_id);
  if (!s) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session %llu does not exist", (unsigned long long)r.session_id);
  const int Hq = c->cfg.n_q_heads, Hkv = c->cfg.n_kv_heads, D = c->cfg.head_dim;
  const bool stale = (r.flags & IKV_REQ_RESCAN) || s->map_ptr != r.slot_map || s->map_epoch != r.map_epoch ||
                     s->covered > q_pos0 || (q_pos0 - s->covered) > 4096;
  if (stale) {
    TRY(session_live_reserve(c, *s, q_pos0 > 0 ? q_pos0 : 1));
    k_build_live<<<1, 1024, 0, st>>>(r.slot_map, q_pos0, c->cfg.dead_slot, s->live_slots, s->d_n_live);
    LAUNCH_CHECK(c);
    s->covered = q_pos0;
    s->map_ptr = r.slot_map;
    s->map_epoch = r.map_epoch;
    s->live_ub = q_pos0;
    s->list_fresh = true;
  }
  PrefillParams p;
  p.k_layer = (const bf16*)c->cfg.k_pool + (int64_t)layer * c->layer_stride;
  p.v_layer = (const bf16*)c->cfg.v_pool + (int64_t)layer * c->layer_stride;
  p.Hkv = Hkv; p.dead = c->cfg.dead_slot; p.S = r.slot_map; p.live_slots = s->live_slots;
  p.row0 = (int64_t)layer * c->cfg.n_slots * Hkv;
  p.out_direct = nullptr;
  p.n_live = s->d_n_live; p.n_cached = s->live_ub; p.covered = s->covered;
  p.scale_log2 = sm_scale * 1.4426950408889634f;
  const bool tc = (c->prefill_tiled == 1 || c->prefill_tiled >= 3) && c->G != 5;
  // two M tiles per CTA from eight M tiles of rows on (configs[1], G = 4: 64 rows 41 us against 47 with two tiles, 256 rows
  // 96 against 85, 2,048 rows 681 against 545); IKV_TUNE_PREFILL_TILED = 5 forces them from two tiles on.  The row groups
  // are then sized to one full wave: (SMs / H_kv) blocks of two M tiles.
  const int bm = 128 / c->G;
  const bool two = tc && c->tm_ok && n_q >= 2 * bm && (c->prefill_tiled == 5 || (c->prefill_tiled == 1 && n_q >= 8 * bm));
  const int grp = two ? std::max(2 * bm, std::min(2048, (c->n_sm / Hkv) * 2 * bm)) : 1024;
  for (int g0 = 0; g0 < n_q; g0 += grp) {
    const int ng = std::min(grp, n_q - g0);
    p.q_pos0 = q_pos0 + g0; p.n_q = ng;
    p.q = q + (size_t)g0 * Hq * D;
    p.m_tiles = (two && ng > bm) ? 2 : 1;
    const int br = tc ? p.m_tiles * 128 / c->G : PF_BR;
    const int rbs = (ng + br - 1) / br;
    const int tiles = (p.n_cached + (p.q_pos0 + ng - p.covered) + PF_TOK - 1) / PF_TOK;   // upper bound
    int ns = c->n_sm / (Hkv * rbs);   // one wave: the kernel's registers leave room for one CTA per SM
    ns = std::max(1, std::min(std::min(ns, tiles), 32));
    p.n_split = ns;
    TRY(ensure_parts(c, (int64_t)ng * Hq * ns));
    p.part_o = c->part_o; p.part_ml = c->part_ml;
    TRY(D == 128 ? dispatch_prefill<128>(c, p, out + (size_t)g0 * Hq * D, st)
                 : dispatch_prefill<64>(c, p, out + (size_t)g0 * Hq * D, st));
  }
  return IKV_OK;
}

// NEXT-1 on tcgen05 (score_rows_tc.cuh): banks of 128 / G rows, two sweeps over the keys per bank.
template <int D>
ikv_status score_rows_tc(ikv_ctx* c, const ikv_request& r, const float* rows, int n_rows, const float* weights,
                         float* scores, cudaStream_t st) {
  const int N = r.seq_len, L = c->cfg.n_layers, Hkv = c->cfg.n_kv_heads, G = c->G;
  if (!session_find(c, r.session_id))
    IKV_FAIL(c, IKV_ERR_NO_SESSION, "session %llu does not exist", (unsigned long long)r.session_id);
  TRY(ensure_scratch(c, N));
  const int n_items = L * Hkv;
  if (!c->rows_bank) CU(c, cudaMalloc((void**)&c->rows_bank, (size_t)n_items * rb_item(D)));
  const int tiles = (N + RB_TOK - 1) / RB_TOK;
  const int grid = std::max(1, std::min(c->n_sm, (tiles + 1) / 2));
  const int n_pairs = (tiles + 2 * grid - 1) / (2 * grid);
  const int n_slots = n_pairs * grid * RB_CQ;   // (pair, CTA, column group)
  const size_t need = (size_t)n_items * n_slots * RB_ROWS;
  if (need > c->rows_partials_cap) {
    c->rows_partials_cap = 0;
    TRY(grow(c, &c->rows_partials, need));
    c->rows_partials_cap = need;
  }
  if (!c->rows_attr_done) {
    CU(c, cudaFuncSetAttribute(k_rows_pass<128, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(128)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<128, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(128)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<64, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(64)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<64, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(64)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<128, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(128)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<128, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(128)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<64, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(64)));
    CU(c, cudaFuncSetAttribute(k_rows_pass<64, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rb_smem(64)));
    c->rows_attr_done = true;
  }
  TRY(launch_partition(c, r, 0, scores, nullptr, st));
  const int64_t row_elems = (int64_t)L * c->cfg.n_q_heads * D;
  const int rpb = RB_ROWS / G;  // rows per bank
  RowsPassParams p;
  p.k_pool = (const bf16*)c->cfg.k_pool; p.layer_stride = c->layer_stride; p.L = L; p.Hkv = Hkv;
  p.bank = c->rows_bank; p.cand_slot = c->cand_slot; p.n_cand = c->d_ncand; p.partials = c->rows_partials;
  p.n_slots = n_slots; p.n_pairs = n_pairs; p.rule_c = c->rule_c;
  for (int r0 = 0; r0 < n_rows; r0 += rpb) {
    const int nr = std::min(rpb, n_rows - r0);
    RowsWeights wts;
    for (int cc = 0; cc < RB_ROWS; ++cc) wts.w[cc] = cc < nr * G ? weights[r0 + cc / G] : 0.f;
    p.n_cols = nr * G;
    p.accumulate = r0 > 0 ? 1 : 0;
    k_rows_prep<D><<<n_items, 256, 0, st>>>(rows + r0 * row_elems, nr, L, Hkv, G, wts, c->rows_bank);
    const bool tg = c->tm_ok && c->rows_tc != 3;   // keys by TMA gather4 through the pool's tensor map
    if (tg) k_rows_pass<D, 1, true><<<grid, RB_THREADS, rb_smem(D), st>>>(p, c->tm_k);
    else k_rows_pass<D, 1, false><<<grid, RB_THREADS, rb_smem(D), st>>>(p, c->tm_k);
    k_rows_lse<D><<<n_items, 1024, 0, st>>>(c->rows_partials, n_slots, c->rows_bank);
    if (tg) k_rows_pass<D, 2, true><<<grid, RB_THREADS, rb_smem(D), st>>>(p, c->tm_k);
    else k_rows_pass<D, 2, false><<<grid, RB_THREADS, rb_smem(D), st>>>(p, c->tm_k);
    LAUNCH_CHECK(c);
  }
  k_axpy_scatter<<<64, 256, 0, st>>>(c->rule_c, c->cand_pos, c->d_ncand, 1.0f, 1, scores);
  LAUNCH_CHECK(c);
  return IKV_OK;
}

// Fills the kernel parameters of one request and updates the session's decode bookkeeping.
ikv_status select_prepare(ikv_ctx* c, const ikv_request& r, const float* scores, int32_t* freed, int32_t* n_freed,
                          int32_t* n_kept, SelParams* out) {
  Session* s = session_find(c, r.session_id);
  if (!s) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session %llu does not exist", (unsigned long long)r.session_id);
  const int N = r.seq_len;
  TRY(ensure_scratch(c, N > 0 ? N : 1));
  TRY(session_live_reserve(c, *s, N > 0 ? N : 1));
  SelParams p;
  p.S = r.slot_map; p.valid = r.valid_mask; p.scores = scores;
  p.N = N; p.pi = r.prefix_len; p.qs = r.q_start; p.qe = r.q_end; p.C = r.budget; p.radix = r.radix_protected_len;
  p.dead = c->cfg.dead_slot;
  p.freed = freed; p.n_freed = n_freed; p.n_kept = n_kept;
  p.live_slots = s->live_slots; p.n_live = s->d_n_live;
  p.kept_bits = c->kept_bits; p.firstpos = c->firstpos; p.keepflag = c->keepflag; p.tmp_slot = c->tmp_slot;
  *out = p;
  s->covered = N;
  s->map_ptr = r.slot_map;
  s->map_epoch = r.map_epoch;
  s->list_fresh = true;
  s->live_ub = N;
  if (N > r.budget) {
    const int forced_ub = r.prefix_len + (r.q_end - r.q_start);
    s->live_ub = (forced_ub > r.budget ? forced_ub : r.budget);
    if (s->live_ub > N) s->live_ub = N;
  }
  return IKV_OK;
}

// One launch for up to SEL_MAX_REQ requests (one cluster each); longer maps take the single-CTA kernel one by one.
ikv_status select_launch(ikv_ctx* c, const SelBatch& b, int n, int max_n, cudaStream_t st) {
  if (n == 0) return IKV_OK;
  auto fn = max_n <= CL_CTAS * 1024 * 4 ? k_select_evict_cl<4>
            : max_n <= CL_CTAS * 1024 * 8 ? k_select_evict_cl<8> : k_select_evict_cl<16>;
  ProfScope prof(c, IKV_PROF_SELECT, st);
  CU(c, launch_pdl(fn, dim3(n * CL_CTAS), dim3(1024), 0, st, c->pdl_prune, b));
  return IKV_OK;
}

}  // namespace

// ======================================================================================================
extern "C" {

#ifdef IKV_TRACE
ikv_status ikv_debug_trace(long long* out) {
  cudaDeviceSynchronize();
  return cudaMemcpyFromSymbol(out, g_rt_trace, sizeof(long long) * 128) == cudaSuccess ? IKV_OK : IKV_ERR_CUDA;
}
ikv_status ikv_debug_lm(long long* out) {
  cudaDeviceSynchronize();
  return cudaMemcpyFromSymbol(out, g_lm_wait, sizeof(long long) * 640) == cudaSuccess ? IKV_OK : IKV_ERR_CUDA;
}
#endif

ikv_status ikv_test_late_writer(void* dst, const void* src, int64_t bytes, int32_t delay_us, void* stream) {
  if (!dst || !src || bytes <= 0 || (bytes & 15)) return IKV_ERR_INVALID_ARG;
  k_late_writer<<<1, 256, 0, (cudaStream_t)stream>>>((uint4*)dst, (const uint4*)src, bytes / 16, (int64_t)delay_us * 1000);
  return cudaGetLastError() == cudaSuccess ? IKV_OK : IKV_ERR_CUDA;
}

const char* ikv_version(void) { return "ikv 0.1 (sm_100a)"; }

static thread_local std::string g_create_err;  // ikv_create has no context to hang its message on

const char* ikv_last_error(const ikv_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

ikv_status ikv_create(const ikv_config* cfg, ikv_ctx** out) {
  if (!cfg || !out) return IKV_ERR_INVALID_ARG;
  *out = nullptr;
  ikv_ctx* c = new ikv_ctx();
  c->cfg = *cfg;
  auto fail = [&](ikv_status code, const char* msg) {
    g_create_err = std::string("ikv_create: ") + msg;
    delete c;
    return code;
  };
  if (cfg->n_layers <= 0 || cfg->n_q_heads <= 0 || cfg->n_kv_heads <= 0 || cfg->n_q_heads % cfg->n_kv_heads != 0)
    return fail(IKV_ERR_INVALID_ARG, "bad layer / head counts");
  if (cfg->head_dim != 64 && cfg->head_dim != 128) return fail(IKV_ERR_UNSUPPORTED, "head_dim must be 64 or 128");
  if (cfg->kv_dtype != IKV_BF16 && cfg->kv_dtype != IKV_F32)
    return fail(IKV_ERR_UNSUPPORTED, "kv_dtype must be IKV_BF16 or IKV_F32 (PAPER.md:263)");
  if (cfg->page_size <= 0 || cfg->n_slots <= 0 || cfg->n_slots > INT32_MAX || !cfg->k_pool || !cfg->v_pool)
    return fail(IKV_ERR_INVALID_ARG, "bad pool description");
  if (cfg->dead_slot < 0 || cfg->dead_slot >= cfg->n_slots) return fail(IKV_ERR_INVALID_ARG, "dead_slot out of range");
  if (cfg->max_sessions <= 0) return fail(IKV_ERR_INVALID_ARG, "max_sessions must be > 0");
  if (!(cfg->lambda >= 0.f)) return fail(IKV_ERR_INVALID_ARG, "lambda must be >= 0");
  c->G = cfg->n_q_heads / cfg->n_kv_heads;
  if (c->G != 1 && c->G != 2 && c->G != 4 && c->G != 5 && c->G != 8)
    return fail(IKV_ERR_UNSUPPORTED, "GQA group size must be one of 1,2,4,5,8");
  c->layer_stride = cfg->n_slots * cfg->n_kv_heads * cfg->head_dim;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return fail(IKV_ERR_CUDA, "no CUDA device");
  cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&c->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  c->use_pdl = !(cfg->flags & IKV_CFG_NO_PDL);
  c->pdl_prune = c->use_pdl && !(cfg->flags & IKV_CFG_NO_PDL_PRUNE);
  const int row = cfg->n_kv_heads * cfg->head_dim;
  if (cfg->kv_dtype == IKV_BF16)
    k_init_dead<bf16><<<cfg->n_layers, 256>>>((bf16*)cfg->k_pool, (bf16*)cfg->v_pool, c->layer_stride, cfg->n_layers,
                                              row, cfg->dead_slot);
  else
    k_init_dead<float><<<cfg->n_layers, 256>>>((float*)cfg->k_pool, (float*)cfg->v_pool, c->layer_stride,
                                               cfg->n_layers, row, cfg->dead_slot);
  bool ok = cudaGetLastError() == cudaSuccess;
  const size_t words = (size_t)(cfg->n_slots + 31) / 32;
  ok = ok && cudaMalloc((void**)&c->kept_bits, words * 4) == cudaSuccess;
  ok = ok && cudaMemset(c->kept_bits, 0, words * 4) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&c->firstpos, (size_t)cfg->n_slots * 4) == cudaSuccess;
  if (ok) {
    k_fill_i32<<<256, 256>>>(c->firstpos, cfg->n_slots, INT_MAX);
    ok = cudaGetLastError() == cudaSuccess;
  }
  ok = ok && scratch_alloc_fixed(*c, *cfg);
  ok = ok && cudaDeviceSynchronize() == cudaSuccess;
  if (!ok) {
    g_create_err = std::string("ikv_create: CUDA initialisation failed: ") + cudaGetErrorString(cudaGetLastError());
    ikv_destroy(c);
    return IKV_ERR_CUDA;
  }
  {  // ikv_decode_attn_static: the static array's device address, once per context, with its device current
    void* sp = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&sp, g_static_scratch);
    if (e == cudaSuccess) c->static_scratch = (unsigned char*)sp;
    else c->static_scratch_err = cudaGetErrorString(e);
    cudaGetLastError();
  }
  if (cfg->kv_dtype == IKV_BF16 && (cfg->head_dim == 64 || cfg->head_dim == 128)) {
    // tensor maps of the pools for the TMA gather4 producers of k_prefill_tc; without them the cp.async producers run
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    EncodeFn enc = nullptr;
    cudaDriverEntryPointQueryResult qr;
    const int64_t rows = (int64_t)cfg->n_layers * cfg->n_slots * cfg->n_kv_heads;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &qr) == cudaSuccess && enc &&
        qr == cudaDriverEntryPointSuccess && rows < INT_MAX && ((uintptr_t)cfg->k_pool & 15) == 0 &&
        ((uintptr_t)cfg->v_pool & 15) == 0) {
      const cuuint64_t gdim[2] = {(cuuint64_t)cfg->head_dim, (cuuint64_t)rows}, gstr[1] = {(cuuint64_t)cfg->head_dim * 2};
      const cuuint32_t box[2] = {64, 1}, estr[2] = {1, 1};
      const CUresult rk = enc(&c->tm_k, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, cfg->k_pool, gdim, gstr, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      const CUresult rv = enc(&c->tm_v, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, cfg->v_pool, gdim, gstr, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      c->tm_ok = rk == CUDA_SUCCESS && rv == CUDA_SUCCESS;
    }
    cudaGetLastError();
  }
  *out = c;
  return IKV_OK;
}

ikv_status ikv_destroy(ikv_ctx* c) {
  if (!c) return IKV_ERR_INVALID_ARG;
  cudaDeviceSynchronize();
  for (auto& kv : c->sessions) session_free(kv.second);
  scratch_free(*c);
  for (int k = 1; k < IKV_MAX_LANES; ++k) scratch_free(c->lane_set[k]);
  for (int k = 0; k < IKV_MAX_LANES; ++k) {
    if (c->lane_stream[k]) cudaStreamDestroy(c->lane_stream[k]);
    for (cudaEvent_t e : c->lane_ev[k]) if (e) cudaEventDestroy(e);
  }
  if (c->fork_ev) cudaEventDestroy(c->fork_ev);
  void* bufs[] = {c->rows_bank, c->rows_partials, c->ts_ring, c->kept_bits, c->firstpos, c->part_o, c->part_ml, c->st_out, c->st_scores,
                  c->st_qrows, c->resid_blob};
  for (void* b : bufs) cudaFree(b);
  if (c->st_host) cudaFreeHost(c->st_host);
  for (int w = 0; w < IKV_PROF_SLOTS; ++w)
    for (auto& pr : c->prof_ev[w]) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
  const cudaError_t e = cudaGetLastError();
  delete c;
  return e == cudaSuccess ? IKV_OK : IKV_ERR_CUDA;
}

ikv_status ikv_tune(ikv_ctx* c, int32_t knob, int32_t value) {
  if (!c) return IKV_ERR_INVALID_ARG;
  switch (knob) {
    case IKV_TUNE_L2_HINTS: c->dbg_l2 = value; return IKV_OK;
    case IKV_TUNE_RESID_TC: c->resid_tc = value; return IKV_OK;
    case IKV_TUNE_LAYER_MAJOR: c->use_lm = value; return IKV_OK;
    case IKV_TUNE_ROWS_TC: c->rows_tc = value; return IKV_OK;
    case IKV_TUNE_PREFILL_TILED: c->prefill_tiled = value; return IKV_OK;
    case IKV_TUNE_BATCH_LANES:
      c->n_lanes = value < 1 ? 1 : (value > IKV_MAX_LANES ? IKV_MAX_LANES : value);
      return IKV_OK;
  }
  IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_tune: unknown knob %d", knob);
}

ikv_status ikv_profile_enable(ikv_ctx* c, int32_t on) {
  if (!c) return IKV_ERR_INVALID_ARG;
  c->prof_on = on < 0 ? 0 : (on > 2 ? 2 : on);
  if (c->prof_on == 1) {
    const size_t bytes = (size_t)ikv_ctx::TS_SLOTS * 16;
    if (!c->ts_ring) CU(c, cudaMalloc((void**)&c->ts_ring, bytes));
    std::vector<unsigned long long> init(2 * ikv_ctx::TS_SLOTS);
    for (int i = 0; i < ikv_ctx::TS_SLOTS; ++i) { init[2 * i] = ~0ull; init[2 * i + 1] = 0ull; }
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(c->ts_ring, init.data(), bytes, cudaMemcpyHostToDevice));
    CU(c, cudaDeviceSynchronize());
    c->ts_used = 0;
  }
  return IKV_OK;
}

ikv_status ikv_profile_read(ikv_ctx* c, float* out_ms, int32_t* out_n) {
  if (!c || !out_ms || !out_n) return IKV_ERR_INVALID_ARG;
  CU(c, cudaDeviceSynchronize());
  for (int w = 0; w < IKV_PROF_SLOTS; ++w) {
    float tot = 0.f;
    for (auto& pr : c->prof_ev[w]) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, pr.first, pr.second);
      tot += ms;
      c->ev_pool.push_back(pr.first);
      c->ev_pool.push_back(pr.second);
    }
    out_ms[w] = tot;
    out_n[w] = (int32_t)c->prof_ev[w].size();
    c->prof_ev[w].clear();
  }
  if (c->ts_ring && c->ts_used > 0) {  // stamps of the layer-major key pass (level 1)
    std::vector<unsigned long long> h(2 * c->ts_used);
    CU(c, cudaMemcpy(h.data(), c->ts_ring, h.size() * 8, cudaMemcpyDeviceToHost));
    double tot = 0.0;
    for (int i = 0; i < c->ts_used; ++i) tot += (double)(h[2 * i + 1] - h[2 * i]) * 1e-6;
    out_ms[IKV_PROF_KEY_PASS] += (float)tot;
    out_n[IKV_PROF_KEY_PASS] += c->ts_used;
    for (int i = 0; i < c->ts_used; ++i) { h[2 * i] = ~0ull; h[2 * i + 1] = 0ull; }
    CU(c, cudaMemcpy(c->ts_ring, h.data(), h.size() * 8, cudaMemcpyHostToDevice));
    CU(c, cudaDeviceSynchronize());
    c->ts_used = 0;
  }
  return IKV_OK;
}

ikv_status ikv_reserve(ikv_ctx* c, int64_t max_tokens, int32_t max_requests) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (max_tokens <= 0 || max_requests <= 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_reserve: sizes must be > 0");
  TRY(ensure_scratch(c, max_tokens));
  TRY(ensure_xq(c, 1024));
  TRY(ensure_parts(c, (int64_t)max_requests * c->cfg.n_q_heads * 4 * c->n_sm));
  TRY(ensure_staging(c, max_tokens, 0));
  CU(c, cudaDeviceSynchronize());
  return IKV_OK;
}

ikv_status ikv_session_open(ikv_ctx* c, uint64_t id) {
  if (!c) return IKV_ERR_INVALID_ARG;
  Session* s;
  return session_create(c, id, &s, (cudaStream_t)0, true);
}

ikv_status ikv_session_fork(ikv_ctx* c, uint64_t parent, uint64_t child, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (parent == child) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "fork onto itself");
  if (!session_find(c, parent)) IKV_FAIL(c, IKV_ERR_NO_SESSION, "parent session does not exist");
  Session* ch;
  TRY(session_create(c, child, &ch, (cudaStream_t)stream, false));
  Session* p = session_find(c, parent);  // re-find: the map may have rehashed
  if (!p) {  // max_sessions == 1: creating the child evicted the parent
    auto it = c->sessions.find(child);
    if (it != c->sessions.end()) { session_free(it->second); c->sessions.erase(it); }
    IKV_FAIL(c, IKV_ERR_CAPACITY, "ikv_session_fork: max_sessions = %d leaves no room for parent and child",
             c->cfg.max_sessions);
  }
  const size_t n = (size_t)c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim * sizeof(float);
  CU(c, cudaMemcpyAsync(ch->d_mem, p->d_mem, n, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  CU(c, cudaMemcpyAsync(ch->d_qenc, p->d_qenc, n, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  ch->has_update = p->has_update;
  return IKV_OK;
}

ikv_status ikv_session_close(ikv_ctx* c, uint64_t id) {
  if (!c) return IKV_ERR_INVALID_ARG;
  auto it = c->sessions.find(id);
  if (it == c->sessions.end()) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session does not exist");
  CU(c, cudaDeviceSynchronize());
  session_free(it->second);
  c->sessions.erase(it);
  return IKV_OK;
}

ikv_status ikv_session_get_memory(ikv_ctx* c, uint64_t id, float* host_out) {
  if (!c || !host_out) return IKV_ERR_INVALID_ARG;
  Session* s = session_find(c, id);
  if (!s) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session does not exist");
  const size_t n = (size_t)c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim * sizeof(float);
  CU(c, cudaDeviceSynchronize());
  CU(c, cudaMemcpy(host_out, s->d_mem, n, cudaMemcpyDeviceToHost));
  return IKV_OK;
}

ikv_status ikv_session_set_memory(ikv_ctx* c, uint64_t id, const float* host_in) {
  if (!c || !host_in) return IKV_ERR_INVALID_ARG;
  Session* s = session_find(c, id);
  if (!s) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session does not exist");
  const size_t n = (size_t)c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim * sizeof(float);
  CU(c, cudaDeviceSynchronize());
  CU(c, cudaMemcpy(s->d_mem, host_in, n, cudaMemcpyHostToDevice));
  CU(c, cudaDeviceSynchronize());  // pageable copies may still be in flight when cudaMemcpy returns
  return IKV_OK;
}

ikv_status ikv_residual_load(ikv_ctx* c, const ikv_residual_weights* w) {
  if (!c || !w) return IKV_ERR_INVALID_ARG;
  if (!w->wq || !w->bq || !w->wk || !w->bk || !w->wv || !w->bv || !w->fc1_w || !w->fc1_b || !w->fc2_w || !w->fc2_b)
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_residual_load: NULL weight array");
  const int D = c->cfg.head_dim, P = 3 * D + 1, IN = P + R_DC;
  // blob layout (floats): wq[128][P] bq[128] wk_t[D][128] bk[128] wv_t[D][128] bv[128] fc1_w[256][IN] fc1_b[256]
  //                       fc2_w[256] fc2_b[1] w1c_frag[4][8][8][32] (uint4: B fragments of fc1's c columns)
  const size_t n_frag = (size_t)4 * 8 * 8 * 32;
  const size_t sizes[11] = {(size_t)R_DC * P, R_DC, (size_t)D * R_DC, R_DC, (size_t)D * R_DC, R_DC,
                            (size_t)R_HID * IN, R_HID, R_HID, 1, n_frag * 4};
  size_t off[12];
  off[0] = 0;
  for (int i = 0; i < 11; ++i) off[i + 1] = off[i] + ((sizes[i] + 3) / 4) * 4;  // keep 16-byte alignment
  std::vector<float> h(off[11], 0.f);
  auto transpose = [&](const float* src, int out_n, int in_n, float* dst) {
    for (int o = 0; o < out_n; ++o)
      for (int i = 0; i < in_n; ++i) dst[(size_t)i * out_n + o] = src[(size_t)o * in_n + i];
  };
  memcpy(&h[off[0]], w->wq, sizes[0] * 4);
  memcpy(&h[off[1]], w->bq, R_DC * 4);
  transpose(w->wk, R_DC, D, &h[off[2]]);
  memcpy(&h[off[3]], w->bk, R_DC * 4);
  transpose(w->wv, R_DC, D, &h[off[4]]);
  memcpy(&h[off[5]], w->bv, R_DC * 4);
  memcpy(&h[off[6]], w->fc1_w, sizes[6] * 4);
  memcpy(&h[off[7]], w->fc1_b, R_HID * 4);
  memcpy(&h[off[8]], w->fc2_w, R_HID * 4);
  h[off[9]] = w->fc2_b[0];
  {  // static B fragments (bf16 hi | lo) of fc1's c columns; k order is natural (the A side comes from accumulators)
    auto bf16_rn = [](float x) -> uint32_t {
      uint32_t u;
      memcpy(&u, &x, 4);
      if ((u & 0x7fffffffu) > 0x7f800000u) return (u >> 16) | 0x40u;  // NaN stays NaN
      return (u + 0x7fffu + ((u >> 16) & 1u)) >> 16;
    };
    auto up = [](uint32_t b) { uint32_t u = b << 16; float f; memcpy(&f, &u, 4); return f; };
    uint32_t* fr = reinterpret_cast<uint32_t*>(&h[off[10]]);
    for (int ch = 0; ch < 4; ++ch)
      for (int s8 = 0; s8 < 8; ++s8)
        for (int t = 0; t < 8; ++t)
          for (int lane = 0; lane < 32; ++lane) {
            const int r = lane >> 2, q = lane & 3;
            const int n = ch * 64 + t * 8 + r;
            const int ks[4] = {2 * q, 2 * q + 1, 2 * q + 8, 2 * q + 9};
            uint32_t hi[4], lo[4];
            for (int e = 0; e < 4; ++e) {
              const float v = w->fc1_w[(size_t)n * IN + P + s8 * 16 + ks[e]];
              hi[e] = bf16_rn(v);
              lo[e] = bf16_rn(v - up(hi[e]));
            }
            uint32_t* o = fr + ((((size_t)ch * 8 + s8) * 8 + t) * 32 + lane) * 4;
            o[0] = hi[0] | (hi[1] << 16); o[1] = hi[2] | (hi[3] << 16);
            o[2] = lo[0] | (lo[1] << 16); o[3] = lo[2] | (lo[3] << 16);
          }
  }
  {  // fc1's c columns as tcgen05 B-operand chunks (k >= D of w1_can; the kbar chunks are folded per call)
    auto bf16_rn = [](float x) -> uint32_t {
      uint32_t u;
      memcpy(&u, &x, 4);
      if ((u & 0x7fffffffu) > 0x7f800000u) return (u >> 16) | 0x40u;
      return (u + 0x7fffu + ((u >> 16) & 1u)) >> 16;
    };
    auto up = [](uint32_t b) { uint32_t u = b << 16; float f; memcpy(&f, &u, 4); return f; };
    const size_t bytes = (size_t)2 * (D / 64 + 2) * W1C_CHUNK;
    std::vector<unsigned char> can(bytes, 0);
    for (int n = 0; n < R_HID; ++n)
      for (int kc = 0; kc < R_DC; ++kc) {
        const float v = w->fc1_w[(size_t)n * IN + P + kc];
        const uint32_t hi = bf16_rn(v), lo = bf16_rn(v - up(hi));
        const size_t o = (D == 128) ? w1_can_offset<128>(n, D + kc) : w1_can_offset<64>(n, D + kc);
        const uint16_t h16 = (uint16_t)hi, l16 = (uint16_t)lo;
        memcpy(&can[o], &h16, 2);
        memcpy(&can[o + W1C_PART], &l16, 2);
      }
    CU(c, cudaDeviceSynchronize());
    CU(c, cudaMemcpy(c->w1_can, can.data(), bytes, cudaMemcpyHostToDevice));
  }
  CU(c, cudaDeviceSynchronize());
  if (!c->resid_blob) CU(c, cudaMalloc((void**)&c->resid_blob, h.size() * 4));
  CU(c, cudaMemcpy(c->resid_blob, h.data(), h.size() * 4, cudaMemcpyHostToDevice));
  CU(c, cudaDeviceSynchronize());  // pageable copies may still be in flight when cudaMemcpy returns
  float* b = c->resid_blob;
  c->rw.wq = b + off[0]; c->rw.bq = b + off[1]; c->rw.wk_t = b + off[2]; c->rw.bk = b + off[3];
  c->rw.wv_t = b + off[4]; c->rw.bv = b + off[5]; c->rw.fc1_w = b + off[6]; c->rw.fc1_b = b + off[7];
  c->rw.fc2_w = b + off[8]; c->rw.fc2_b = b + off[9];
  c->rw.w1c_frag = reinterpret_cast<const uint4*>(b + off[10]);
  float a = w->alpha;  // "clipped at inference"
  c->rw.alpha = a > 5.f ? 5.f : (a < -5.f ? -5.f : a);
  c->has_resid = true;
  return IKV_OK;
}

ikv_status ikv_memory_update(ikv_ctx* c, uint64_t id, const void* q_rows, int32_t n, int32_t q_dtype, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (!q_rows || n <= 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_memory_update: need n > 0 query rows");
  if (q_dtype != IKV_F32 && q_dtype != IKV_BF16) IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "q_dtype must be IKV_F32 or IKV_BF16");
  Session* s = session_find(c, id);
  if (!s) TRY(session_create(c, id, &s, (cudaStream_t)stream, false));
  const int L = c->cfg.n_layers, Hq = c->cfg.n_q_heads, D = c->cfg.head_dim;
  const float decay = expf(-c->cfg.lambda);
  const int64_t rs = (int64_t)L * Hq * D;
  ProfScope prof(c, IKV_PROF_MEM_UPDATE, (cudaStream_t)stream);
  if (q_dtype == IKV_F32)
    k_memory_update<float><<<L * Hq, D, 0, (cudaStream_t)stream>>>(s->d_mem, s->d_qenc, (const float*)q_rows, n, rs, D,
                                                                   decay);
  else
    k_memory_update<bf16><<<L * Hq, D, 0, (cudaStream_t)stream>>>(s->d_mem, s->d_qenc, (const bf16*)q_rows, n, rs, D,
                                                                  decay);
  LAUNCH_CHECK(c);
  s->has_update = true;
  return IKV_OK;
}

ikv_status ikv_score(ikv_ctx* c, const ikv_request* reqs, int32_t n_req, int32_t mode, float* scores, float* rule_out,
                     void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (n_req < 0 || (n_req > 0 && (!reqs || !scores))) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_score: NULL argument");
  const int bm = mode & 0xff;
  if (bm != IKV_MODE_MEMORY && bm != IKV_MODE_LEARNABLE && bm != IKV_MODE_QUERY)
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "unknown scorer mode %d", bm);
  for (int r = 0; r < n_req; ++r) TRY(check_request(c, reqs[r]));
  cudaStream_t st = (cudaStream_t)stream;
  int n_busy = 0;
  for (int r = 0; r < n_req; ++r) n_busy += reqs[r].seq_len > 0;
  const int K = n_busy < c->n_lanes ? n_busy : c->n_lanes;
  if (K < 2 || c->cfg.kv_dtype != IKV_BF16) {
    int64_t off = 0;
    for (int r = 0; r < n_req; ++r) {
      TRY(score_one(c, reqs[r], mode, scores + off, rule_out ? rule_out + off : nullptr, st));
      off += reqs[r].seq_len;
    }
    return IKV_OK;
  }
  // Batch: the latency chain of one request (partition, fragments, fold, residual head: ~60 us of small kernels) runs
  // beside the key passes of the others.  Lane k = stream + scratch set; request r takes lane r % K; the key passes
  // stay on the caller's stream in request order (two layer-major passes must never be resident together: each
  // waits for all of its own CTAs).
  TRY(lanes_prepare(c, K));
  const bool learn = (mode & 0xff) == IKV_MODE_LEARNABLE && !(mode & IKV_FLAG_NO_RESIDUAL);
  {  // every allocation before the first launch: cudaMalloc would serialise the lanes
    int64_t need[IKV_MAX_LANES] = {}, need_x[IKV_MAX_LANES] = {};
    int k = 0;
    for (int r = 0; r < n_req; ++r) {
      if (reqs[r].seq_len == 0) continue;
      need[k] = std::max<int64_t>(need[k], reqs[r].seq_len);
      const int n_x = reqs[r].xattn_pos ? reqs[r].n_xattn_pos : (reqs[r].q_end - reqs[r].q_start);
      need_x[k] = std::max<int64_t>(need_x[k], n_x > 0 ? n_x : 1);
      k = (k + 1) % K;
    }
    for (k = 0; k < K; ++k) {
      LaneSwap sw(c, k);
      TRY(ensure_scratch(c, need[k]));
      if (learn) TRY(ensure_xq(c, need_x[k]));
    }
  }
  CU(c, cudaEventRecord(c->fork_ev, st));
  for (int k = 0; k < K; ++k) CU(c, cudaStreamWaitEvent(c->lane_stream[k], c->fork_ev, 0));
  ikv_status rc = IKV_OK;
  int64_t off = 0;
  for (int r = 0, k = 0; r < n_req && rc == IKV_OK; ++r) {
    if (reqs[r].seq_len > 0) {
      LaneSwap sw(c, k);
      const KeyLane lane{st, c->lane_ev[k][0], c->lane_ev[k][1]};
      rc = score_one(c, reqs[r], mode, scores + off, rule_out ? rule_out + off : nullptr, c->lane_stream[k], nullptr,
                     true, true, &lane);
      k = (k + 1) % K;
    }
    off += reqs[r].seq_len;
  }
  for (int k = 0; k < K; ++k) {  // join, also after a failure: the caller's stream must not run ahead of the lanes
    if (cudaEventRecord(c->lane_ev[k][2], c->lane_stream[k]) != cudaSuccess ||
        cudaStreamWaitEvent(st, c->lane_ev[k][2], 0) != cudaSuccess) {
      if (rc == IKV_OK) { c->err = "ikv_score: joining the lanes failed"; rc = IKV_ERR_CUDA; }
    }
  }
  return rc;
}

ikv_status ikv_score_rows(ikv_ctx* c, const ikv_request* reqs, int32_t n_req, const float* rows, int32_t n_rows,
                          const float* weights, float* scores, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (n_req < 0 || n_rows <= 0 || !rows || !weights || (n_req > 0 && (!reqs || !scores)))
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_score_rows: bad argument");
  for (int r = 0; r < n_req; ++r) TRY(check_request(c, reqs[r]));
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t row_elems = (int64_t)c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim;
  // banks on tcgen05 from the row count at which two sweeps over the keys beat single-row passes: four rows with the TMA
  // gather4 warps (1.13 ms against 0.38 ms per pass on configs[1]), six with cp.async; rows_tc >= 2 forces it from two
  const int tc_from = (c->tm_ok && c->rows_tc != 3) ? 4 : 6;
  if (c->rows_tc && c->cfg.kv_dtype == IKV_BF16 && (n_rows >= tc_from || (c->rows_tc >= 2 && n_rows >= 2))) {
    int64_t off = 0;
    for (int r = 0; r < n_req; ++r) {
      if (reqs[r].seq_len > 0)
        TRY(c->cfg.head_dim == 128 ? score_rows_tc<128>(c, reqs[r], rows, n_rows, weights, scores + off, st)
                                   : score_rows_tc<64>(c, reqs[r], rows, n_rows, weights, scores + off, st));
      off += reqs[r].seq_len;
    }
    return IKV_OK;
  }
  int64_t off = 0;
  for (int r = 0; r < n_req; ++r) {
    for (int k = 0; k < n_rows; ++k) {
      // one pass of the Eq. 3 scorer per row (row k in place of M_t), rule_c left in scratch, then the weighted sum
      TRY(score_one(c, reqs[r], IKV_MODE_MEMORY, scores + off, nullptr, st, rows + k * row_elems, k == 0, false));
      if (reqs[r].seq_len > 0)
        CU(c, launch_pdl(k_axpy_scatter, dim3(64), dim3(256), 0, st, c->pdl_prune, (const float*)c->rule_c,
                         (const int32_t*)c->cand_pos, (const int32_t*)c->d_ncand, weights[k], k == 0 ? 1 : 0, scores + off));
    }
    off += reqs[r].seq_len;
  }
  return IKV_OK;
}

ikv_status ikv_score_baseline(ikv_ctx* c, const ikv_request* reqs, int32_t n_req, const ikv_baseline* b, float* scores,
                              void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (!b || n_req < 0 || (n_req > 0 && (!reqs || !scores))) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_score_baseline: NULL argument");
  cudaStream_t st = (cudaStream_t)stream;
  if (b->kind == IKV_BASE_STREAMING) {
    if (b->n_sink < 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "n_sink < 0");
    int64_t off = 0;
    for (int r = 0; r < n_req; ++r) {
      TRY(check_request(c, reqs[r]));
      const ikv_request& q = reqs[r];
      const int N = q.seq_len;
      if (N > 0) {
        TRY(ensure_scratch(c, N));
        // a1 partition: fillers and the candidate list (no keys are read by this scorer)
        if (N <= CL_MAX_N) {
          auto fn = N <= CL_CTAS * 1024 * 4 ? k_partition_cl<4> : N <= CL_CTAS * 1024 * 8 ? k_partition_cl<8> : k_partition_cl<16>;
          CU(c, launch_pdl(fn, dim3(CL_CTAS), dim3(1024), 0, st, false, (const int32_t*)q.slot_map, N, c->cfg.dead_slot,
                           q.prefix_len, q.q_start, q.q_end, scores + off, (float*)nullptr, c->cand_pos, c->cand_slot,
                           c->d_ncand, (const int32_t*)nullptr, 0, (int32_t*)nullptr, (int32_t*)nullptr));
        } else {
          k_partition<<<1, 1024, 0, st>>>(q.slot_map, N, c->cfg.dead_slot, q.prefix_len, q.q_start, q.q_end, scores + off,
                                          nullptr, c->cand_pos, c->cand_slot, c->d_ncand);
        }
        k_streaming_scores<<<64, 256, 0, st>>>(c->cand_pos, c->d_ncand, b->n_sink, scores + off);
        LAUNCH_CHECK(c);
      }
      off += N;
    }
    return IKV_OK;
  }
  if (b->kind != IKV_BASE_SNAPKV && b->kind != IKV_BASE_H2O) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "unknown baseline %d", b->kind);
  if (!b->rows || b->n_rows <= 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "baseline needs query rows");
  if (b->kind == IKV_BASE_SNAPKV && (b->pool_kernel < 1 || !(b->pool_kernel & 1)))
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "pool_kernel must be odd");
  std::vector<float> ones((size_t)b->n_rows, 1.0f);
  int64_t off = 0;
  for (int r = 0; r < n_req; ++r) {
    // observation-window / heavy-hitter mass: the multi-row scorer over the given rows, weights 1
    TRY(ikv_score_rows(c, reqs + r, 1, b->rows, b->n_rows, ones.data(), scores + off, stream));
    const int N = reqs[r].seq_len;
    if (N > 0) {
      if (b->kind == IKV_BASE_SNAPKV) {
        k_maxpool_cand<<<64, 256, 0, st>>>(scores + off, c->cand_pos, c->d_ncand, N, (b->pool_kernel - 1) / 2, c->rule_c);
        k_axpy_scatter<<<64, 256, 0, st>>>(c->rule_c, c->cand_pos, c->d_ncand, 1.0f, 1, scores + off);
      } else {
        k_h2o_boost<<<1, 1024, 0, st>>>(c->cand_pos, c->d_ncand, N, reqs[r].budget, b->recent_ratio, b->recent_floor,
                                        scores + off);
      }
      LAUNCH_CHECK(c);
    }
    off += N;
  }
  return IKV_OK;
}

ikv_status ikv_prefill_attn(ikv_ctx* c, int32_t layer, const ikv_request* req, int32_t q_pos0, int32_t n_q, const void* q,
                            void* out, float sm_scale, int64_t* kv_reads, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (!req || !q || !out || n_q < 0 || q_pos0 < 0) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_prefill_attn: bad argument");
  if ((int64_t)q_pos0 + n_q > req->seq_len) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "the chunk ends beyond seq_len");
  if (n_q == 0) return IKV_OK;
  const size_t esz = c->cfg.kv_dtype == IKV_BF16 ? 2 : 4;
  const size_t row = (size_t)c->cfg.n_q_heads * c->cfg.head_dim * esz;
  // Row i is a decode query at position q_pos0 + i: causal = its request ends at seq_len_i = q_pos0 + i + 1.  The rows of
  // a launch share the session's survivor list and read the chunk's own positions from the slot map; the K/V rows of the
  // request are re-read by every row out of L2 (33.5 MB per layer at 8,192 survivors).
  if (c->prefill_tiled && c->cfg.kv_dtype == IKV_BF16) {
    if (req->seq_len < 0 || !req->slot_map) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "bad request");
    if (layer < 0 || layer >= c->cfg.n_layers) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "layer %d out of range", layer);
    TRY(prefill_tiled(c, layer, *req, q_pos0, n_q, (const bf16*)q, (bf16*)out, sm_scale, (cudaStream_t)stream));
    if (kv_reads) {  // the session's list now covers [0, covered), covered <= q_pos0: its length is the count up to there
      const Session* s = session_find(c, req->session_id);
      k_prefill_reads<<<1, 1024, 0, (cudaStream_t)stream>>>(req->slot_map, c->cfg.dead_slot, q_pos0, n_q,
                                                            reinterpret_cast<unsigned long long*>(kv_reads),
                                                            s->d_n_live, s->covered);
      LAUNCH_CHECK(c);
    }
    return IKV_OK;
  }
  ikv_request rr[DEC_MAX_REQ];
  for (int i0 = 0; i0 < n_q; i0 += DEC_MAX_REQ) {
    const int nb = (n_q - i0 < DEC_MAX_REQ) ? n_q - i0 : DEC_MAX_REQ;
    for (int i = 0; i < nb; ++i) {
      rr[i] = *req;
      rr[i].seq_len = q_pos0 + i0 + i + 1;
    }
    TRY(ikv_decode_attn(c, layer, rr, nb, (const char*)q + (size_t)i0 * row, (char*)out + (size_t)i0 * row, sm_scale, stream));
  }
  if (kv_reads) {
    k_prefill_reads<<<1, 1024, 0, (cudaStream_t)stream>>>(req->slot_map, c->cfg.dead_slot, q_pos0, n_q,
                                                          reinterpret_cast<unsigned long long*>(kv_reads), nullptr, 0);
    LAUNCH_CHECK(c);
  }
  return IKV_OK;
}

ikv_status ikv_select_evict(ikv_ctx* c, const ikv_request* reqs, int32_t n_req, const float* scores,
                            int32_t* freed_slots, int32_t* n_freed, int32_t* n_kept, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (n_req < 0 || (n_req > 0 && (!reqs || !scores || !freed_slots || !n_freed || !n_kept)))
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_select_evict: NULL argument");
  for (int r = 0; r < n_req; ++r) TRY(check_request(c, reqs[r]));
  for (int r = 0; r < n_req; ++r)  // validate the whole batch before any session bookkeeping changes
    if (c->sessions.find(reqs[r].session_id) == c->sessions.end())
      IKV_FAIL(c, IKV_ERR_NO_SESSION, "session %llu does not exist", (unsigned long long)reqs[r].session_id);
  int64_t off = 0;
  SelBatch batch;
  int nb = 0, max_n = 0;
  for (int r = 0; r < n_req; ++r) {
    SelParams p;
    TRY(select_prepare(c, reqs[r], scores + off, freed_slots + off, n_freed + r, n_kept + r, &p));
    off += reqs[r].seq_len;
    if (p.N > CL_MAX_N) {  // beyond the cluster kernel's register blocking: single-CTA kernel, in stream order
      TRY(select_launch(c, batch, nb, max_n, (cudaStream_t)stream));
      nb = 0; max_n = 0;
      k_select_evict<<<1, 1024, 0, (cudaStream_t)stream>>>(p);
      LAUNCH_CHECK(c);
      continue;
    }
    batch.p[nb++] = p;
    if (p.N > max_n) max_n = p.N;
    if (nb == SEL_MAX_REQ) {
      TRY(select_launch(c, batch, nb, max_n, (cudaStream_t)stream));
      nb = 0; max_n = 0;
    }
  }
  TRY(select_launch(c, batch, nb, max_n, (cudaStream_t)stream));
  return IKV_OK;
}

ikv_status ikv_decode_attn(ikv_ctx* c, int32_t layer, const ikv_request* reqs, int32_t n_req, const void* q, void* out,
                           float sm_scale, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (n_req < 0 || (n_req > 0 && (!reqs || !q || !out))) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_decode_attn: NULL argument");
  if (layer < 0 || layer >= c->cfg.n_layers) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "layer %d out of range", layer);
  cudaStream_t st = (cudaStream_t)stream;
  const int Hq = c->cfg.n_q_heads, Hkv = c->cfg.n_kv_heads, D = c->cfg.head_dim;
  const size_t esz = c->cfg.kv_dtype == IKV_BF16 ? 2 : 4;
  for (int r0 = 0; r0 < n_req; r0 += DEC_MAX_REQ) {
    const int nb = (n_req - r0 < DEC_MAX_REQ) ? n_req - r0 : DEC_MAX_REQ;
    DecBatch batch;
    int max_items = 1;
    int items_of[DEC_MAX_REQ];
    bool fresh = false;  // a survivor list of this batch was just rewritten: no programmatic launch (R27)
    for (int i = 0; i < nb; ++i) {
      const ikv_request& r = reqs[r0 + i];
      if (r.seq_len < 0 || (r.seq_len > 0 && !r.slot_map)) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "bad request %d", r0 + i);
      Session* s = session_find(c, r.session_id);
      if (!s) IKV_FAIL(c, IKV_ERR_NO_SESSION, "session %llu does not exist", (unsigned long long)r.session_id);
      const bool stale = (r.flags & IKV_REQ_RESCAN) || s->map_ptr != r.slot_map || s->map_epoch != r.map_epoch ||
                         s->covered > r.seq_len ||
                         (s->covered == 0 && r.seq_len > 0) || (r.seq_len - s->covered) > 4096;
      if (stale) {
        TRY(session_live_reserve(c, *s, r.seq_len > 0 ? r.seq_len : 1));
        k_build_live<<<1, 1024, 0, st>>>(r.slot_map, r.seq_len, c->cfg.dead_slot, s->live_slots, s->d_n_live);
        LAUNCH_CHECK(c);
        s->covered = r.seq_len;
        s->map_ptr = r.slot_map;
        s->map_epoch = r.map_epoch;
        s->live_ub = r.seq_len;
        s->list_fresh = true;
      }
      fresh = fresh || s->list_fresh;
      s->list_fresh = false;
      batch.r[i].S = r.slot_map;
      batch.r[i].live_slots = s->live_slots;
      batch.r[i].n_live = s->d_n_live;
      batch.r[i].seq_len = r.seq_len;
      batch.r[i].covered = s->covered;
      batch.r[i].n_items = s->live_ub;
      batch.r[i].flags = r.flags;
      const int items = s->live_ub + (r.seq_len - s->covered);
      items_of[i] = items;
      if (items > max_items) max_items = items;
    }
    int n_split;
    if (c->cfg.kv_dtype == IKV_BF16) {
      // One request: one CTA (all KV heads of a token range) per SM, minus a few SMs left to the merge grid (2 of its
      // CTAs per SM): launched programmatically, it is then resident before the split drains, and the next call's
      // split overlaps it (measured: 148 -> 132 splits takes 7.7 -> 6.2 us per call).  A batch: two CTAs per SM, and
      // every request gets splits in proportion to its length (at least 16 tokens per split).
      const int n_hg = (Hkv + DM_CWARPS - 1) / DM_CWARPS;
      int reserve = (Hq * nb + 1) / 2;
      if (reserve > c->n_sm / 4) reserve = c->n_sm / 4;
      const int cap = ((nb == 1 ? 1 : 2) * c->n_sm - reserve) / n_hg;
      int64_t tot_items = 0;
      for (int i = 0; i < nb; ++i) tot_items += items_of[i] > 0 ? items_of[i] : 1;
      n_split = 1;
      for (int i = 0; i < nb; ++i) {
        int ns = (int)(((int64_t)(items_of[i] > 0 ? items_of[i] : 1) * cap) / tot_items);  // its share of the CTAs
        const int by_len = (items_of[i] + 15) / 16;
        if (ns > by_len) ns = by_len;
        if (ns < 1) ns = 1;
        if (ns > DMG_MAX_SPLIT) ns = DMG_MAX_SPLIT;
        batch.r[i].n_split = ns;
        if (ns > n_split) n_split = ns;
      }
    } else {
      // ~4 CTAs per SM, at least 64 tokens per split
      n_split = (4 * c->n_sm + Hkv * nb - 1) / (Hkv * nb);
      const int by_len = (max_items + 63) / 64;
      if (n_split > by_len) n_split = by_len;
      if (n_split < 1) n_split = 1;
      if (n_split > DMG_MAX_SPLIT) n_split = DMG_MAX_SPLIT;
      for (int i = 0; i < nb; ++i) batch.r[i].n_split = n_split;
    }
    TRY(ensure_parts(c, (int64_t)nb * Hq * n_split));
    TRY(dispatch_decode(c, layer, batch, nb, n_split, (const char*)q + (size_t)r0 * Hq * D * esz,
                        (char*)out + (size_t)r0 * Hq * D * esz, sm_scale, st, c->use_pdl && !fresh));
  }
  return IKV_OK;
}

ikv_status ikv_decode_attn_static(ikv_ctx* c, int32_t layer, const ikv_request* req, const void* q, void* out,
                                  float sm_scale, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (!req || !q || !out) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_decode_attn_static: NULL argument");
  if (layer < 0 || layer >= c->cfg.n_layers) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "layer %d out of range", layer);
  if (req->seq_len < 0 || (req->seq_len > 0 && !req->slot_map)) IKV_FAIL(c, IKV_ERR_INVALID_ARG, "bad request");
  if (!c->static_scratch)
    IKV_FAIL(c, IKV_ERR_CUDA, "ikv_decode_attn_static: cudaGetSymbolAddress failed in ikv_create: %s",
             c->static_scratch_err.c_str());
  cudaStream_t st = (cudaStream_t)stream;
  const int Hq = c->cfg.n_q_heads, Hkv = c->cfg.n_kv_heads, D = c->cfg.head_dim;
  const int items = req->seq_len;
  // split plan of ikv_decode_attn for one request
  int n_split;
  if (c->cfg.kv_dtype == IKV_BF16) {
    const int n_hg = (Hkv + DM_CWARPS - 1) / DM_CWARPS;
    int reserve = (Hq + 1) / 2;
    if (reserve > c->n_sm / 4) reserve = c->n_sm / 4;
    n_split = (c->n_sm - reserve) / n_hg;
    const int by_len = (items + 15) / 16;
    if (n_split > by_len) n_split = by_len;
  } else {
    n_split = (4 * c->n_sm + Hkv - 1) / Hkv;
    const int by_len = (items + 63) / 64;
    if (n_split > by_len) n_split = by_len;
  }
  if (n_split < 1) n_split = 1;
  if (n_split > DMG_MAX_SPLIT) n_split = DMG_MAX_SPLIT;
  const size_t o_bytes = (size_t)Hq * n_split * D * sizeof(float), ml_bytes = (size_t)Hq * n_split * sizeof(float2);
  const size_t need = 256 + o_bytes + ml_bytes;
  if (need > (size_t)IKV_STATIC_SCRATCH_BYTES)
    IKV_FAIL(c, IKV_ERR_CAPACITY,
             "ikv_decode_attn_static: %d query heads x %d splits x head_dim %d need %zu bytes of partials, the static "
             "scratch holds %d (use ikv_decode_attn)", Hq, n_split, D, need, (int)IKV_STATIC_SCRATCH_BYTES);
  // the array keeps the previous call's contents: the list length must read zero; the partials are overwritten
  CU(c, cudaMemsetAsync(c->static_scratch, 0, 256, st));
  DecBatch batch;
  memset(&batch, 0, sizeof batch);
  batch.r[0].S = req->slot_map;
  batch.r[0].live_slots = reinterpret_cast<const int32_t*>(c->static_scratch);  // empty list: never indexed
  batch.r[0].n_live = reinterpret_cast<const int32_t*>(c->static_scratch);
  batch.r[0].seq_len = req->seq_len;
  batch.r[0].covered = 0;       // every position comes from the slot map
  batch.r[0].n_items = 0;
  batch.r[0].flags = req->flags & IKV_REQ_INPUTS_COMPLETE;
  batch.r[0].n_split = n_split;
  // the kernels take their scratch from the context: lend them the static array for this launch
  float* po = c->part_o;
  float2* pm = c->part_ml;
  c->part_o = reinterpret_cast<float*>(c->static_scratch + 256);
  c->part_ml = reinterpret_cast<float2*>(c->static_scratch + 256 + o_bytes);
  const ikv_status rc = dispatch_decode(c, layer, batch, 1, n_split, q, out, sm_scale, st, false);
  c->part_o = po;
  c->part_ml = pm;
  return rc;
}

ikv_status ikv_train_loss(ikv_ctx* c, const float* scores, const int32_t* labels, int32_t n, const float* mem_rows,
                          int32_t n_rows, int32_t row_dim, const ikv_loss_cfg* cfg, float* terms, float* grad,
                          void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (n < 0 || !cfg || !terms || (n > 0 && (!scores || !labels || !grad)) || n_rows < 0 || (n_rows > 0 && (!mem_rows || row_dim <= 0)))
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_train_loss: bad argument");
  if (n > LOSS_MAX_N) IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "ikv_train_loss: n = %d exceeds %d", n, LOSS_MAX_N);
  LossParams p;
  p.s = scores; p.y = labels; p.n = n; p.mem_rows = mem_rows; p.n_rows = n_rows; p.row_dim = row_dim;
  p.rho = cfg->rho; p.gamma = cfg->gamma; p.eta = cfg->eta; p.terms = terms; p.grad = grad;
  k_train_loss<<<1, 1024, 0, (cudaStream_t)stream>>>(p);
  LAUNCH_CHECK(c);
  return IKV_OK;
}

ikv_status ikv_prune_host(ikv_ctx* c, const ikv_request* req, const void* q_rows_host, int32_t n_rows, int32_t q_dtype,
                          int32_t mode,
                          int32_t* slot_map_host, uint8_t* valid_host, float* scores_host, int32_t* freed_host,
                          int32_t* n_freed_host, int32_t* n_kept_host, void* stream) {
  if (!c) return IKV_ERR_INVALID_ARG;
  if (!req || !slot_map_host || !freed_host || !n_freed_host || !n_kept_host)
    IKV_FAIL(c, IKV_ERR_INVALID_ARG, "ikv_prune_host: NULL argument");
  cudaStream_t st = (cudaStream_t)stream;
  const int N = req->seq_len;
  if (q_dtype != IKV_F32 && q_dtype != IKV_BF16) IKV_FAIL(c, IKV_ERR_UNSUPPORTED, "q_dtype must be IKV_F32 or IKV_BF16");
  const size_t qes = (q_dtype == IKV_F32) ? 4 : 2;
  const int64_t qel = (int64_t)(n_rows > 0 ? n_rows : 0) * c->cfg.n_layers * c->cfg.n_q_heads * c->cfg.head_dim;
  TRY(ensure_staging(c, N > 0 ? N : 1, qel));
  ikv_request r = *req;
  r.slot_map = c->st_map;
  r.valid_mask = c->st_valid;
  r.xattn_pos = nullptr;
  r.n_xattn_pos = 0;
  TRY(check_request(c, r));
  CU(c, cudaMemcpyAsync(c->st_map, slot_map_host, (size_t)N * 4, cudaMemcpyHostToDevice, st));
  if (q_rows_host && n_rows > 0) {
    CU(c, cudaMemcpyAsync(c->st_qrows, q_rows_host, (size_t)qel * qes, cudaMemcpyHostToDevice, st));
    TRY(ikv_memory_update(c, r.session_id, c->st_qrows, n_rows, q_dtype, stream));
  }
  TRY(ikv_score(c, &r, 1, mode, c->st_scores, nullptr, stream));
  TRY(ikv_select_evict(c, &r, 1, c->st_scores, c->st_freed, c->st_counts, c->st_counts + 1, stream));
  // one device-to-host copy of [counts | slot map | freed list | valid mask] into the pinned mirror, then host copies
  const size_t out_bytes = 16 + (size_t)c->st_cap * 8 + (size_t)N;
  CU(c, cudaMemcpyAsync(c->st_host, c->st_out, out_bytes, cudaMemcpyDeviceToHost, st));
  if (scores_host) CU(c, cudaMemcpyAsync(scores_host, c->st_scores, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
  CU(c, cudaStreamSynchronize(st));
  const int32_t* h_counts = reinterpret_cast<const int32_t*>(c->st_host);
  const int32_t* h_map = reinterpret_cast<const int32_t*>(c->st_host + 16);
  const int32_t* h_freed = h_map + c->st_cap;
  const uint8_t* h_valid = reinterpret_cast<const uint8_t*>(h_freed + c->st_cap);
  *n_freed_host = h_counts[0];
  *n_kept_host = h_counts[1];
  memcpy(slot_map_host, h_map, (size_t)N * 4);
  if (valid_host) memcpy(valid_host, h_valid, (size_t)N);
  if (h_counts[0] > 0) memcpy(freed_host, h_freed, (size_t)h_counts[0] * 4);
  return IKV_OK;
}

}  // extern "C"
