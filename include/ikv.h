/*
 * ikv.h -- C-ABI of libikv: IntentKV's pruning pass and slot-map paged decode on one B200 (sm_100a).
 *
 * Source of every definition: arxiv 2606.09916 (cited as PAPER.md:<line> of /root/reference/PAPER.md);
 * readings of silent points are R1..R24 in DESIGN.md section 3.
 *
 * Conventions
 *  - "DEVICE" pointers are CUDA device memory of the current device; "HOST" pointers are ordinary host memory.
 *  - Ownership: the caller owns K/V pools, slot maps, q / out / scores buffers and the allocator that
 *    consumes freed slots.  The library owns session memories, its copy of the residual weights, scratch,
 *    the contents of the dead slot and the derived compact live lists.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Hot calls
 *    (ikv_memory_update, ikv_score, ikv_select_evict, ikv_decode_attn) only enqueue work on `stream`; they
 *    never synchronise the host, provided scratch was sized once with ikv_reserve (otherwise a call that
 *    needs more scratch grows it with cudaMalloc first, which synchronises).
 *  - Errors: every call returns an ikv_status.  Argument errors are reported before anything is launched.
 *    CUDA launch errors surface as IKV_ERR_CUDA.  Nothing throws or aborts across the ABI.
 *    ikv_last_error() returns a human-readable description of the last failure on that context.
 *  - Pool layout: K and V are [n_layers][n_slots][n_kv_heads][head_dim] (token-major), element type
 *    kv_dtype; slot = page * page_size + offset.  A request reaches K/V only through its slot map
 *    S[0:seq_len).
 */
#ifndef IKV_H
#define IKV_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ikv_ctx ikv_ctx; /* opaque, library-owned */
typedef int32_t ikv_status;

#define IKV_OK 0
#define IKV_ERR_INVALID_ARG (-1)
#define IKV_ERR_NO_SESSION (-2)
#define IKV_ERR_CAPACITY (-3)
#define IKV_ERR_OOM (-4)
#define IKV_ERR_CUDA (-5)
#define IKV_ERR_UNSUPPORTED (-6)

/* kv_dtype / q_dtype */
#define IKV_F32 0
#define IKV_BF16 1

/* scorer modes ("three scorer modes") and ablation knobs, OR-ed into `mode` */
#define IKV_MODE_MEMORY 0    /* rule score against the session QueryMemory M_t (Eq. 3)              */
#define IKV_MODE_LEARNABLE 1 /* rule + alpha * MLP(phi (+) c) (Eq. 4-6); needs ikv_residual_load    */
#define IKV_MODE_QUERY 2     /* rule score against normalize(Enc(q_t)) of the latest update only    */
#define IKV_FLAG_NO_XATTN 0x100    /* "- x-attn": c_j = 0                                            */
#define IKV_FLAG_NO_RESIDUAL 0x200 /* "- residual": alpha = 0, recovers the rule scorer exactly      */

/* request flags */
#define IKV_REQ_RESCAN 1          /* ikv_decode_attn: ignore the cached live list, rescan the slot map            */
#define IKV_REQ_INPUTS_COMPLETE 2 /* ikv_decode_attn: q, the slot-map tail and the K/V rows of this call were
                                     complete before the PRECEDING kernel of the stream started (e.g. precomputed
                                     queries): the kernel may read them before it orders itself after that kernel */

/* ikv_config.flags */
#define IKV_CFG_NO_PDL 1       /* never launch with programmatic stream serialization (plain stream order)          */
#define IKV_CFG_NO_PDL_PRUNE 2 /* ... only the kernels of the pruning pass                                          */

typedef struct {
  int32_t n_layers, n_q_heads, n_kv_heads, head_dim; /* L, H_q, H_kv, D; H_q % H_kv == 0; D in {64,128}   */
  int32_t page_size;                                 /* 16 (R18)                                          */
  int32_t kv_dtype;                                  /* IKV_BF16 | IKV_F32 (R20)            */
  int64_t n_slots;                                   /* pool capacity in token slots, dead slot included  */
  void *k_pool, *v_pool;                             /* DEVICE, caller-owned, [L][n_slots][H_kv][D]       */
  int32_t dead_slot;                                 /* s+ ; ikv_create writes K=-1e4, V=0 there on every
                                                        layer                              */
  float lambda;                                      /* decay of Eq. 2; the paper uses 0.5 */
  int32_t max_sessions;                              /* LRU capacity; the paper uses 1024  */
  int32_t flags;                                     /* IKV_CFG_*; 0 = defaults                           */
} ikv_config;

/* One request of a batch.  The array of requests lives on the HOST. */
typedef struct {
  uint64_t session_id;         /* explicit session key (first priority)                     */
  int32_t *slot_map;           /* DEVICE, caller-owned, length >= seq_len; rewritten in place by
                                  ikv_select_evict (Eq. 7)                                                */
  uint8_t *valid_mask;         /* DEVICE, optional (may be NULL), length >= seq_len (R21)                 */
  int32_t seq_len;             /* N -- never modified                                                     */
  int32_t prefix_len;          /* pi: protected system prefix [0,pi)                                      */
  int32_t q_start, q_end;      /* actionable query span [q_s,q_e); 0 <= pi <= q_s <= q_e <= N             */
  int32_t budget;              /* C >= 0                                                                  */
  int32_t radix_protected_len; /* positions below it are never reported as freed (PAPER.md:132 (a))       */
  const int32_t *xattn_pos;    /* DEVICE, positions forming K^q (Eq. 6); NULL => [q_s,q_e) (R7)           */
  int32_t n_xattn_pos;
  int32_t flags;               /* IKV_REQ_*                                                               */
  uint32_t map_epoch;          /* version of the CONTENT behind slot_map: a caller that reuses a slot-map allocation
                                  for different content (freed and reallocated at the same address, edited by hand)
                                  bumps it; ikv_decode_attn rescans when it differs from the epoch seen by the last
                                  ikv_select_evict / rescan of the session.  0 is an ordinary value.            */
} ikv_request;

/* Residual head parameters (R9), HOST fp32 arrays, row-major [out][in]:
 * wq[128][3D+1] bq[128]  wk[128][D] bk[128]  wv[128][D] bv[128]  fc1_w[256][3D+1+128] fc1_b[256]
 * fc2_w[256] fc2_b[1]; alpha is clipped to [-5,5] at inference. */
typedef struct {
  const float *wq, *bq, *wk, *bk, *wv, *bv, *fc1_w, *fc1_b, *fc2_w, *fc2_b;
  float alpha;
} ikv_residual_weights;

/* ---- lifecycle ------------------------------------------------------------------------------------- */
/* Validates the config, initialises the dead slot's K/V rows on every layer, allocates the session slab.
 * Synchronises.  *out receives the context.  For bf16 pools with head_dim 64 or 128 it also encodes two TMA tensor maps
 * (cuTensorMapEncodeTiled through the runtime's driver entry point; no device memory) that describe k_pool and v_pool as
 * 2-D tensors [n_layers * n_slots * n_kv_heads][head_dim]: ikv_prefill_attn and ikv_score_rows fetch their tiles through
 * them (tile::gather4).  If that fails (old driver, more than 2^31 - 1 rows, pools not 16-byte aligned) those calls use
 * their cp.async producers instead; nothing else changes. */
ikv_status ikv_create(const ikv_config *cfg, ikv_ctx **out);
ikv_status ikv_destroy(ikv_ctx *ctx);
/* ctx == NULL: the reason of the last failed ikv_create on this thread. */
const char *ikv_last_error(const ikv_ctx *ctx);

/* Pre-sizes every scratch buffer so that later hot calls never allocate: `max_tokens` = largest sum of
 * seq_len over one batch, `max_requests` = largest batch.  Synchronises. */
ikv_status ikv_reserve(ikv_ctx *ctx, int64_t max_tokens, int32_t max_requests);

/* ---- sessions (explicit session id, LRU store) ------------------------------------------ */
/* M_0 = 0 (R3).  Opening an existing id resets it.  Beyond max_sessions the least-recently-used session is
 * evicted. */
ikv_status ikv_session_open(ikv_ctx *ctx, uint64_t id);
/* child <- copy of the parent's QueryMemory (a forked trajectory); shares no K/V state. */
ikv_status ikv_session_fork(ikv_ctx *ctx, uint64_t parent, uint64_t child, void *stream);
ikv_status ikv_session_close(ikv_ctx *ctx, uint64_t id);
/* Debug/test access to the state: copies M_t ([L][H_q][D] fp32) to / from HOST memory.  Synchronises. */
ikv_status ikv_session_get_memory(ikv_ctx *ctx, uint64_t id, float *host_out);
ikv_status ikv_session_set_memory(ikv_ctx *ctx, uint64_t id, const float *host_in);

/* Copies the residual head to the device (synchronises). */
ikv_status ikv_residual_load(ikv_ctx *ctx, const ikv_residual_weights *w);

/* ---- hot path ------------------------------------------------------------------------------------------ */
/* a0, Eq. 2: Enc = mean of the n post-RoPE Q rows; M <- e^{-lambda} M + Enc; each
 * (layer, head) row <- row / max(||row||_2, 1e-12).  q_rows: DEVICE [n][L][H_q][D], q_dtype IKV_F32 or
 * IKV_BF16.  Also stores normalize(Enc) for IKV_MODE_QUERY.  The session is created if it does not exist. */
ikv_status ikv_memory_update(ikv_ctx *ctx, uint64_t id, const void *q_rows, int32_t n, int32_t q_dtype,
                             void *stream);

/* a1-a5, Eq. 3-6: scores of every position of every request.
 * scores: DEVICE fp32, requests concatenated (request r starts at sum of seq_len of requests < r), indexed by
 * logical position: s_j at candidate positions, +INF at forced live positions, -INF at dead positions (R6).
 * rule_out: optional DEVICE fp32 of the same shape receiving rule_j (Eq. 3) at candidates, 0 elsewhere. */
ikv_status ikv_score(ikv_ctx *ctx, const ikv_request *reqs, int32_t n_req, int32_t mode, float *scores,
                     float *rule_out, void *stream);

/* a6-a7, Eq. 1 and Eq. 7.  For each request: if N <= C nothing changes
 * (R15).  Otherwise K* = F u top-C*(candidates by score desc, position asc), C* = max(0, C - |F|) (R13, R14);
 * S[j] <- s+ for every live j outside K*; valid_mask[j] = (S'[j] != s+); no K/V byte moves.
 * freed_slots: DEVICE int32, requests concatenated like `scores` (capacity seq_len each); receives, per
 * request, the slots that pass the prefix-safe test (a)(b)(c) of PAPER.md:132, each once, ordered by first
 * dropped position (R22).  n_freed / n_kept: DEVICE int32[n_req].
 * Also refreshes the session's compact live list used by ikv_decode_attn.
 * Stream ordering: the kernel is launched with programmatic stream serialization and reads the slot maps before it
 * orders itself after the preceding kernel of the stream (the producer of `scores`); `scores` are read after that
 * point.  The slot maps of the batch must therefore not be written by the kernel enqueued directly before this call
 * (they never are when that kernel is ikv_score's or any other scorer: a map is edited between events, not inside one). */
ikv_status ikv_select_evict(ikv_ctx *ctx, const ikv_request *reqs, int32_t n_req, const float *scores,
                            int32_t *freed_slots, int32_t *n_freed, int32_t *n_kept, void *stream);

/* a8 (R16): paged GQA decode attention of one layer through the slot map, dead entries
 * skipped:  out[r,h] = sum_{j<seq_len, S_r[j] != s+} softmax_j(q[r,h] . K[layer, h div G, S_r[j]] * sm_scale)
 *                       V[layer, h div G, S_r[j]].
 * q, out: DEVICE [n_req][H_q][D]; bf16 for a bf16 pool, fp32 for an fp32 pool.  Positions below the seq_len of
 * the last ikv_select_evict on the same (session, slot_map) come from the cached compact live list; positions
 * appended since are read from slot_map.  A caller that edited the slot map itself passes IKV_REQ_RESCAN.
 * Stream ordering (R27): the kernels of this call are launched with programmatic stream serialization.  Before
 * they order themselves after the preceding kernel of the stream they read only the session's survivor list and the K/V
 * rows of the positions it covers -- state that kernel cannot be producing (after ikv_select_evict or a rescan the library
 * launches the first decode call without the programmatic attribute).  q, the slot-map tail and the K/V rows of positions
 * appended since the last select are read after that point, so any producer kernel is safe, including one that triggers
 * its dependents early.  IKV_REQ_INPUTS_COMPLETE lifts this for a request whose inputs were complete before the preceding
 * kernel started (precomputed queries): the whole call then overlaps that kernel.  IKV_CFG_NO_PDL turns programmatic
 * launches off.  Up to 32 requests go into one launch; larger batches are chunked. */
ikv_status ikv_decode_attn(ikv_ctx *ctx, int32_t layer, const ikv_request *reqs, int32_t n_req, const void *q,
                           void *out, float sm_scale, void *stream);

/* a8 without any allocation, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses
 * that forbid it).  One request, no session: every position [0, seq_len) is read through req->slot_map, entries equal to
 * the dead slot are skipped (session_id, budget and the span fields of the request are ignored); q and out as in
 * ikv_decode_attn with n_req = 1.  The split partials -- the only scratch of the decode kernels -- live in a file-scope
 * device array of IKV_STATIC_SCRATCH_BYTES that every GPU holds from the moment it loads the library until exit; its
 * address is resolved once, in ikv_create (cudaGetSymbolAddress on the context's device).  The call performs no
 * cudaMalloc / cudaFree and calls no allocating routine.
 * Limit: 256 + n_q_heads * n_split * (head_dim + 2) * 4 bytes must fit the array, n_split being the split count the
 * library picks for seq_len (at most one per SM; 32 or 40 query heads at head_dim 128 always fit, 64 heads up to 92
 * splits = sequences up to 1,472 positions); beyond it the call returns IKV_ERR_CAPACITY and enqueues nothing.
 * Every call on a device shares the array, which keeps the previous call's contents (the call clears the one word that
 * must start at zero): calls that can overlap on the GPU (different streams, or a captured graph replayed concurrently)
 * race on it -- keep them on one stream.  Errors: IKV_ERR_INVALID_ARG, IKV_ERR_CAPACITY, IKV_ERR_CUDA. */
#define IKV_STATIC_SCRATCH_BYTES (3 * 1024 * 1024)
ikv_status ikv_decode_attn_static(ikv_ctx *ctx, int32_t layer, const ikv_request *req, const void *q, void *out,
                                  float sm_scale, void *stream);

/* ---- follow-ups of the hot path ------------------------------------------------------------ */
/* Multi-row scorer ("window of W tail Q rows", O(W L H_q N); :159 W = 32; :310; R28): n_rows
 * un-collapsed rows per (layer, query head), rows[r][L][H_q][D] DEVICE fp32, used as given; every row is its own softmax
 * over the candidates of Eq. 3 and the rows are combined with the HOST weights[n_rows]:
 *   s_j = sum_r weights[r] sum_{l,h} softmax_{i in A}(rows[r,l,h] . K[l, h div G, S[i]] / sqrt(D))_j.
 * n_rows = 1, weights = {1}, rows = M_t is ikv_score(IKV_MODE_MEMORY) bit for bit.  scores as in ikv_score (fillers
 * included).  Below four rows: one pass over the keys per row.  From four rows on (bf16 pools; six without the pool's
 * tensor map): banks of 128 / G rows as a dense tile on tcgen05, two sweeps over the keys per bank (IKV_TUNE_ROWS_TC).  The first call allocates the bank and
 * its partials (cudaMalloc). */
ikv_status ikv_score_rows(ikv_ctx *ctx, const ikv_request *reqs, int32_t n_req, const float *rows, int32_t n_rows,
                          const float *weights, float *scores, void *stream);

/* Baseline scorers on the same dead-slot substrate (R29-R31).  They only
 * produce `scores` (same layout and fillers as ikv_score); budget, forced set, slot-map redirection and the prefix-safe
 * free are ikv_select_evict's, shared by every scorer.
 *   IKV_BASE_STREAMING  StreamingLLM: candidates at positions < n_sink first, then the most recent ones (no key is read)
 *   IKV_BASE_SNAPKV     SnapKV: the multi-row scorer over the W observation rows `rows` (weights 1), then max-pool
 *                       smoothing of width pool_kernel (7) over the logical positions, candidates only
 *   IKV_BASE_H2O        H2O: heavy-hitter mass = the multi-row scorer over the bank `rows` (weights 1); the
 *                       min(C*, max(recent_floor, round(recent_ratio C*))) most recent candidates are kept first */
#define IKV_BASE_STREAMING 1
#define IKV_BASE_SNAPKV 2
#define IKV_BASE_H2O 3
typedef struct {
  int32_t kind;          /* IKV_BASE_*                                            */
  const float *rows;     /* DEVICE [n_rows][L][H_q][D] fp32 (SNAPKV, H2O)         */
  int32_t n_rows;
  int32_t n_sink;        /* STREAMING: 4                           */
  int32_t pool_kernel;   /* SNAPKV: 7, odd                         */
  float recent_ratio;    /* H2O                                                   */
  int32_t recent_floor;  /* H2O                                                   */
} ikv_baseline;
ikv_status ikv_score_baseline(ikv_ctx *ctx, const ikv_request *reqs, int32_t n_req, const ikv_baseline *b, float *scores,
                              void *stream);

/* Prefill / chunked-prefill attention of one layer through the slot map (R32): n_q query
 * rows at logical positions q_pos0 .. q_pos0 + n_q - 1 of the request (q_pos0 + n_q <= req->seq_len); row i attends,
 * causally, every position j <= q_pos0 + i with S[j] != s+.  q, out: DEVICE [n_q][H_q][D], pool dtype.
 * kv_reads: optional DEVICE int64[2], ACCUMULATED: [0] += sum_i (q_pos0 + i + 1) = Raw KV Reads sum |R_t|,
 * [1] += sum_i #{j <= q_pos0 + i : S[j] != s+} = Eff. KV Reads sum |K_t|.
 * bf16 pools: one tiled launch per 1,024 rows (IKV_TUNE_PREFILL_TILED); the session's cached survivor list is brought to
 * cover a prefix [0, covered), covered <= q_pos0 (rebuilt from the slot map when it is stale or reaches into the chunk),
 * exactly as ikv_decode_attn maintains it; the scratch for the split partials grows on demand (cudaMalloc). */
ikv_status ikv_prefill_attn(ikv_ctx *ctx, int32_t layer, const ikv_request *req, int32_t q_pos0, int32_t n_q, const void *q,
                            void *out, float sm_scale, int64_t *kv_reads, void *stream);

/* The whole pruning pass of one request with HOST buffers (used for end-to-end timing): copies
 * q_rows_host ([n_rows][L][H_q][D], q_dtype IKV_F32 or IKV_BF16; may be NULL/0 to skip the memory update) and
 * slot_map_host[seq_len] to the device, runs ikv_memory_update -> ikv_score(mode) -> ikv_select_evict, brings the new
 * slot map, valid mask (optional), freed list and counts back in one device-to-host copy and synchronises `stream`.
 * req->slot_map / valid_mask / xattn_pos are ignored (xattn_pos defaults to the span). */
ikv_status ikv_prune_host(ikv_ctx *ctx, const ikv_request *req, const void *q_rows_host, int32_t n_rows,
                          int32_t q_dtype, int32_t mode, int32_t *slot_map_host, uint8_t *valid_host,
                          float *scores_host, int32_t *freed_host, int32_t *n_freed_host, int32_t *n_kept_host,
                          void *stream);

/* Kernel-level timing for bench.py's roofline and breakdown: while enabled, the library brackets kernels with CUDA
 * events on the caller's stream (no host synchronisation; skipped during stream capture).  level 1: only the two dominant
 * kernels (slots IKV_PROF_KEY_PASS, IKV_PROF_DECODE; the layer-major key pass stamps its own start and end with
 * %globaltimer instead, so that no event sits between programmatically launched kernels); level 2: every kernel of the path -- the events between the launches
 * take away the overlap of programmatically launched kernels, so level 2 is a diagnostic, not a timing of the pass.
 * ikv_profile_read synchronises, sums the elapsed times recorded per slot since the last read and clears them:
 * out_ms[IKV_PROF_SLOTS] = total ms per slot, out_n[IKV_PROF_SLOTS] = launch counts. */
#define IKV_PROF_KEY_PASS 0     /* k_key_pass / k_score_logits */
#define IKV_PROF_DECODE 1       /* k_decode_mma / k_decode_split */
#define IKV_PROF_MEM_UPDATE 2
#define IKV_PROF_PARTITION 3
#define IKV_PROF_MEM_PREP 4
#define IKV_PROF_POST_KEY 5
#define IKV_PROF_RULE 6
#define IKV_PROF_RESIDUAL 7
#define IKV_PROF_SELECT 8
#define IKV_PROF_DECODE_MERGE 9
#define IKV_PROF_SLOTS 12
ikv_status ikv_profile_enable(ikv_ctx *ctx, int32_t level);
ikv_status ikv_profile_read(ikv_ctx *ctx, float *out_ms, int32_t *out_n);

/* Experiment knobs (A/B measurements; defaults are the tuned values).  Unknown knobs return
 * IKV_ERR_INVALID_ARG.  Never needed for correctness. */
#define IKV_TUNE_L2_HINTS 1 /* bit 0: key stream evict_first; bit 1: logits scratch evict_last; bit 2: rule reads
                               evict_first (default 7)                                                         */
#define IKV_TUNE_RESID_TC 2 /* 1 (default): residual head with folded cross attention on tcgen05 when the call has at
                               most 64 cross-attention positions; 0: always the unfolded kernel                */
#define IKV_TUNE_LAYER_MAJOR 3 /* 1 (default): layer-major key pass with deferred normalisation (no logits scratch) when
                                  the call fits its on-chip capacity and has at least three 32-token tiles per SM;
                                  2: whenever it fits; 0: always the logits-scratch key pass                      */
#define IKV_TUNE_ROWS_TC 5 /* 1 (default): ikv_score_rows with four or more rows on a bf16 pool runs banks of 128 / G rows
                              on tcgen05, two sweeps over the keys per bank, the keys fetched by TMA gather4 through the
                              tensor map of the pool (six or more rows, cp.async gather warps, when ikv_create could
                              not build the map); 2: from two rows up; 3: as 2 with the cp.async gather warps; 0: one
                              single-row pass per row                                                            */
#define IKV_TUNE_PREFILL_TILED 6 /* ikv_prefill_attn on a bf16 pool.  1 (default): tcgen05 kernel (128 / G query rows x G
                                    heads per CTA) for G in {1, 2, 4, 8}, its K/V tiles fetched by TMA gather4 through the
                                    tensor maps ikv_create builds over the pools; the mma.sync tiled kernel for G = 5;
                                    chunks of eight or more such tiles put two of them on a CTA (they share every
                                    gathered K/V tile);
                                    3: the tcgen05 kernel with cp.async producers (also the fallback when the tensor maps
                                    could not be built); 4: TMA producers, always one tile per CTA; 5: TMA producers, two
                                    tiles per CTA from two tiles on; 2: always the mma.sync tiled kernel (32 rows per
                                    CTA); 0: row by row through the decode kernels                                  */
#define IKV_TUNE_BATCH_LANES 4 /* lanes of a batched ikv_score (default 4, 1..8): the partition / fold / residual kernels
                                 of request r run on internal stream r % lanes with that lane's own scratch, the key
                                 passes in request order on the caller's stream; 1 = one request after another      */
ikv_status ikv_tune(ikv_ctx *ctx, int32_t knob, int32_t value);

/* NEXT-4: the training objective of the residual head, Eq. 8, and its gradient with respect to the
 * scores, for one (session, turn) row:  L = L_BCE + rho L_rank + gamma mean sigma(s) + eta mean_r (||row_r||_2 - 1)^2
 * (readings R34-R37 in DESIGN.md).  scores [n] DEVICE fp32 logits; labels [n] DEVICE int32: 1 positive, 0 negative, any
 * other value (-100) excluded; mem_rows [n_rows][row_dim] DEVICE fp32, the un-normalised memory rows of the norm term
 * (NULL / 0: term 0); terms [5] DEVICE = {L, L_BCE, L_rank, keep, norm}, the last three unweighted; grad [n] DEVICE =
 * dL/dscores (0 at excluded entries).  The backward pass through the residual head and the optimiser are not part of
 * the library.  n <= 131,072 (one CTA), else IKV_ERR_UNSUPPORTED.  Enqueues on `stream`; no host synchronisation. */
typedef struct {
  float rho, gamma, eta; /* the paper's defaults: 0.05, 0.01, 0.001 */
} ikv_loss_cfg;
ikv_status ikv_train_loss(ikv_ctx *ctx, const float *scores, const int32_t *labels, int32_t n, const float *mem_rows,
                          int32_t n_rows, int32_t row_dim, const ikv_loss_cfg *cfg, float *terms, float *grad,
                          void *stream);

/* Test support: enqueues a kernel that signals its dependents first (griddepcontrol.launch_dependents), idles for
 * delay_us microseconds and only then copies `bytes` (a multiple of 16) from src to dst (both DEVICE).  Models a producer of
 * q that triggers early; tests/test_gpu_parity.py uses it to check the stream ordering of ikv_decode_attn. */
ikv_status ikv_test_late_writer(void *dst, const void *src, int64_t bytes, int32_t delay_us, void *stream);

/* Library / build identification, e.g. "ikv 0.1 sm_100a". */
const char *ikv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* IKV_H */
