/*
 * ikv_oracle.c -- CPU ORACLE for the IntentKV hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is a plain, slow, obviously-correct restatement of what the path
 * computes, written from /root/reference/PAPER.md (arxiv 2606.09916) step by
 * step in the paper's order and notation.  It shares NO code with the CUDA
 * path (paper_2606_09916_b200/csrc) and may only be used by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg.
 *
 * Arithmetic: every floating-point step is carried out in IEEE double.
 * bf16 / fp32 inputs are up-converted exactly.  There is no blocking, fusion
 * or reordering beyond what the paper's formulas state; OpenMP is used only
 * around outermost independent loops (each iteration writes disjoint output).
 *
 * Pool layout: K and V are [L][n_slots][H_kv][D],
 * reached only through the slot map S ("slot map of request r").
 *
 * Readings of the paper where it is silent are listed in DESIGN.md section 3
 * (R1..R22) and referenced below as "reading Rn".
 *
 * Pins (tests/test_oracle_*.py): see DESIGN.md section 4.  The only part that is
 * "parity unpinned" is the absolute numeric value of scores on the paper's
 * real data (the paper prints no worked numeric example of Eq. 2-6).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define IKV_O_F32 0
#define IKV_O_BF16 1

#define CLS_DEAD 0
#define CLS_FORCED 1
#define CLS_CAND 2

/* residual-head constants, PAPER.md:108 ("H_c = 4 heads and width d_c = 128")
 * and PAPER.md:115 ("two-layer GELU network of hidden width h=256"). */
#define DC 128
#define HC 4
#define HID 256

#define FLAG_NO_XATTN 1    /* "- x-attn forces c_j = 0" */
#define FLAG_NO_RESIDUAL 2 /* "- residual clamps alpha = 0" */

/* exact bf16 -> double: bf16 is the top 16 bits of an IEEE binary32 */
static double bf16_to_double(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return (double)f;
}

/* element e of a pool row, exact up-conversion */
static double pool_elem(const void *pool, int dtype, int64_t idx) {
  if (dtype == IKV_O_BF16) return bf16_to_double(((const uint16_t *)pool)[idx]);
  return (double)((const float *)pool)[idx];
}

/* index of K[l, kvh, slot, d] in the [L][n_slots][H_kv][D] pool */
static int64_t pool_index(int64_t n_slots, int Hkv, int D, int l, int64_t slot, int kvh, int d) {
  return (((int64_t)l * n_slots + slot) * Hkv + kvh) * D + d;
}

/* ------------------------------------------------------------------------
 * O1  QueryMemory update.  PAPER.md:77-81, Eq. (2):
 *     M_t = e^{-lambda} M_{t-1} + Enc(q_t),
 * Enc(q_t) "averages the post-RoPE Q rows over the actionable query span";
 * "After each update, M_t is projected to unit norm along the head dimension".
 * Readings R2 (Enc is not pre-normalised), R3 (M_0 = 0; divide by
 * max(norm, 1e-12) so a zero row stays zero).
 * M: [L][Hq][D] double, in/out.  q_rows: [n][L][Hq][D] fp32.
 * ---------------------------------------------------------------------- */
void oracle_memory_update(double *M, const float *q_rows, int n, int L, int Hq, int D,
                          double lambda) {
  const double decay = exp(-lambda);
  for (int l = 0; l < L; ++l)
    for (int h = 0; h < Hq; ++h) {
      double *m = M + ((int64_t)l * Hq + h) * D;
      for (int d = 0; d < D; ++d) {
        double enc = 0.0;
        for (int r = 0; r < n; ++r)
          enc += (double)q_rows[(((int64_t)r * L + l) * Hq + h) * D + d];
        enc /= (double)n;
        m[d] = decay * m[d] + enc;
      }
      double nrm2 = 0.0;
      for (int d = 0; d < D; ++d) nrm2 += m[d] * m[d];
      double nrm = sqrt(nrm2);
      if (nrm < 1e-12) nrm = 1e-12;
      for (int d = 0; d < D; ++d) m[d] /= nrm;
    }
}

/* "query" scorer mode ("- memory replaces M_t with Enc(q_t)"):
 * the state used for scoring is normalize(Enc(q_t)) -- one update from M_0=0. */
void oracle_query_encoding(double *M_out, const float *q_rows, int n, int L, int Hq, int D) {
  memset(M_out, 0, sizeof(double) * (size_t)L * Hq * D);
  oracle_memory_update(M_out, q_rows, n, L, Hq, D, 0.0);
}

/* ------------------------------------------------------------------------
 * O2  partition.  PAPER.md:59 (F = [0,pi) U [q_s,q_e), H = [0,N) \ F) and
 * PAPER.md:489-491 (live set L = {j : S[j] != s+}; split L into forced F and
 * candidates A).  cls[j] in {DEAD, FORCED, CAND}.
 * ---------------------------------------------------------------------- */
void oracle_partition(const int32_t *S, int N, int32_t dead, int pi, int qs, int qe,
                      uint8_t *cls, int32_t *counts /* [3]: dead, forced, cand */) {
  counts[0] = counts[1] = counts[2] = 0;
  for (int j = 0; j < N; ++j) {
    uint8_t c;
    if (S[j] == dead) c = CLS_DEAD;
    else if (j < pi || (j >= qs && j < qe)) c = CLS_FORCED;
    else c = CLS_CAND;
    cls[j] = c;
    counts[c]++;
  }
}

/* ------------------------------------------------------------------------
 * O3-O5  rule score.  PAPER.md:83-88, Eq. (3):
 *   a_{l,h,j} = exp(M[l,h].K[l,h,j]/sqrt(D)) / sum_{i in H} exp(M[l,h].K[l,h,i]/sqrt(D))
 *   rule_j    = sum_{l,h} a_{l,h,j}
 * "KV heads expanded to H_q under GQA": query head h reads KV head h div G
 * (reading R4).  The softmax runs over candidates only (reading R5).
 * rule: [N] double; written at candidate positions, 0 elsewhere.
 * logits_out (optional): [L][Hq][N] double, x_{l,h,j} at candidates, 0 elsewhere.
 * ---------------------------------------------------------------------- */
void oracle_rule_score(const void *k_pool, int kv_dtype, int64_t n_slots, int L, int Hq, int Hkv,
                       int D, const double *M, const int32_t *S, const uint8_t *cls, int N,
                       double *rule, double *logits_out) {
  const int G = Hq / Hkv;
  const double inv_sqrt_d = 1.0 / sqrt((double)D);
  const int64_t LH = (int64_t)L * Hq;
  /* a[(l,h)][j] */
  double *a = (double *)malloc(sizeof(double) * (size_t)LH * (size_t)N);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t lh = 0; lh < LH; ++lh) {
    const int l = (int)(lh / Hq), h = (int)(lh % Hq), kvh = h / G;
    const double *m = M + lh * D;
    double *x = a + lh * N;
    /* O3 logits */
    double xmax = -INFINITY;
    for (int j = 0; j < N; ++j) {
      x[j] = 0.0;
      if (cls[j] != CLS_CAND) continue;
      double dot = 0.0;
      for (int d = 0; d < D; ++d)
        dot += m[d] * pool_elem(k_pool, kv_dtype, pool_index(n_slots, Hkv, D, l, S[j], kvh, d));
      x[j] = dot * inv_sqrt_d;
      if (x[j] > xmax) xmax = x[j];
    }
    if (logits_out) memcpy(logits_out + lh * N, x, sizeof(double) * (size_t)N);
    /* O4 softmax over the candidate set, with max subtraction */
    double denom = 0.0;
    for (int j = 0; j < N; ++j)
      if (cls[j] == CLS_CAND) denom += exp(x[j] - xmax);
    for (int j = 0; j < N; ++j)
      x[j] = (cls[j] == CLS_CAND) ? exp(x[j] - xmax) / denom : 0.0;
  }
  /* O5 rule_j = sum over (l,h) in fixed order */
#pragma omp parallel for schedule(static)
  for (int j = 0; j < N; ++j) {
    double r = 0.0;
    if (cls[j] == CLS_CAND)
      for (int64_t lh = 0; lh < LH; ++lh) r += a[lh * N + j];
    rule[j] = r;
  }
  free(a);
}

/* ------------------------------------------------------------------------
 * O6a  mean key.  PAPER.md:102: "k_bar_j be the mean of K[l,h,j] over
 * GQA-expanded heads and layers": (1/(L*Hq)) sum_{l,h} K[l, h div G, S[j]].
 * pos: list of positions; kbar: [npos][D].
 * ---------------------------------------------------------------------- */
void oracle_mean_key(const void *k_pool, int kv_dtype, int64_t n_slots, int L, int Hq, int Hkv,
                     int D, const int32_t *S, const int32_t *pos, int npos, double *kbar) {
  const int G = Hq / Hkv;
#pragma omp parallel for schedule(static)
  for (int p = 0; p < npos; ++p) {
    const int64_t slot = S[pos[p]];
    for (int d = 0; d < D; ++d) {
      double acc = 0.0;
      for (int l = 0; l < L; ++l)
        for (int h = 0; h < Hq; ++h)
          acc += pool_elem(k_pool, kv_dtype, pool_index(n_slots, Hkv, D, l, slot, h / G, d));
      kbar[(int64_t)p * D + d] = acc / (double)(L * Hq);
    }
  }
}

/* O6b  m_bar: "the analogous mean over M_t" */
void oracle_mean_memory(const double *M, int L, int Hq, int D, double *mbar) {
  for (int d = 0; d < D; ++d) {
    double acc = 0.0;
    for (int64_t lh = 0; lh < (int64_t)L * Hq; ++lh) acc += M[lh * D + d];
    mbar[d] = acc / (double)(L * Hq);
  }
}

static double gelu_erf(double x) { return 0.5 * x * (1.0 + erf(x / sqrt(2.0))); } /* reading R11 */

/* ------------------------------------------------------------------------
 * O6c  residual head.  PAPER.md:95-115, Eq. (4)-(6).
 *   phi_j = [ kbar_j || mbar || kbar_j (.) mbar || rule_j ]   in R^{3D+1}   (Eq. 5)
 *   c_j   = CrossAttn(W_Q phi_j, W_K Kq, W_V Kq),  H_c = 4, d_c = 128       (Eq. 6)
 *   s_j   = rule_j + alpha * MLP(phi_j (+) c_j), alpha clipped to [-5,5]    (Eq. 4)
 * Topology (reading R9, pinned by the 214,274 parameter count PAPER.md:115):
 * all five linear maps carry a bias, no attention output projection, MLP input
 * is phi (+) c (3D+1+128), hidden 256, exact-erf GELU, scalar output.
 * Heads are contiguous d_c/H_c = 32-wide chunks, scale 1/sqrt(32) (reading R10).
 * Kq: [nq][D] aggregated K at the live query positions, computed
 * by oracle_mean_key (reading R8).  nq == 0 or FLAG_NO_XATTN => c_j = 0 (R7).
 * Weight layout row-major [out][in]: wq[DC][3D+1], wk[DC][D], wv[DC][D],
 * fc1_w[HID][3D+1+DC], fc2_w[HID].
 * rule/kbar/s_out are indexed by candidate list entry c = 0..nc-1.
 * ---------------------------------------------------------------------- */
void oracle_residual(const double *rule, const double *kbar, int nc, const double *mbar,
                     const double *Kq, int nq, int D, const float *wq, const float *bq,
                     const float *wk, const float *bk, const float *wv, const float *bv,
                     const float *fc1_w, const float *fc1_b, const float *fc2_w,
                     const float *fc2_b, double alpha, int flags, double *s_out,
                     double *z_out /* optional [nc] */) {
  const int P = 3 * D + 1; /* |phi| */
  const int dh = DC / HC;
  if (alpha > 5.0) alpha = 5.0; /* "alpha in [-5,5] ... clipped at inference" PAPER.md:100 */
  if (alpha < -5.0) alpha = -5.0;
  if (flags & FLAG_NO_RESIDUAL) alpha = 0.0;
  const int use_x = !(flags & FLAG_NO_XATTN) && nq > 0;
  /* keys / values of the cross attention: Kc = W_K Kq + b_K, Vc = W_V Kq + b_V */
  double *Kc = (double *)calloc((size_t)(nq > 0 ? nq : 1) * DC, sizeof(double));
  double *Vc = (double *)calloc((size_t)(nq > 0 ? nq : 1) * DC, sizeof(double));
  for (int i = 0; i < nq; ++i)
    for (int o = 0; o < DC; ++o) {
      double ak = (double)bk[o], av = (double)bv[o];
      for (int d = 0; d < D; ++d) {
        ak += (double)wk[(int64_t)o * D + d] * Kq[(int64_t)i * D + d];
        av += (double)wv[(int64_t)o * D + d] * Kq[(int64_t)i * D + d];
      }
      Kc[(int64_t)i * DC + o] = ak;
      Vc[(int64_t)i * DC + o] = av;
    }
#pragma omp parallel for schedule(static)
  for (int c = 0; c < nc; ++c) {
    double phi[3 * 256 + 1 + DC]; /* phi (+) c ; D <= 256 */
    double Q[DC], hbuf[HID];
    for (int d = 0; d < D; ++d) {
      const double k = kbar[(int64_t)c * D + d];
      phi[d] = k;
      phi[D + d] = mbar[d];
      phi[2 * D + d] = k * mbar[d];
    }
    phi[3 * D] = rule[c];
    double *cj = phi + P;
    for (int o = 0; o < DC; ++o) cj[o] = 0.0;
    if (use_x) {
      for (int o = 0; o < DC; ++o) {
        double acc = (double)bq[o];
        for (int i = 0; i < P; ++i) acc += (double)wq[(int64_t)o * P + i] * phi[i];
        Q[o] = acc;
      }
      for (int hc = 0; hc < HC; ++hc) {
        double *logit = (double *)malloc(sizeof(double) * (size_t)nq);
        double mx = -INFINITY;
        for (int i = 0; i < nq; ++i) {
          double dot = 0.0;
          for (int e = 0; e < dh; ++e) dot += Q[hc * dh + e] * Kc[(int64_t)i * DC + hc * dh + e];
          logit[i] = dot / sqrt((double)dh);
          if (logit[i] > mx) mx = logit[i];
        }
        double den = 0.0;
        for (int i = 0; i < nq; ++i) den += exp(logit[i] - mx);
        for (int e = 0; e < dh; ++e) {
          double acc = 0.0;
          for (int i = 0; i < nq; ++i)
            acc += (exp(logit[i] - mx) / den) * Vc[(int64_t)i * DC + hc * dh + e];
          cj[hc * dh + e] = acc;
        }
        free(logit);
      }
    }
    /* MLP(phi (+) c) = fc2(GELU(fc1(.))) */
    const int IN = P + DC;
    for (int u = 0; u < HID; ++u) {
      double acc = (double)fc1_b[u];
      for (int i = 0; i < IN; ++i) acc += (double)fc1_w[(int64_t)u * IN + i] * phi[i];
      hbuf[u] = gelu_erf(acc);
    }
    double z = (double)fc2_b[0];
    for (int u = 0; u < HID; ++u) z += (double)fc2_w[u] * hbuf[u];
    if (z_out) z_out[c] = z;
    /* Eq. (4).  alpha == 0 or z == 0 adds an exact 0.0, so s_j == rule_j bit for bit */
    s_out[c] = rule[c] + alpha * z;
  }
  free(Kc);
  free(Vc);
}

/* ------------------------------------------------------------------------
 * O7  select.  PAPER.md:59-61, Eq. (1): K* = F U argtop_{|K|=C*} sum s_j with
 * C* = max(0, C - |F|); K = F U topk(A, max(0, C-|F|)).
 * Plain definition: fully sort the candidates by (score descending, position
 * ascending) and keep the first C* (reading R13: ties -> lower position wins;
 * -0.0 == +0.0; a NaN sorts below every number).  Scores are fp32: the
 * selection decision is taken in the precision the scores are stored in.
 * keep[j] = 1 for j in K*, else 0.   Skip rule ("skips compression
 * when N <= C", reading R15): every live position is kept.
 * ---------------------------------------------------------------------- */
typedef struct { float s; int32_t pos; } cand_t;

static int cand_cmp(const void *pa, const void *pb) {
  const cand_t *a = (const cand_t *)pa, *b = (const cand_t *)pb;
  const int an = isnan(a->s), bn = isnan(b->s);
  if (an != bn) return an ? 1 : -1;          /* NaN after every number */
  if (!an && a->s != b->s) return (a->s > b->s) ? -1 : 1; /* higher score first */
  return (a->pos < b->pos) ? -1 : (a->pos > b->pos); /* lower position first */
}

void oracle_select(const float *scores, const uint8_t *cls, int N, int C, uint8_t *keep,
                   int32_t *n_kept) {
  int nf = 0, nc = 0;
  for (int j = 0; j < N; ++j) {
    keep[j] = 0;
    if (cls[j] == CLS_FORCED) nf++;
    if (cls[j] == CLS_CAND) nc++;
  }
  if (N <= C) { /* no compression event */
    for (int j = 0; j < N; ++j) keep[j] = (cls[j] != CLS_DEAD);
    *n_kept = nf + nc;
    return;
  }
  int cstar = C - nf;
  if (cstar < 0) cstar = 0; /* reading R14: |F| > C keeps all of F and no candidate */
  if (cstar > nc) cstar = nc;
  cand_t *v = (cand_t *)malloc(sizeof(cand_t) * (size_t)(nc > 0 ? nc : 1));
  int k = 0;
  for (int j = 0; j < N; ++j)
    if (cls[j] == CLS_CAND) { v[k].s = scores[j]; v[k].pos = j; k++; }
  qsort(v, (size_t)nc, sizeof(cand_t), cand_cmp); /* comparator is a total order */
  for (int j = 0; j < N; ++j)
    if (cls[j] == CLS_FORCED) keep[j] = 1;
  for (int i = 0; i < cstar; ++i) keep[v[i].pos] = 1;
  *n_kept = nf + cstar;
  free(v);
}

/* ------------------------------------------------------------------------
 * O8  slot-map rewrite.  PAPER.md:121-126, Eq. (7): S[j] <- s+ for all
 * j in [0,N) \ K*, "with the token-id stream and sequence length N untouched";
 * kept rows stay at their slot.  PAPER.md:491: "persists a boolean valid mask,
 * redirects newly dropped positions to s+, and leaves all kept slot ids
 * unchanged".  Prefix-safe free: the old slot u = S[j] of a
 * newly dropped j is freed only if (a) j is outside the radix-protected prefix,
 * (b) u != s+, (c) u not in {S[i] : i in K*}.  Freed slots are reported once
 * each, in ascending order of the first dropped position that held them.
 * valid[j] = (S'[j] != s+).  K/V pools are never touched.
 * ---------------------------------------------------------------------- */
void oracle_rewrite(int32_t *S, int N, int32_t dead, const uint8_t *keep, int radix_len,
                    int64_t n_slots, uint8_t *valid, int32_t *freed, int32_t *n_freed) {
  uint8_t *kept_slot = (uint8_t *)calloc((size_t)n_slots, 1);
  uint8_t *seen = (uint8_t *)calloc((size_t)n_slots, 1);
  for (int j = 0; j < N; ++j)
    if (keep[j]) kept_slot[S[j]] = 1;
  int nf = 0;
  for (int j = 0; j < N; ++j) {
    if (keep[j]) { valid[j] = 1; continue; }
    const int32_t u = S[j];
    valid[j] = 0;
    if (u == dead) continue; /* was already dead: not "newly dropped" */
    S[j] = dead;
    if (j >= radix_len && u != dead && !kept_slot[u] && !seen[u]) {
      seen[u] = 1;
      freed[nf++] = u;
    }
  }
  *n_freed = nf;
  free(kept_slot);
  free(seen);
}

/* ------------------------------------------------------------------------
 * O9  decode attention through the slot map.  PAPER.md:130 (the sentinel "is
 * numerically equivalent to a hard visibility mask") and PAPER.md:359 ("the
 * flashinfer backend strips the sentinel before attention so decode reads only
 * the kept entries").  Plain definition (reading R16): for query head h,
 *   o_h = sum_{j : S[j] != s+} softmax_j(q_h . K[l, h div G, S[j]] * scale) V[l, h div G, S[j]].
 * q: [Hq][D] fp32 (exact up-conversion of the bf16 query); out: [Hq][D] double.
 * No live position => out = 0.
 * ---------------------------------------------------------------------- */
void oracle_decode(const void *k_pool, const void *v_pool, int kv_dtype, int64_t n_slots, int L,
                   int Hq, int Hkv, int D, int layer, const int32_t *S, int N, int32_t dead,
                   const float *q, double sm_scale, double *out) {
  (void)L;
  const int G = Hq / Hkv;
#pragma omp parallel for schedule(static)
  for (int h = 0; h < Hq; ++h) {
    const int kvh = h / G;
    double *x = (double *)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double mx = -INFINITY;
    for (int j = 0; j < N; ++j) {
      if (S[j] == dead) continue;
      double dot = 0.0;
      for (int d = 0; d < D; ++d)
        dot += (double)q[(int64_t)h * D + d] *
               pool_elem(k_pool, kv_dtype, pool_index(n_slots, Hkv, D, layer, S[j], kvh, d));
      x[j] = dot * sm_scale;
      if (x[j] > mx) mx = x[j];
    }
    double den = 0.0;
    for (int j = 0; j < N; ++j)
      if (S[j] != dead) den += exp(x[j] - mx);
    for (int d = 0; d < D; ++d) {
      double acc = 0.0;
      for (int j = 0; j < N; ++j)
        if (S[j] != dead)
          acc += (exp(x[j] - mx) / den) *
                 pool_elem(v_pool, kv_dtype, pool_index(n_slots, Hkv, D, layer, S[j], kvh, d));
      out[(int64_t)h * D + d] = acc;
    }
    free(x);
  }
}

/* Variant used only by the side test of reading R16: attend to
 * EVERY position, dead ones included, reading whatever the pool holds at s+
 * (K = -1e4, V = 0 as initialised).  Same arithmetic, no skip. */
void oracle_decode_attend_all(const void *k_pool, const void *v_pool, int kv_dtype,
                              int64_t n_slots, int L, int Hq, int Hkv, int D, int layer,
                              const int32_t *S, int N, const float *q, double sm_scale,
                              double *out) {
  /* a dead value that never matches any slot id */
  oracle_decode(k_pool, v_pool, kv_dtype, n_slots, L, Hq, Hkv, D, layer, S, N, (int32_t)-1, q,
                sm_scale, out);
}

/* ------------------------------------------------------------------------
 * Composite: one scoring call, as the compression event of PAPER.md:489-491
 * orders it.  scores[N] fp32 (rounded once from double): +INF at forced live
 * positions, -INF at dead positions (reading R6), s_j at candidates.
 * mode: 0 = memory (rule only), 1 = learnable (rule + residual).  The "query"
 * mode is the same call with M = oracle_query_encoding(...).
 * xattn_pos: positions forming Kq; dead ones are filtered.
 * ---------------------------------------------------------------------- */
void oracle_score(const void *k_pool, int kv_dtype, int64_t n_slots, int L, int Hq, int Hkv, int D,
                  const double *M, const int32_t *S, int N, int32_t dead, int pi, int qs, int qe,
                  int mode, int flags, const int32_t *xattn_pos, int n_xattn, const float *wq,
                  const float *bq, const float *wk, const float *bk, const float *wv,
                  const float *bv, const float *fc1_w, const float *fc1_b, const float *fc2_w,
                  const float *fc2_b, double alpha, float *scores, double *rule_out /* opt [N] */) {
  uint8_t *cls = (uint8_t *)malloc((size_t)(N > 0 ? N : 1));
  int32_t counts[3];
  oracle_partition(S, N, dead, pi, qs, qe, cls, counts);
  double *rule = (double *)calloc((size_t)(N > 0 ? N : 1), sizeof(double));
  oracle_rule_score(k_pool, kv_dtype, n_slots, L, Hq, Hkv, D, M, S, cls, N, rule, NULL);
  if (rule_out) memcpy(rule_out, rule, sizeof(double) * (size_t)N);
  const int nc = counts[CLS_CAND];
  double *s = (double *)malloc(sizeof(double) * (size_t)(nc > 0 ? nc : 1));
  int32_t *cpos = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nc > 0 ? nc : 1));
  double *rc = (double *)malloc(sizeof(double) * (size_t)(nc > 0 ? nc : 1));
  int k = 0;
  for (int j = 0; j < N; ++j)
    if (cls[j] == CLS_CAND) { cpos[k] = j; rc[k] = rule[j]; k++; }
  if (mode == 1) {
    double *kbar = (double *)malloc(sizeof(double) * (size_t)(nc > 0 ? nc : 1) * D);
    double *mbar = (double *)malloc(sizeof(double) * (size_t)D);
    oracle_mean_key(k_pool, kv_dtype, n_slots, L, Hq, Hkv, D, S, cpos, nc, kbar);
    oracle_mean_memory(M, L, Hq, D, mbar);
    int32_t *qpos = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_xattn > 0 ? n_xattn : 1));
    int nq = 0;
    for (int i = 0; i < n_xattn; ++i)
      if (xattn_pos[i] >= 0 && xattn_pos[i] < N && S[xattn_pos[i]] != dead) qpos[nq++] = xattn_pos[i];
    double *Kq = (double *)malloc(sizeof(double) * (size_t)(nq > 0 ? nq : 1) * D);
    oracle_mean_key(k_pool, kv_dtype, n_slots, L, Hq, Hkv, D, S, qpos, nq, Kq);
    oracle_residual(rc, kbar, nc, mbar, Kq, nq, D, wq, bq, wk, bk, wv, bv, fc1_w, fc1_b, fc2_w,
                    fc2_b, alpha, flags, s, NULL);
    free(kbar); free(mbar); free(qpos); free(Kq);
  } else {
    for (int c = 0; c < nc; ++c) s[c] = rc[c];
  }
  for (int j = 0; j < N; ++j)
    scores[j] = (cls[j] == CLS_FORCED) ? INFINITY : -INFINITY;
  for (int c = 0; c < nc; ++c) scores[cpos[c]] = (float)s[c];
  free(cls); free(rule); free(s); free(cpos); free(rc);
}

/* number of trainable parameters of the residual head for head dim D
 * (214,274 at D=128) -- counted from the topology above. */
int64_t oracle_residual_param_count(int D) {
  const int64_t P = 3 * (int64_t)D + 1;
  return (P * DC + DC)            /* W_Q, b_Q */
         + 2 * ((int64_t)D * DC + DC) /* W_K, b_K, W_V, b_V */
         + ((P + DC) * HID + HID) /* fc1 */
         + (HID + 1)              /* fc2 */
         + 1;                     /* alpha */
}
