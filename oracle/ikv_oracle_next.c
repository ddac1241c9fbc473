/*
 * ikv_oracle_next.c -- CPU ORACLE for the SURVEY 8(f) follow-ups.  TEST INFRASTRUCTURE ONLY.
 *
 * Same rules as ikv_oracle.c: plain C, every floating-point step in IEEE double, inputs
 * up-converted exactly, no blocking or fusion, OpenMP only around outermost independent
 * loops.  Shares no code with the CUDA path.  Written from /root/reference/PAPER.md; the
 * paper gives these items only by name and parameters, so each function states the reading
 * it implements (R28-R32).
 *
 *   N1  multi-row scorer            PAPER.md:91 ("SnapKV's window of W tail Q rows",
 *                                   O(W L H_q N)), :159 ("tail window W=32"), :310
 *   N2  prefill attention + reads   PAPER.md:55 (the event follows prefill), :163-175
 *                                   (Raw KV Reads sum |R_t|, Eff. KV Reads sum |K_t|)
 *   N3  baseline scorers            PAPER.md:161, :310 (StreamingLLM sink 4 + recent window;
 *                                   SnapKV W=32, kernel 7, max-pool; H2O ratio mode with a
 *                                   recent-window floor), :359 (shared dead-slot substrate)
 *
 * Pins: tests/test_oracle_next.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define IKV_O_BF16 1
#define CLS_DEAD 0
#define CLS_FORCED 1
#define CLS_CAND 2

static double bf16_to_double(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, sizeof f);
  return (double)f;
}
static double pool_elem(const void *pool, int dtype, int64_t idx) {
  if (dtype == IKV_O_BF16) return bf16_to_double(((const uint16_t *)pool)[idx]);
  return (double)((const float *)pool)[idx];
}
static int64_t pool_index(int64_t n_slots, int Hkv, int D, int l, int64_t slot, int kvh, int d) {
  return (((int64_t)l * n_slots + slot) * Hkv + kvh) * D + d;
}

/* ------------------------------------------------------------------------
 * N1  multi-row scorer (reading R28).  R un-collapsed rows per (layer, query head),
 * rows[r][l][h][:] used as given (no decay, no normalisation); every row is its own
 * softmax over the candidates; the rows are combined with weights w_r:
 *   a_{r,l,h,j} = softmax_{i in A}( rows[r,l,h] . K[l, h div G, S[i]] / sqrt(D) )_j
 *   s_j         = sum_r w_r sum_{l,h} a_{r,l,h,j}
 * R = 1, w = 1, rows[0] = M_t is Eq. (3).  out: [N], 0 outside the candidates.
 * ---------------------------------------------------------------------- */
void oracle_multirow_score(const void *k_pool, int kv_dtype, int64_t n_slots, int L, int Hq, int Hkv,
                           int D, const double *rows, int R, const double *w, const int32_t *S,
                           const uint8_t *cls, int N, double *out) {
  const int G = Hq / Hkv;
  const double inv_sqrt_d = 1.0 / sqrt((double)D);
  const int64_t LH = (int64_t)L * Hq;
  for (int j = 0; j < N; ++j) out[j] = 0.0;
  double *a = (double *)malloc(sizeof(double) * (size_t)LH * (size_t)(N > 0 ? N : 1));
  for (int r = 0; r < R; ++r) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t lh = 0; lh < LH; ++lh) {
      const int l = (int)(lh / Hq), h = (int)(lh % Hq), kvh = h / G;
      const double *m = rows + ((int64_t)r * LH + lh) * D;
      double *x = a + lh * N;
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
      double denom = 0.0;
      for (int j = 0; j < N; ++j)
        if (cls[j] == CLS_CAND) denom += exp(x[j] - xmax);
      for (int j = 0; j < N; ++j) x[j] = (cls[j] == CLS_CAND) ? exp(x[j] - xmax) / denom : 0.0;
    }
#pragma omp parallel for schedule(static)
    for (int j = 0; j < N; ++j) {
      if (cls[j] != CLS_CAND) continue;
      double s = 0.0;
      for (int64_t lh = 0; lh < LH; ++lh) s += a[lh * N + j];
      out[j] += w[r] * s;
    }
  }
  free(a);
}

/* ------------------------------------------------------------------------
 * N3a  max-pool smoothing (SnapKV "kernel 7 ... max-pool"; reading R29):
 * pooled_j = max over candidate positions i with |i - j| <= (kernel-1)/2 of s_i.  The window
 * runs over LOGICAL positions; positions that are not candidates (dead, forced) do not
 * take part.  out: [N]; non-candidates keep their input value.
 * ---------------------------------------------------------------------- */
void oracle_maxpool_candidates(const double *s, const uint8_t *cls, int N, int kernel, double *out) {
  const int half = (kernel - 1) / 2;
  for (int j = 0; j < N; ++j) {
    out[j] = s[j];
    if (cls[j] != CLS_CAND) continue;
    double m = s[j];
    for (int i = j - half; i <= j + half; ++i)
      if (i >= 0 && i < N && cls[i] == CLS_CAND && s[i] > m) m = s[i];
    out[j] = m;
  }
}

/* ------------------------------------------------------------------------
 * N3b  StreamingLLM scores (sink + recent window; reading R30): a
 * candidate at position j < n_sink scores 2^30 (attention sinks are kept first), any
 * other candidate scores its position j, so that top-C* keeps the most recent ones.
 * out: [N], 0 outside the candidates.
 * ---------------------------------------------------------------------- */
void oracle_streaming_scores(const uint8_t *cls, int N, int n_sink, double *out) {
  for (int j = 0; j < N; ++j)
    out[j] = (cls[j] != CLS_CAND) ? 0.0 : (j < n_sink ? 1073741824.0 : (double)j);
}

/* ------------------------------------------------------------------------
 * N3c  H2O scores (heavy hitters, "ratio mode with a recent-window floor", PAPER.md:161,
 * :310; reading R31).  hh_j = accumulated attention mass of candidate j (N1 over the bank
 * of past query rows, weights 1).  With C* = max(0, C - |F|) the n_recent =
 * min(C*, max(floor, round(ratio C*))) most recent candidates score 1e30 + j (always
 * kept), the others their mass.  out: [N]; non-candidates keep hh.
 * ---------------------------------------------------------------------- */
void oracle_h2o_scores(const double *hh, const uint8_t *cls, int N, int C, double ratio, int floor_,
                       double *out) {
  int nF = 0, nC = 0;
  for (int j = 0; j < N; ++j) {
    if (cls[j] == CLS_FORCED) ++nF;
    if (cls[j] == CLS_CAND) ++nC;
  }
  const int cstar = (C - nF) > 0 ? (C - nF) : 0;
  int n_recent = (int)floor(ratio * (double)cstar + 0.5);
  if (n_recent < floor_) n_recent = floor_;
  if (n_recent > cstar) n_recent = cstar;
  int seen = 0;
  for (int j = N - 1; j >= 0; --j) {
    out[j] = hh[j];
    if (cls[j] != CLS_CAND) continue;
    if (seen < n_recent) out[j] = 1.0e30 + (double)j;
    ++seen;
  }
  (void)nC;
}

/* ------------------------------------------------------------------------
 * N2  prefill / chunked-prefill attention through the slot map (reading R32): n_q query
 * rows at logical positions q_pos0 .. q_pos0 + n_q - 1; row i attends, causally, every
 * position j <= q_pos0 + i with S[j] != s+ (dead entries skipped exactly as in decode,
 * PAPER.md:130, :359):
 *   o_{i,h} = sum_j softmax_j( q_{i,h} . K[l, h div G, S[j]] * scale ) V[l, h div G, S[j]].
 * reads[0] += sum_i (q_pos0 + i + 1)        -- Raw KV Reads  sum |R_t|
 * reads[1] += sum_i #{j <= q_pos0 + i : S[j] != s+}   -- Eff. KV Reads  sum |K_t|
 * q: [n_q][Hq][D] fp32; out: [n_q][Hq][D] double.
 * ---------------------------------------------------------------------- */
void oracle_prefill(const void *k_pool, const void *v_pool, int kv_dtype, int64_t n_slots, int Hq,
                    int Hkv, int D, int layer, const int32_t *S, int32_t dead, int q_pos0, int n_q,
                    const float *q, double sm_scale, double *out, int64_t *reads) {
  const int G = Hq / Hkv;
  for (int i = 0; i < n_q; ++i) {
    const int last = q_pos0 + i;
    int live = 0;
    for (int j = 0; j <= last; ++j)
      if (S[j] != dead) ++live;
    reads[0] += (int64_t)last + 1;
    reads[1] += live;
  }
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
  for (int i = 0; i < n_q; ++i)
    for (int h = 0; h < Hq; ++h) {
      const int last = q_pos0 + i, kvh = h / G;
      const float *qr = q + ((int64_t)i * Hq + h) * D;
      double *x = (double *)malloc(sizeof(double) * (size_t)(last + 1));
      double mx = -INFINITY;
      for (int j = 0; j <= last; ++j) {
        if (S[j] == dead) continue;
        double dot = 0.0;
        for (int d = 0; d < D; ++d)
          dot += (double)qr[d] * pool_elem(k_pool, kv_dtype, pool_index(n_slots, Hkv, D, layer, S[j], kvh, d));
        x[j] = dot * sm_scale;
        if (x[j] > mx) mx = x[j];
      }
      double den = 0.0;
      for (int j = 0; j <= last; ++j)
        if (S[j] != dead) den += exp(x[j] - mx);
      for (int d = 0; d < D; ++d) {
        double acc = 0.0;
        for (int j = 0; j <= last; ++j)
          if (S[j] != dead)
            acc += (exp(x[j] - mx) / den) *
                   pool_elem(v_pool, kv_dtype, pool_index(n_slots, Hkv, D, layer, S[j], kvh, d));
        out[((int64_t)i * Hq + h) * D + d] = acc;
      }
      free(x);
    }
}

/* ------------------------------------------------------------------------
 * N4  training objective of the residual head, Eq. 8, and its gradient
 * with respect to the scores (readings R34-R37):
 *   L = L_BCE(s, y) + rho L_rank + gamma mean sigma(s) + eta (||M_t||_2 - 1)^2
 * s[n]: scores (logits) of the candidate tokens of one (session, turn) row; y[n]: 1 = positive
 * ("matches a literal substring of a future tool argument"), 0 = negative, anything else
 * (-100) = excluded from the loss.  V = valid entries, n_v = |V|, P = positives.
 *   p = |P| / n_v,  p~ = clip(p, 0.02, 0.5),  w+ = (1 - p~) / p~                        (:147)
 *   L_BCE  = (1/n_v) sum_V [ w+ y softplus(-s) + (1 - y) softplus(s) ]
 *   L_rank = (1 / (|P| |H|)) sum_{i in P} sum_{j in H} softplus(s_j - s_i),
 *            H = the 64 highest-scored negatives (ties: lower position first); 0 if P or H is empty
 *   keep   = (1/n_v) sum_V sigma(s)
 *   norm   = mean over the rows r of mem_rows[R][D] of (||row_r||_2 - 1)^2   (0 if R = 0)
 * terms[5] = {L, L_BCE, L_rank, keep, norm} (L_rank, keep, norm unweighted); grad[n] = dL/ds
 * (0 at excluded entries).  n_v = 0: everything 0 except the norm term.
 * ---------------------------------------------------------------------- */
static double softplus_d(double x) { return x > 0 ? x + log1p(exp(-x)) : log1p(exp(x)); }
static double sigmoid_d(double x) { return x >= 0 ? 1.0 / (1.0 + exp(-x)) : exp(x) / (1.0 + exp(x)); }

void oracle_train_loss(const double *s, const int32_t *y, int n, const double *mem_rows, int R, int D,
                       double rho, double gamma, double eta, double *terms, double *grad) {
  int n_v = 0, n_p = 0;
  for (int i = 0; i < n; ++i) {
    grad[i] = 0.0;
    if (y[i] == 0 || y[i] == 1) { ++n_v; n_p += y[i]; }
  }
  double bce = 0.0, rank = 0.0, keep = 0.0, norm = 0.0;
  if (n_v > 0) {
    double p = (double)n_p / (double)n_v;
    double pt = p < 0.02 ? 0.02 : (p > 0.5 ? 0.5 : p);
    const double wp = (1.0 - pt) / pt;
    for (int i = 0; i < n; ++i) {
      if (y[i] != 0 && y[i] != 1) continue;
      if (y[i] == 1) {
        bce += wp * softplus_d(-s[i]);
        grad[i] += -wp * sigmoid_d(-s[i]) / n_v;
      } else {
        bce += softplus_d(s[i]);
        grad[i] += sigmoid_d(s[i]) / n_v;
      }
      const double sg = sigmoid_d(s[i]);
      keep += sg;
      grad[i] += gamma * sg * (1.0 - sg) / n_v;
    }
    bce /= n_v;
    keep /= n_v;
    /* hard negatives: repeatedly take the best remaining negative */
    int hn[64], n_h = 0;
    char *taken = (char *)calloc((size_t)n, 1);
    for (int k = 0; k < 64; ++k) {
      int best = -1;
      for (int i = 0; i < n; ++i)
        if (y[i] == 0 && !taken[i] && (best < 0 || s[i] > s[best])) best = i;  /* lower position wins ties */
      if (best < 0) break;
      taken[best] = 1;
      hn[n_h++] = best;
    }
    free(taken);
    if (n_p > 0 && n_h > 0) {
      const double c = 1.0 / ((double)n_p * (double)n_h);
      for (int i = 0; i < n; ++i) {
        if (y[i] != 1) continue;
        for (int k = 0; k < n_h; ++k) {
          const double z = s[hn[k]] - s[i];
          rank += softplus_d(z);
          const double gz = sigmoid_d(z) * c * rho;
          grad[hn[k]] += gz;
          grad[i] -= gz;
        }
      }
      rank *= c;
    }
  }
  for (int r = 0; r < R; ++r) {
    double q = 0.0;
    for (int d = 0; d < D; ++d) q += mem_rows[(int64_t)r * D + d] * mem_rows[(int64_t)r * D + d];
    const double e = sqrt(q) - 1.0;
    norm += e * e;
  }
  if (R > 0) norm /= R;
  terms[1] = bce; terms[2] = rank; terms[3] = keep; terms[4] = norm;
  terms[0] = bce + rho * rank + gamma * keep + eta * norm;
}
