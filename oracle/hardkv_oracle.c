/*
 * hardkv_oracle.c -- TEST INFRASTRUCTURE ONLY (see hardkv_oracle.h).
 *
 * Plain nested loops in the paper's order.  No blocking, no fusion, no SIMD
 * intrinsics; the only library routines are exp/log/ceil/nearbyint and qsort.
 * Citations are PAPER.md line numbers (L...) and DESIGN.md readings (C...).
 */
#include "hardkv_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static uint32_t f32_bits(float x) { uint32_t b; memcpy(&b, &x, 4); return b; }

/* Pool = Tier-2 address range [c_lo, n-W) (L72, DESIGN "tiers"); empty if n-W <= c_lo. */
static int32_t pool_hi(const hko_config *c, const hko_unit *u) {
  int32_t hi = u->n - c->recent;
  return hi > u->c_lo ? hi : u->c_lo;
}

/* ---- Step 1 (L78): "linearly append KV pairs to the Tier 1 Dense Cache" -------- */
void hko_append(const hko_config *c, hko_unit *u, const float *k_new, const float *v_new) {
  memcpy(u->K + (size_t)u->n * c->d, k_new, sizeof(float) * c->d);
  memcpy(u->V + (size_t)u->n * c->d, v_new, sizeof(float) * c->d);
  u->n += 1;
}

/* ---- Step 4 (L78) / Tier 3 (L76) / vote ranking (L86), reading C7 --------------
 * While the pool exceeds l_upper, its oldest token t = c_lo retires.  The
 * condensed tier has C_cap constant slots; a free slot takes t; otherwise the
 * resident with the lexicographically smallest (votes, pos) is the candidate
 * victim and t replaces it iff votes[t] >= its votes (t is newer, so it wins
 * ties); else t is evicted for good. */
/* Store rounding of a merged row element: the tier holds kv_dtype values, so a bf16 tier
 * rounds the exact (fp64) combination once, to nearest-even, to 8 significant bits. */
static float hko_store_round(const hko_config *c, double x) {
  if (!c->kv_bf16 || x == 0.0 || !isfinite(x)) return (float)x;
  int e;
  double m = frexp(x, &e);                       /* x = m 2^e, 0.5 <= |m| < 1 */
  return (float)ldexp(nearbyint(m * 256.0), e - 8);
}

/* ---- LSE-preserving weighted merging (Appendix G, Eq. 9 / Thm G.1; reading
 * C17): the evictee e is not dropped but folded into the resident a with the highest
 * score under the current queries ("let q K_j >> q K_k", Eq. 11), with the softmax
 * weights of the pair:  K_hat = w_a K_a + w_e K_e,  w_a = e^{x_a} / (e^{x_a} + e^{x_e}),
 * x = group mean of sm_scale q_g . K (one pair of weights per KV head); V takes the same
 * weights (the paper leaves g(V_j, V_k) open, L806-811).  pos / votes of a are unchanged. */
static void hko_merge_evictee(const hko_config *c, hko_unit *u, const float *q,
                              const float *Ke, const float *Ve) {
  if (u->cond_count <= 0) return;
  int32_t a = 0;
  double xa = -INFINITY, xe = 0.0;
  for (int32_t r = 0; r < u->cond_count; ++r) {
    double x = 0.0;
    for (int32_t g = 0; g < c->G; ++g) {
      double dot = 0.0;
      for (int32_t e = 0; e < c->d; ++e)
        dot += (double)q[(size_t)g * c->d + e] * (double)u->cond_k[(size_t)r * c->d + e];
      x += (double)c->sm_scale * dot;
    }
    x /= (double)c->G;
    if (x > xa) { xa = x; a = r; }               /* ties: the lowest slot */
  }
  for (int32_t g = 0; g < c->G; ++g) {
    double dot = 0.0;
    for (int32_t e = 0; e < c->d; ++e) dot += (double)q[(size_t)g * c->d + e] * (double)Ke[e];
    xe += (double)c->sm_scale * dot;
  }
  xe /= (double)c->G;
  double wa = 1.0 / (1.0 + exp(xe - xa)), we = 1.0 - wa;
  for (int32_t e = 0; e < c->d; ++e) {
    float *ka = u->cond_k + (size_t)a * c->d + e, *va = u->cond_v + (size_t)a * c->d + e;
    *ka = hko_store_round(c, wa * (double)*ka + we * (double)Ke[e]);
    *va = hko_store_round(c, wa * (double)*va + we * (double)Ve[e]);
  }
}

int hko_retire_q(const hko_config *c, hko_unit *u, const float *q) {
  int retired = 0;
  float *ek = (float *)malloc(sizeof(float) * (size_t)c->d), *ev = (float *)malloc(sizeof(float) * (size_t)c->d);
  while (u->n - c->recent - u->c_lo > u->l_upper) {
    int32_t t = u->c_lo;
    int32_t slot = -1;
    int have_evictee = 0;
    if (u->cond_count < c->cond_cap) {
      slot = u->cond_count;
      u->cond_count += 1;
    } else if (c->cond_cap > 0) {
      int32_t m = 0;
      for (int32_t j = 1; j < c->cond_cap; ++j) {
        if (u->cond_votes[j] < u->cond_votes[m] ||
            (u->cond_votes[j] == u->cond_votes[m] && u->cond_pos[j] < u->cond_pos[m]))
          m = j;
      }
      if (u->votes[t] >= u->cond_votes[m]) {
        slot = m;                                  /* the displaced resident is the evictee */
        memcpy(ek, u->cond_k + (size_t)m * c->d, sizeof(float) * c->d);
        memcpy(ev, u->cond_v + (size_t)m * c->d, sizeof(float) * c->d);
      } else {                                     /* the newcomer itself is the evictee */
        memcpy(ek, u->K + (size_t)t * c->d, sizeof(float) * c->d);
        memcpy(ev, u->V + (size_t)t * c->d, sizeof(float) * c->d);
      }
      have_evictee = 1;
    }
    if (slot >= 0) {
      memcpy(u->cond_k + (size_t)slot * c->d, u->K + (size_t)t * c->d, sizeof(float) * c->d);
      memcpy(u->cond_v + (size_t)slot * c->d, u->V + (size_t)t * c->d, sizeof(float) * c->d);
      u->cond_pos[slot] = t;
      u->cond_votes[slot] = u->votes[t];
    }
    if (have_evictee && c->cond_merge && q) hko_merge_evictee(c, u, q, ek, ev);
    u->c_lo += 1;
    retired += 1;
  }
  free(ek); free(ev);
  /* a compression step re-anchors the dense tier at sinks + the last W tokens (L71, L276-277) */
  {
    int32_t s_end = c->sink < u->n ? c->sink : u->n;
    int32_t r_lo = u->n - c->recent;
    u->dense_lo = r_lo > s_end ? r_lo : s_end;
  }
  return retired;
}

int hko_retire(const hko_config *c, hko_unit *u) { return hko_retire_q(c, u, NULL); }

/* ---- score: exponent of Eq. 4 (L735-739) with the scale of reading C1 ---------- */
void hko_score(const hko_config *c, hko_unit *u, const float *q) {
  int32_t hi = pool_hi(c, u);
  for (int32_t g = 0; g < c->G; ++g) {
    for (int32_t i = u->c_lo; i < hi; ++i) {
      double dot = 0.0;
      for (int32_t e = 0; e < c->d; ++e)
        dot += (double)q[(size_t)g * c->d + e] * (double)u->K[(size_t)i * c->d + e];
      u->logits[(size_t)g * c->max_ctx + i] = (float)((double)c->sm_scale * dot);
    }
  }
}

/* ---- metric transform g(z) of one query head (Appendix E "Reduce-Scatter", L278):
 * SNAPKV (score_mode 2) max-pools the raw logits along the sequence with an odd
 * window pool_kernel, stride 1, clipped to the pool (reading C15); every other mode
 * is the identity (VANILLA, L276).  zhat has N = hi - lo entries. */
static void hko_metric_logits(const hko_config *c, const hko_unit *u, int32_t g, int mode, double *zhat) {
  int32_t lo = u->c_lo, hi = pool_hi(c, u);
  const float *z = u->logits + (size_t)g * c->max_ctx;
  int32_t r = (mode == 2 && c->pool_kernel > 1) ? (c->pool_kernel - 1) / 2 : 0;
  for (int32_t i = lo; i < hi; ++i) {
    double m = (double)z[i];
    for (int32_t j = i - r; j <= i + r; ++j)
      if (j >= lo && j < hi && (double)z[j] > m) m = (double)z[j];
    zhat[i - lo] = m;
  }
}

/* P[i] = (1/G) sum_g softmax_i(g(z_g)[i] / T) over the pool: Solution 1, L120
 * ("S_hat = S(g(z/T))"; for max-pooling g(z/T) = g(z)/T exactly when T > 0), group
 * mean of reading C2, softmax over the pool only (reading C3). */
static void hko_metric_probs(const hko_config *c, const hko_unit *u, int mode, double T, double *P) {
  int32_t lo = u->c_lo, hi = pool_hi(c, u), N = hi - lo;
  double *zh = (double *)malloc(sizeof(double) * (size_t)N);
  for (int32_t i = 0; i < N; ++i) P[i] = 0.0;
  for (int32_t g = 0; g < c->G; ++g) {
    hko_metric_logits(c, u, g, mode, zh);
    double m = -INFINITY;
    for (int32_t i = 0; i < N; ++i) { double x = zh[i] / T; if (x > m) m = x; }
    double s = 0.0;
    for (int32_t i = 0; i < N; ++i) s += exp(zh[i] / T - m);
    for (int32_t i = 0; i < N; ++i) P[i] += exp(zh[i] / T - m) / s;
  }
  for (int32_t i = 0; i < N; ++i) P[i] /= (double)c->G;
  free(zh);
}

/* ---- query cache (L448: "for decoding-time KV cache compression, we store the query cache in a sliding
 * window"): the queries of the last accum_window decode steps of this head's GQA group. */
void hko_qcache_push(const hko_config *c, hko_unit *u, const float *q) {
  if (!u->qcache || c->accum_window <= 0) return;
  memcpy(u->qcache + (size_t)u->qc_slot * c->G * c->d, q, sizeof(float) * (size_t)c->G * c->d);
  u->qc_slot = (u->qc_slot + 1) % c->accum_window;
  if (u->qc_count < c->accum_window) u->qc_count += 1;
}

/* ---- accumulated attention recomputed from the query cache (reading C18; "vanilla attention averaging in
 * H2O" is an order-preserving g, Solution 1, L122-124): every cached query scores the CURRENT pool,
 *   A(i) = sum over cached steps tau, heads g of softmax_i(sm_scale q_{tau,g} . k_i / T) / G,   P_hat = A / sum_i A,
 * plain loops: one logit row per (tau, g), its softmax over the pool, added up in fp64, rounded once. */
static void hko_calibrate_qcache(const hko_config *c, hko_unit *u) {
  int32_t lo = u->c_lo, hi = pool_hi(c, u), N = hi - lo;
  double *A = (double *)calloc((size_t)N, sizeof(double));
  double *z = (double *)malloc(sizeof(double) * (size_t)N);
  for (int32_t tau = 0; tau < u->qc_count; ++tau) {
    for (int32_t g = 0; g < c->G; ++g) {
      const float *q = u->qcache + ((size_t)tau * c->G + g) * c->d;
      double m = -INFINITY, s = 0.0;
      for (int32_t i = 0; i < N; ++i) {
        double dot = 0.0;
        for (int32_t e = 0; e < c->d; ++e) dot += (double)q[e] * (double)u->K[(size_t)(lo + i) * c->d + e];
        z[i] = (double)c->sm_scale * dot / (double)u->T;
        if (z[i] > m) m = z[i];
      }
      for (int32_t i = 0; i < N; ++i) s += exp(z[i] - m);
      for (int32_t i = 0; i < N; ++i) A[i] += exp(z[i] - m) / s / (double)c->G;
    }
  }
  double tot = 0.0;
  for (int32_t i = 0; i < N; ++i) tot += A[i];
  for (int32_t i = 0; i < N; ++i) u->probs[lo + i] = tot > 0.0 ? (float)(A[i] / tot) : 0.0f;
  free(A); free(z);
}

/* ---- Logits Calibration, apply-T (L120 "S_hat = S(g(z/T))", g = identity for
 * VANILLA L276, sequence max-pool for SNAPKV L278; H2O-style averaging L124 for
 * ACCUM, reading C4).  One score per KV head = mean over the GQA group of
 * per-query-head softmax probabilities (reading C2), softmax taken over the pool
 * only (reading C3). */
void hko_calibrate(const hko_config *c, hko_unit *u) {
  int32_t lo = u->c_lo, hi = pool_hi(c, u);
  if (hi <= lo) return;
  if (u->score_mode == 3) { hko_calibrate_qcache(c, u); return; }
  double *P = (double *)calloc((size_t)(hi - lo), sizeof(double));
  hko_metric_probs(c, u, u->score_mode, (double)u->T, P);

  if (u->score_mode != 1) {
    for (int32_t i = lo; i < hi; ++i) u->probs[i] = (float)P[i - lo];
  } else {
    /* ACCUM (reading C4): sliding sum of the last accum_window per-step rows, kept
     * incrementally: acc <- max(0, acc - ring[slot] + P_t); ring[slot] <- P_t;
     * then renormalised over the current pool. acc and ring are fp32 state. */
    float *ring = u->ring + (size_t)u->ring_slot * c->max_ctx;
    double tot = 0.0;
    for (int32_t i = lo; i < hi; ++i) {
      float pt = (float)P[i - lo];
      double a = ((double)u->acc[i] - (double)ring[i]) + (double)pt;
      if (a < 0.0) a = 0.0;
      u->acc[i] = (float)a;
      ring[i] = pt;
      tot += (double)u->acc[i];
    }
    u->ring_slot = (u->ring_slot + 1) % c->accum_window;
    for (int32_t i = lo; i < hi; ++i)
      u->probs[i] = tot > 0.0 ? (float)((double)u->acc[i] / tot) : 0.0f;
  }
  free(P);
}

/* ---- Top-p nucleus (L108: "Top-p sampling over {S_i} yield k tokens"), made a
 * single well-defined result by reading C5: integer mass w_i = rn(P_i * 2^32),
 * total order (P as fp32 bit pattern descending, position ascending), shortest
 * prefix whose mass >= Theta = ceil(p * Wtot).  Reading C6: k = min(k_topp, k_cap),
 * the clamp keeps the best of the same order (L233 "k as the maximum block usage
 * for Top-p pruned each head"). */
typedef struct { uint32_t bits; int32_t pos; } hko_key;
static int hko_key_cmp(const void *a, const void *b) {
  const hko_key *x = (const hko_key *)a, *y = (const hko_key *)b;
  if (x->bits != y->bits) return x->bits > y->bits ? -1 : 1;   /* P descending  */
  if (x->pos != y->pos) return x->pos < y->pos ? -1 : 1;       /* pos ascending */
  return 0;
}
static int hko_i32_cmp(const void *a, const void *b) {
  int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
  return (x > y) - (x < y);
}

void hko_topp_select(const hko_config *c, hko_unit *u, float p, int count_votes) {
  int32_t lo = u->c_lo, hi = pool_hi(c, u);
  int32_t N = hi - lo;
  for (int32_t j = 0; j < c->k_cap; ++j) u->sel_idx[j] = -1;
  u->sel_count = 0; u->k_topp = 0; u->tau_bits = 0;
  if (N <= 0) return;

  hko_key *keys = (hko_key *)malloc(sizeof(hko_key) * (size_t)N);
  for (int32_t i = 0; i < N; ++i) { keys[i].bits = f32_bits(u->probs[lo + i]); keys[i].pos = lo + i; }
  qsort(keys, (size_t)N, sizeof(hko_key), hko_key_cmp);   /* total order: no ties left */

  int32_t k_topp;
  if (p >= 1.0f || N <= u->l_lower) {
    k_topp = N;                                      /* no sparsity yet (L197, C8) */
  } else {
    uint64_t Wtot = 0;
    for (int32_t i = 0; i < N; ++i)
      Wtot += (uint64_t)nearbyint((double)u->probs[lo + i] * 4294967296.0);
    uint64_t Theta = (uint64_t)ceil((double)p * (double)Wtot);
    if (Theta < 1) Theta = 1;
    uint64_t cum = 0;
    k_topp = N;
    for (int32_t j = 0; j < N; ++j) {
      float Pj; memcpy(&Pj, &keys[j].bits, 4);
      cum += (uint64_t)nearbyint((double)Pj * 4294967296.0);
      if (cum >= Theta) { k_topp = j + 1; break; }
    }
  }
  int32_t k = k_topp < c->k_cap ? k_topp : c->k_cap;
  u->k_topp = k_topp;
  u->sel_count = k;
  if (k > 0) u->tau_bits = keys[k - 1].bits;
  for (int32_t j = 0; j < k; ++j) u->sel_idx[j] = keys[j].pos;
  qsort(u->sel_idx, (size_t)k, sizeof(int32_t), hko_i32_cmp);   /* I ascending (C9) */
  if (count_votes)
    for (int32_t j = 0; j < k; ++j) u->votes[u->sel_idx[j]] += 1;   /* L86 cumulative mask */
  free(keys);
}

/* ---- Logits Calibration, solve-T: Algorithm 2 "Binary Search on T" (L625-648; the
 * listing is garbled, read as in DESIGN.md C14/C16) for Problem 1 (L108-110):
 *   k <- Num_Selected_TopP(S, p)           S = raw attention scores (g = id, T = 1)
 *   do  T_mid <- (T_min + T_max) / 2
 *       S_hat <- Softmax(g(z) / T_mid)      (Solution 1 / 2 coincide for the metrics built)
 *       M_k(S) < M_k(S_hat) (too sharp): T_min <- T_mid   else: T_max <- T_mid
 *   while |M_k(S) - M_k(S_hat)| > eps and T_min < T_max (and fewer than max_iter rounds)
 * M_k(X) = mass of the k largest entries of X (order: fp32 bits desc, position asc),
 * as integer mass over total integer mass (reading C5).  T_mid and the bounds are fp32.
 * ACCUM heads are left alone (reading C4 keeps T inside the per-step softmax).
 * Writes u->T = last T_mid, u->k_topp = k; returns the number of rounds; *resid = final
 * |M_k(S) - M_k(S_hat)|. */
static double hko_topk_mass(const float *probs, int32_t lo, int32_t N, int32_t k) {
  hko_key *keys = (hko_key *)malloc(sizeof(hko_key) * (size_t)N);
  uint64_t Wtot = 0, Wk = 0;
  for (int32_t i = 0; i < N; ++i) { keys[i].bits = f32_bits(probs[lo + i]); keys[i].pos = lo + i; }
  qsort(keys, (size_t)N, sizeof(hko_key), hko_key_cmp);
  for (int32_t j = 0; j < N; ++j) {
    float Pj; memcpy(&Pj, &keys[j].bits, 4);
    uint64_t w = (uint64_t)nearbyint((double)Pj * 4294967296.0);
    Wtot += w;
    if (j < k) Wk += w;
  }
  free(keys);
  return Wtot ? (double)Wk / (double)Wtot : 0.0;
}

/* Num_Selected_TopP(S, p) of Algorithm 1/2 line 1: length of the shortest prefix of the
 * order (bits desc, position asc) whose integer mass reaches Theta (reading C5). */
static int32_t hko_num_selected_topp(const float *probs, int32_t lo, int32_t N, float p) {
  if (p >= 1.0f) return N;
  hko_key *keys = (hko_key *)malloc(sizeof(hko_key) * (size_t)N);
  uint64_t Wtot = 0;
  for (int32_t i = 0; i < N; ++i) {
    keys[i].bits = f32_bits(probs[lo + i]); keys[i].pos = lo + i;
    Wtot += (uint64_t)nearbyint((double)probs[lo + i] * 4294967296.0);
  }
  qsort(keys, (size_t)N, sizeof(hko_key), hko_key_cmp);
  uint64_t Theta = (uint64_t)ceil((double)p * (double)Wtot), cum = 0;
  if (Theta < 1) Theta = 1;
  int32_t k = N;
  for (int32_t j = 0; j < N; ++j) {
    float Pj; memcpy(&Pj, &keys[j].bits, 4);
    cum += (uint64_t)nearbyint((double)Pj * 4294967296.0);
    if (cum >= Theta) { k = j + 1; break; }
  }
  free(keys);
  return k;
}

int hko_solve_temperature(const hko_config *c, hko_unit *u, float p, float t_min, float t_max,
                          float eps, int max_iter, double *resid) {
  int32_t lo = u->c_lo, hi = pool_hi(c, u), N = hi - lo;
  if (resid) *resid = 0.0;
  if (N <= 0 || u->score_mode == 1 || u->score_mode == 3) return 0;   /* accumulated metrics keep their T (C4, C18) */
  double *P = (double *)malloc(sizeof(double) * (size_t)N);
  /* line 1: k from the raw attention scores; the k_cap clamp and l_lower do not apply */
  hko_metric_probs(c, u, 0, 1.0, P);
  for (int32_t i = 0; i < N; ++i) u->probs[lo + i] = (float)P[i];
  int32_t k = hko_num_selected_topp(u->probs, lo, N, p);
  double MkS = hko_topk_mass(u->probs, lo, N, k);
  float tlo = t_min, thi = t_max, Tm = u->T;
  double r = 0.0;
  int it = 0;
  while (it < max_iter) {
    Tm = 0.5f * (tlo + thi);
    hko_metric_probs(c, u, u->score_mode, (double)Tm, P);
    for (int32_t i = 0; i < N; ++i) u->probs[lo + i] = (float)P[i];
    double MkH = hko_topk_mass(u->probs, lo, N, k);
    r = fabs(MkS - MkH);
    ++it;
    if (!(r > (double)eps)) break;
    if (MkS < MkH) tlo = Tm; else thi = Tm;
    if (!(tlo < thi)) break;
  }
  u->T = Tm;
  u->k_topp = k;
  if (resid) *resid = r;
  free(P);
  return it;
}

/* ---- Rewrite Cache (L172: "read the selected blocks and write them into a
 * regularized, contiguous range"); ascending position, tail of the last valid
 * page zero (reading C9). */
void hko_rewrite(const hko_config *c, hko_unit *u) {
  int32_t k = u->sel_count;
  for (int32_t j = 0; j < k; ++j) {
    memcpy(u->sel_k + (size_t)j * c->d, u->K + (size_t)u->sel_idx[j] * c->d, sizeof(float) * c->d);
    memcpy(u->sel_v + (size_t)j * c->d, u->V + (size_t)u->sel_idx[j] * c->d, sizeof(float) * c->d);
  }
  int32_t end = ((k + c->page - 1) / c->page) * c->page;
  for (int32_t j = k; j < end; ++j) {
    memset(u->sel_k + (size_t)j * c->d, 0, sizeof(float) * c->d);
    memset(u->sel_v + (size_t)j * c->d, 0, sizeof(float) * c->d);
  }
}

/* ---- Appendix F.  Attention state of an index set I (Eq. 5):
 * o(I) = sum_i SE_i v_i / SE(I), SE(I) = sum_i exp(x_i), x_i = sm_scale q.k_i,
 * carried as (o, m, l) with SE = l*exp(m) (max-shifted, mathematically identical;
 * reading C1).  Rows come from K/V at K + idx[j]*d (idx NULL => rows 0..n_idx-1). */
void hko_state_of_set(const hko_config *c, const float *q_g, const float *K, const float *V,
                      const int32_t *idx, int32_t n_idx, double *o, double *m, double *l) {
  int32_t d = c->d;
  for (int32_t e = 0; e < d; ++e) o[e] = 0.0;
  *m = -INFINITY; *l = 0.0;
  if (n_idx <= 0) return;
  double *x = (double *)malloc(sizeof(double) * (size_t)n_idx);
  for (int32_t j = 0; j < n_idx; ++j) {
    size_t r = (size_t)(idx ? idx[j] : j) * d;
    double dot = 0.0;
    for (int32_t e = 0; e < d; ++e) dot += (double)q_g[e] * (double)K[r + e];
    x[j] = (double)c->sm_scale * dot;
    if (x[j] > *m) *m = x[j];
  }
  for (int32_t j = 0; j < n_idx; ++j) {
    size_t r = (size_t)(idx ? idx[j] : j) * d;
    double w = exp(x[j] - *m);
    *l += w;
    for (int32_t e = 0; e < d; ++e) o[e] += w * (double)V[r + e];
  }
  for (int32_t e = 0; e < d; ++e) o[e] /= *l;
  free(x);
}

/* Merge operator of Eq. 6 (L748-762): o = (o_a SE_a + o_b SE_b)/(SE_a+SE_b),
 * SE = SE_a + SE_b, with SE = l*exp(m).  An empty state has l = 0 (identity). */
void hko_merge(int32_t d, double *o_a, double *m_a, double *l_a,
               const double *o_b, double m_b, double l_b) {
  if (l_b == 0.0) return;
  if (*l_a == 0.0) { for (int32_t e = 0; e < d; ++e) o_a[e] = o_b[e]; *m_a = m_b; *l_a = l_b; return; }
  double m = *m_a > m_b ? *m_a : m_b;
  double sa = *l_a * exp(*m_a - m), sb = l_b * exp(m_b - m);
  for (int32_t e = 0; e < d; ++e) o_a[e] = (o_a[e] * sa + o_b[e] * sb) / (sa + sb);
  *m_a = m; *l_a = sa + sb;
}

/* ---- attention over D u I u C (L84: "exact full-sequence attention from the
 * partial attention outputs of three tiers").  D = sinks [0,min(s,n)) and recent
 * [dense_lo, n) read from the base rows (dense_lo = max(s, n-W) at the last compression step); I = the rewritten selected tier;
 * C = condensed residents.  The calibration temperature is NOT applied here. */
void hko_attend(const hko_config *c, hko_unit *u, const float *q) {
  int32_t d = c->d;
  int32_t s_end = c->sink < u->n ? c->sink : u->n;
  int32_t r_lo = u->dense_lo; if (r_lo < s_end) r_lo = s_end;   /* [dense_lo, n): W tokens at a compression step,
                                                                    growing by one per step until the next (L78) */
  int32_t n_dense = s_end + (u->n - r_lo);
  int32_t *didx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_dense > 0 ? n_dense : 1));
  int32_t t = 0;
  for (int32_t i = 0; i < s_end; ++i) didx[t++] = i;
  for (int32_t i = r_lo; i < u->n; ++i) didx[t++] = i;
  double *o = (double *)malloc(sizeof(double) * (size_t)d * 2);
  double *o2 = o + d;
  for (int32_t g = 0; g < c->G; ++g) {
    const float *qg = q + (size_t)g * d;
    double m, l, m2, l2;
    hko_state_of_set(c, qg, u->K, u->V, didx, n_dense, o, &m, &l);               /* Tier 1 */
    hko_state_of_set(c, qg, u->sel_k, u->sel_v, NULL, u->sel_count, o2, &m2, &l2); /* Tier 2 */
    hko_merge(d, o, &m, &l, o2, m2, l2);
    hko_state_of_set(c, qg, u->cond_k, u->cond_v, NULL, u->cond_count, o2, &m2, &l2); /* Tier 3 */
    hko_merge(d, o, &m, &l, o2, m2, l2);
    for (int32_t e = 0; e < d; ++e) u->out[(size_t)g * d + e] = (float)o[e];
    u->lse[g] = (float)(m + log(l));
  }
  free(o); free(didx);
}

/* ---- one decode step in the order of L78 (Step 1 append; Step 4 compaction of the
 * oldest "before new dense blocks are allocated"; Step 2 calibrated Top-p; Step 3
 * rewrite) followed by the tiered attention of L84.  do_select = 0 reproduces the
 * steps between two compressions (L274 "every 128 steps"): only Step 1 runs, the dense
 * tier grows (L78 steps 1-2), the previous selected tier and condensed tier are reused. */
void hko_decode_step(const hko_config *c, hko_unit *u, const float *q,
                     const float *k_new, const float *v_new, float p, int do_select) {
  hko_append(c, u, k_new, v_new);
  hko_qcache_push(c, u, q);     /* the window slides on every decode step, compression or not (L448) */
  if (do_select) {
    hko_retire_q(c, u, q);      /* Step 4 belongs to the compression step; it also re-anchors dense_lo */
    hko_score(c, u, q);
    hko_calibrate(c, u);
    hko_topp_select(c, u, p, 1);
    hko_rewrite(c, u);
  }
  hko_attend(c, u, q);
}

int hko_decode_step_batch(const hko_config *c, hko_unit *units, int32_t n_units,
                          const float *q, const float *k_new, const float *v_new,
                          float p, int do_select) {
  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1)
#endif
  for (int32_t i = 0; i < n_units; ++i)
    hko_decode_step(c, &units[i], q + (size_t)i * c->G * c->d,
                    k_new + (size_t)i * c->d, v_new + (size_t)i * c->d, p, do_select);
  return nthreads;
}

/* Head-wise block table of the selected tier (L207-209, Fig. 6; reading C9):
 * entry j is the static physical page id while j < ceil(k/page), else -1. */
void hko_sel_table(const hko_config *c, const hko_unit *u, const int32_t *sel_pages, int32_t *sel_table) {
  int32_t used = (u->sel_count + c->page - 1) / c->page;
  for (int32_t j = 0; j < c->k_cap / c->page; ++j) sel_table[j] = j < used ? sel_pages[j] : -1;
}

/* Head-wise mask over the whole sequence "packed in uint8 format" (L439):
 * bit (i % 8) of byte (i / 8), LSB first, set iff position i is selected. */
void hko_sel_mask(const hko_config *c, const hko_unit *u, uint8_t *mask) {
  memset(mask, 0, (size_t)(c->max_ctx / 8));
  for (int32_t j = 0; j < u->sel_count; ++j) {
    int32_t i = u->sel_idx[j];
    mask[i / 8] |= (uint8_t)(1u << (i % 8));
  }
}
