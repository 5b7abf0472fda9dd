/*
 * hardkv_oracle.h -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, CPU implementation of the HARD-KV per-decode-step hot path
 * (arxiv/paper_2606_28831), written from PAPER.md and the readings C1-C14 listed
 * in DESIGN.md.  It shares no code with the CUDA path under
 * paper_2606_28831_b200/csrc and must never be linked, imported or executed by
 * the product path.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may use it.
 *
 * All floating point is fp64 ("double") unless a value is *state that the method
 * stores in fp32* (logits, probabilities, the ACCUM window, outputs), in which
 * case it is computed in fp64 and rounded once on store.  The Top-p decision is
 * integer arithmetic on the fp32 bit pattern of the probabilities (reading C5).
 *
 * One "unit" is one (sequence b, KV head h) pair: the paper's selection,
 * rewriting and attention are independent per KV head ("Different
 * heads have different budgets, and independently selected indices").
 *
 * Pins (tests/test_oracle_pins.py):  P1 dense-attention equivalence at p=1,
 * P2 brute-force Top-p minimality, P3 ties, P4 degenerate, P5 closed form,
 * P6 order/temperature invariance, P7 Gaussian budget law, P8 merge algebra,
 * P9 rewrite copies, P10 condensed tier == top-C_cap of the retirement log,
 * P11 bookkeeping invariants, P12 integer mass vs fp64 cumsum, P13 temperature
 * solve (g = id => T* = 1; g = a z => T* = a; M_k decreasing in T), P17 query-cache
 * ACCUM (static pool => equals the ring-sum form; library softmax), P14 SNAPKV
 * max-pool == torch.nn.functional.max_pool1d, P15 weighted merging (Eq. 9 weights ==
 * torch.softmax of the pair, SE_evict <= SE_merge <= SE_keep, Thm G.1 limit).
 * Parity unpinned by the paper: readings C2 (GQA group mean), C3 (softmax over
 * the pool only), C4 (ACCUM window form), C7 (condensed-tier retention rule),
 * C8 (threshold mapping).  The paper prints no worked example for them; they
 * are checked for self-consistency only.
 */
#ifndef HARDKV_ORACLE_H
#define HARDKV_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t G;            /* query heads per KV head (GQA group)                     */
  int32_t d;            /* head_dim                                                */
  int32_t page;         /* tokens per page (16)                                    */
  int32_t max_ctx;      /* static capacity in tokens                               */
  int32_t sink;         /* s                                                       */
  int32_t recent;       /* W                                                       */
  int32_t k_cap;        /* selected-tier capacity (tokens)                         */
  int32_t cond_cap;     /* C_cap                                                   */
  int32_t accum_window; /* ACCUM ring depth (32)                                   */
  float   sm_scale;     /* reading C1: 1/sqrt(d) by default                        */
  int32_t pool_kernel;  /* SNAPKV max-pool window (odd; <= 1: identity), C15       */
  int32_t cond_merge;   /* 1: evictees of a full condensed tier are merged (App. G) */
  int32_t kv_bf16;      /* 1: merged rows are stored rounded to bf16 (RNE)          */
} hko_config;

typedef struct {
  /* --- persistent state of one (b,h) unit ------------------------------------ */
  float   *K, *V;              /* [max_ctx][d]  base KV rows, inputs widened exactly */
  int32_t  n;                  /* current context length                            */
  int32_t  c_lo;               /* first pool position                               */
  int32_t  dense_lo;           /* first position of the recent part of the dense tier: n - W at the last
                                  compression step; the dense tier grows from there until the next one (L78
                                  steps 1-2: "append ... to the Tier 1 Dense Cache" until the threshold)      */
  int32_t  l_lower, l_upper;   /* thresholds (reading C8)                           */
  int32_t *votes;              /* [max_ctx] Cautious-Update votes (L86)             */
  float   *cond_k, *cond_v;    /* [cond_cap][d] condensed tier rows                 */
  int32_t *cond_pos, *cond_votes; /* [cond_cap]                                     */
  int32_t  cond_count;
  int32_t  score_mode;         /* 0 RAW, 1 ACCUM (ring of per-step rows), 2 SNAPKV (max-pooled logits, L278),
                                  3 ACCUM recomputed from the query cache (L448, reading C18)            */
  float    T;                  /* calibration temperature of this KV head           */
  float   *acc;                /* [max_ctx] ACCUM running window sum (or NULL)      */
  float   *ring;               /* [accum_window][max_ctx] (or NULL)                 */
  int32_t  ring_slot;
  /* --- per-step products -------------------------------------------------------- */
  float   *logits;             /* [G][max_ctx], valid on the pool                   */
  float   *probs;              /* [max_ctx], valid on the pool                      */
  int32_t *sel_idx;            /* [k_cap] ascending positions, pad -1               */
  int32_t  sel_count;          /* k_h                                               */
  int32_t  k_topp;             /* nucleus size before the k_cap clamp               */
  uint32_t tau_bits;           /* fp32 bit pattern of the smallest selected P       */
  float   *sel_k, *sel_v;      /* [k_cap][d] rewritten tier rows                    */
  float   *out;                /* [G][d]                                            */
  float   *lse;                /* [G]                                               */
  /* --- query cache: "we store the query cache in a sliding window" (L448) -------- */
  float   *qcache;             /* [accum_window][G][d] queries of the last steps (or NULL) */
  int32_t  qc_count, qc_slot;  /* valid entries (<= accum_window), next slot to overwrite  */
} hko_unit;

/* Step 1 of PAPER.md L78: append one (k,v) row at position n; n <- n+1. */
void hko_append(const hko_config *c, hko_unit *u, const float *k_new, const float *v_new);
/* Step 4 of L78 / Tier 3 of L76 / votes ranking L86 (reading C7). Returns #retired. */
int  hko_retire(const hko_config *c, hko_unit *u);
/* The same with the step's queries q [G][d]: when c->cond_merge, the evictee of a full tier is folded into the
 * highest-scoring resident with the LSE-preserving weights of Appendix G (Eq. 9; reading C17). */
int  hko_retire_q(const hko_config *c, hko_unit *u, const float *q);
/* Slides the step's queries q [G][d] into the query cache (L448); a no-op when u->qcache is NULL. */
void hko_qcache_push(const hko_config *c, hko_unit *u, const float *q);
/* z[g][i] = sm_scale * q_g . k_i over the pool (Eq. 4 exponent, reading C1). */
void hko_score(const hko_config *c, hko_unit *u, const float *q);
/* Logits Calibration, apply-T form (L120 Solution 1), group mean (reading C2). */
void hko_calibrate(const hko_config *c, hko_unit *u);
/* Algorithm 2 (L625-648): bisection on T for Problem 1 (L108-110). Returns #rounds. */
int  hko_solve_temperature(const hko_config *c, hko_unit *u, float p, float t_min, float t_max,
                           float eps, int max_iter, double *resid);
/* Top-p nucleus on u->probs (L108; reading C5/C6). votes++ when count_votes. */
void hko_topp_select(const hko_config *c, hko_unit *u, float p, int count_votes);
/* Rewrite Cache (L172), ascending position order, zero tail (reading C9). */
void hko_rewrite(const hko_config *c, hko_unit *u);
/* Eq. 4-6 (L735-762): three tier states merged with the operator of Eq. 6. */
void hko_attend(const hko_config *c, hko_unit *u, const float *q);
/* One whole decode step in the order of L78 (append, retire, select, rewrite, attend).
 * do_select = 0 is a step BETWEEN two compressions (L274): only Step 1 runs -- the new token joins the dense tier,
 * which keeps growing from dense_lo (L78 steps 1-2); nothing retires, nothing is re-selected, and attention covers
 * sinks + [dense_lo, n) + the tier selected at the last compression + the condensed tier: every live token exactly
 * once.  Retirement of the tokens that aged meanwhile happens at the next compression step. */
void hko_decode_step(const hko_config *c, hko_unit *u, const float *q,
                     const float *k_new, const float *v_new, float p, int do_select);
/* The same over many units; q is [n_units][G][d], k_new/v_new [n_units][d].
 * OpenMP over units when built with -fopenmp; returns the thread count used. */
int  hko_decode_step_batch(const hko_config *c, hko_unit *units, int32_t n_units,
                           const float *q, const float *k_new, const float *v_new,
                           float p, int do_select);

/* Attention state algebra of Appendix F, exposed for pin P8.
 * state = (o[d], m, l) with SE = l * exp(m). */
void hko_state_of_set(const hko_config *c, const float *q_g, const float *K, const float *V,
                      const int32_t *idx, int32_t n_idx, double *o, double *m, double *l);
void hko_merge(int32_t d, double *o_a, double *m_a, double *l_a,
               const double *o_b, double m_b, double l_b);

/* sel_table / packed mask helpers (reading C9, "packed in uint8"). */
void hko_sel_table(const hko_config *c, const hko_unit *u, const int32_t *sel_pages, int32_t *sel_table);
void hko_sel_mask(const hko_config *c, const hko_unit *u, uint8_t *mask /*[max_ctx/8]*/);

#ifdef __cplusplus
}
#endif
#endif
