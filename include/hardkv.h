/*
 * hardkv.h -- C ABI of libhardkv.so: the per-decode-step hot path of HARD-KV
 * (arxiv/paper_2606_28831) as hand-written sm_100a CUDA kernels.
 *
 * One call = one stage of the paper's pipeline ("linearly append KV
 * pairs to the Tier 1 Dense Cache" -> "Logits Calibration ... Top-p sampling" ->
 * "Index Regularization" -> eviction of the oldest blocks) followed by the tiered
 * attention of L84 / Appendix F, for ONE layer, for every (sequence b, KV head h).
 *
 * Conventions (all entry points)
 *  - Every pointer inside hardkv_state, and q / k_new / v_new / out / lse, is a
 *    DEVICE pointer owned by the caller.  hardkv_config / hardkv_state structs
 *    themselves and `bytes`/`out` arguments of the create calls are HOST memory.
 *  - The library allocates nothing, never synchronises, never reads device data
 *    back to the host, and launches only on the stream passed in: every stage call
 *    is CUDA-Graph capturable (L53, L63, L168: static shapes, persistent pointers).
 *    Data-dependent sizes (per-head budget k_h, context length) stay on the device;
 *    grids are sized for the static capacities and exit early.
 *  - Return value: HARDKV_OK or an error detectable on the host (bad config,
 *    unsupported (dtype, head_dim, G), NULL required pointer, workspace too small,
 *    a failed launch).  Nothing throws across the ABI.  Inconsistencies only the
 *    device can see set *err_flag != 0 (first error wins; the caller reads the flag after
 *    synchronising): 1 = ctx_len >= max_ctx on append (the sequence is left untouched),
 *    2 = more reuse steps than cfg.reuse_max, 3 = hardkv_topp_select was given a row that is
 *    not a probability row (it sums to more than 4: the integer mass would not be exact),
 *    >= 100 = a device-side wait gave up (a launch-order protocol error, never expected).
 *  - Layouts (row = head_dim elements of kv_dtype; page = page_size rows):
 *      k_pool, v_pool         [n_pages][page][d]
 *      base_table             [B][Hkv][max_ctx/page]   physical page of logical page j
 *      sel_k_pool, sel_v_pool [n_sel_pages][page][d]
 *      sel_pages              [B][Hkv][k_cap/page]     static physical ids (L207-209, L498:
 *                                                      the same id addresses every layer)
 *      cond_k, cond_v         [B][Hkv][cond_cap][d]
 *      q                      [B][Hq][d] kv_dtype, query head g of KV head h is h*G+g
 *      out                    [B][Hq][d] f32,  lse [B][Hq] f32
 *      logits                 [B][Hq][max_ctx] f32 (valid on the pool)
 *      probs                  [B][Hkv][max_ctx] f32 (valid on the pool)
 *  - "pool" of sequence b = positions [c_lo[b], max(c_lo[b], ctx_len[b]-recent)):
 *    Tier-2 candidates (L72); dense tier = [0,sink) u [dense_lo, ctx_len) (L71) with dense_lo =
 *    ctx_len-recent at every compression step; between two compressions it stays put and the
 *    dense tier grows (L78 steps 1-2).
 */
#ifndef HARDKV_H
#define HARDKV_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hardkv_ctx hardkv_ctx;        /* opaque, host-side only */
typedef struct CUstream_st *hardkv_stream;   /* == cudaStream_t */

typedef enum {
  HARDKV_OK = 0,
  HARDKV_ERR_INVALID_ARG = 1,
  HARDKV_ERR_UNSUPPORTED = 2,   /* (kv_dtype, head_dim, G, page_size) not built */
  HARDKV_ERR_WORKSPACE = 3,
  HARDKV_ERR_CUDA = 4,
  HARDKV_ERR_NOALLOC_LIMIT = 5  /* hardkv_decode_attn_noalloc: the problem needs more than HARDKV_NOALLOC_SCRATCH_BYTES */
} hardkv_status;

typedef enum { HARDKV_F32 = 0, HARDKV_BF16 = 1 } hardkv_dtype;
/* Importance metric of a KV head (L276-278): raw attention logits (VANILLA), accumulated attention over the
 * last accum_window steps (H2O-style, L124), or logits max-pooled along the sequence (SNAPKV, L150 / L278). */
typedef enum {
  HARDKV_SCORE_RAW = 0, HARDKV_SCORE_ACCUM = 1, HARDKV_SCORE_SNAPKV = 2,
  /* accumulated attention RECOMPUTED from the sliding-window query cache (L448): every cached query of the last
   * accum_window steps scores the current pool; the head's metric is the mean of their softmax rows (L122-124) */
  HARDKV_SCORE_ACCUM_QCACHE = 3
} hardkv_score_mode;

/* Static for the lifetime of a ctx (and of any graph captured with it). */
typedef struct {
  int32_t batch, num_q_heads, num_kv_heads, head_dim, page_size; /* page_size must be 16            */
  int32_t max_ctx;        /* static capacity in tokens per sequence, multiple of page_size          */
  int32_t sink, recent;   /* s, W: dense tier (L71, L276-277 "sinks + local window")                */
  int32_t k_cap;          /* selected-tier capacity in tokens, multiple of page_size (L233)         */
  int32_t cond_cap;       /* C_cap: constant size of the condensed tier (L76)                       */
  int32_t accum_window;   /* ring depth of SCORE_ACCUM heads (<= 0: no ACCUM state)                 */
  int32_t kv_dtype;       /* hardkv_dtype of q, K, V                                                */
  float   sm_scale;       /* <= 0: 1/sqrt(head_dim)                                                 */
  int32_t pool_kernel;    /* SNAPKV max-pool window: odd, 3..63; 0 or 1: the config has no SNAPKV   */
                          /* head (the pooling pass is not launched)                                */
  int32_t cond_merge;     /* 1: the evictee of a full condensed tier is merged into a resident with  */
                          /* the LSE-preserving weights of Appendix G (Eq. 9) instead of dropped     */
  int32_t reuse_max;      /* most decode steps between two compressions (L274: 128; 0 when every step */
                          /* selects): the dense tier grows by one token per such step (L78 steps 1-2) */
                          /* and the attention grid is sized for recent + reuse_max dense rows        */
} hardkv_config;

/* Caller-owned device state of one layer.  Pointers marked (opt) may be NULL. */
typedef struct {
  void *k_pool, *v_pool;            const int32_t *base_table;
  void *sel_k_pool, *sel_v_pool;    const int32_t *sel_pages;
  void *cond_k, *cond_v;            int32_t *cond_pos, *cond_votes, *cond_count; /* [B][Hkv][C], [B][Hkv]  */
  int32_t *ctx_len, *c_lo;          const int32_t *l_lower, *l_upper;           /* [B] each               */
  int32_t *votes;                                                               /* [B][Hkv][max_ctx]      */
  const float *temperature;         const uint8_t *score_mode;                  /* [B][Hkv], [Hkv]; temperature is
                                                                                   written by hardkv_solve_temperature only */
  float *acc, *ring;                int32_t *ring_slot;  /* (opt) ACCUM: [B][Hkv][max_ctx], [B][Hkv][win][max_ctx], [B][Hkv] */
  int32_t *sel_idx, *sel_count, *sel_table;  /* [B][Hkv][k_cap] asc. positions pad -1, [B][Hkv], [B][Hkv][k_cap/page] */
  uint8_t *sel_mask;                /* (opt) [B][Hkv][max_ctx/8], bit i%8 of byte i/8 (L439)                */
  float *logits, *probs;
  int32_t *err_flag;                /* one device int                                                    */
  void *qcache;                     /* (opt) [B][Hq][accum_window][d] kv_dtype: the queries of the last steps (L448)         */
  int32_t *qc_count, *qc_slot;      /* (opt) [B]: valid steps in the window, next slot; needed by SCORE_ACCUM_QCACHE heads    */
  int32_t *dense_lo;                /* [B] first position of the recent part of the dense tier: ctx_len - recent at the
                                       last compression step (written by the append stage of a compression step); the
                                       caller initialises it to max(min(sink, n), n - recent)                     */
} hardkv_state;

/* Scratch the caller must provide to hardkv_create (device memory, 256-byte aligned). */
hardkv_status hardkv_workspace_bytes(const hardkv_config *cfg, size_t *bytes);
/* Validates cfg and records the workspace.  The caller zeroes the workspace once
 * (it holds arrival counters) before the first stage call; kernels restore the zeros. */
hardkv_status hardkv_create(const hardkv_config *cfg, void *workspace, size_t bytes, hardkv_ctx **out);
void          hardkv_destroy(hardkv_ctx *ctx);
const char   *hardkv_status_string(hardkv_status s);
/* Kernel variant switch for A/B measurements: 0 = generic FMA kernels, 1 = tuned separate kernels,
 * 2 = the same with the TMA-staged (cp.async.bulk + mbarrier ring) persistent score kernel, 3 = score and selection
 * fused into one persistent kernel (bf16, no SNAPKV head, a unit's pool must fit one SM's shared memory:
 * HARDKV_ERR_UNSUPPORTED elsewhere), 4 = score || select: in hardkv_decode_step the persistent score kernel of variant 2
 * streams the units longest pool first and publishes each one when its last chunk is scanned, and the select kernel,
 * launched programmatically behind it and co-resident on the same SMs, selects a unit while later ones are still being
 * scanned (bf16, no SNAPKV head, state without a query cache; elsewhere its stages run back to back as in variant 1).
 * Default 1 (3 measured slower on B200: DESIGN.md section 7). */
hardkv_status hardkv_set_variant(hardkv_ctx *ctx, int32_t variant);
/* Geometry of the select kernel, for A/B measurements and tests: cluster = CTAs per (b, h) in {1, 2, 4, 8}, threads per
 * CTA in {512, 1024}; 0 keeps the automatic choice for that argument.  HARDKV_ERR_UNSUPPORTED when a CTA's slice of the
 * pool would not fit one SM's shared memory.  Host-side only; call it before capturing a graph with this ctx. */
hardkv_status hardkv_set_select_geometry(hardkv_ctx *ctx, int32_t cluster, int32_t threads);
/* 1 (default): in hardkv_decode_step's compression steps on the bf16 paths the attention kernel is launched
 * programmatically behind the select kernel: its CTAs take the SMs that finished selections leave and wait per unit for
 * that unit's selection (flag published by the select kernel), units in the order their selections finish, so the
 * latency-bound selection of the long units hides under the attention of the short ones.  In the same steps the
 * append / retire kernel runs on a side branch BESIDE the score kernel (the score kernel computes the two scalars it
 * needs itself and never reads the appended row) and joins before the select kernel: fork and join are event record /
 * wait on a stream the ctx owns (created by hardkv_create, capturable, no device memory); during the step the new
 * ctx_len / c_lo / dense_lo live in the workspace and the attention kernel writes them back, so when the call's work
 * has completed the state is exactly that of plain stream order.  A ctx therefore serves ONE stream at a time.
 * 0: plain stream order, one stream.  Results are bit-identical either way. */
hardkv_status hardkv_set_overlap(hardkv_ctx *ctx, int32_t on);
/* Measurement hook: while `slots` (DEVICE memory, 2 * capacity u64, the caller presets every pair to (~0, 0)) is set,
 * the i-th hot-kernel launch made through this ctx (append, score, select, score_select, attend; generic variants
 * excepted) records the globaltimer ns at which its first CTA started and its last CTA ended in slots[2 i], slots[2 i
 * + 1] -- also inside a captured graph, which is how bench.py reports per-kernel times of the graph it times.  Calling
 * it again restarts the slot counter; slots = NULL (the default) turns it off and the kernels pay nothing. */
hardkv_status hardkv_set_timing(hardkv_ctx *ctx, unsigned long long *slots, int32_t capacity);
/* 1: launch the hot kernels with the programmatic-dependent-launch attribute (each kernel waits for its predecessor at
 * its top, so ordering is that of a plain stream launch).  Default 0: measured slower inside a captured graph. */
hardkv_status hardkv_set_pdl(hardkv_ctx *ctx, int32_t on);

/* Step 1 + Step 4 of L78 (the bookkeeping of a compression step).  Writes (k_new, v_new) [B][Hkv][d] at position
 * ctx_len[b]; ctx_len += 1; while the pool exceeds l_upper[b] its oldest token retires into the
 * condensed tier of every head, ranked on its Cautious-Update votes (L76, L86); dense_lo = ctx_len - recent. */
hardkv_status hardkv_append_kv(hardkv_ctx *, const hardkv_state *, const void *k_new, const void *v_new,
                               hardkv_stream);
/* hardkv_append_kv with the step's queries q [B][Hq][d]: when cfg.cond_merge is set, every retirement from a full
 * condensed tier folds its evictee (the displaced resident, or the newcomer when it loses on votes) into the
 * resident a with the highest group-mean score x = mean_g sm_scale q_g . K (Thm G.1: "q K_j >> q K_k"):
 * K_a <- w_a K_a + w_e K_e, V_a likewise, w_a = e^{x_a} / (e^{x_a} + e^{x_e}) (Eq. 9), stored rounded to
 * kv_dtype; cond_pos / cond_votes of a are unchanged.  hardkv_decode_step takes this path when cfg.cond_merge is set;
 * hardkv_append_kv (no queries) always evicts. */
hardkv_status hardkv_append_kv_merge(hardkv_ctx *, const hardkv_state *, const void *k_new, const void *v_new,
                                     const void *q, hardkv_stream);
/* logits[b][h*G+g][i] = sm_scale * q . K[i] over the pool (exponent of Eq. 4). */
hardkv_status hardkv_score(hardkv_ctx *, const hardkv_state *, const void *q, hardkv_stream);
/* Slides the step's queries q [B][Hq][d] into state->qcache (L448).  hardkv_decode_step does this itself on every
 * step when state->qcache is set; the stage-by-stage caller does it once per decode step before hardkv_calibrate_topp. */
hardkv_status hardkv_qcache_push(hardkv_ctx *, const hardkv_state *, const void *q, hardkv_stream);
/* Logits Calibration (apply-T) -> probs, then hardkv_topp_select.  Heads in mode SCORE_ACCUM_QCACHE take their
 * probabilities from two more passes over the pool with the cached queries (qcache_kernels.cuh) instead of the logits.  SNAPKV heads (cfg.pool_kernel > 1)
 * are calibrated on their logits max-pooled along the sequence, window clipped to the pool (L278). */
hardkv_status hardkv_calibrate_topp(hardkv_ctx *, const hardkv_state *, float p, hardkv_stream);
/* hardkv_score followed by hardkv_calibrate_topp as ONE call (stages 1 + 2a-2c; same results).  With
 * kernel variant 3 this is a single persistent launch: CTAs stream K pages, and the CTA that retires the last chunk of
 * a unit runs that unit's calibration + Top-p + compaction while the others keep streaming. */
hardkv_status hardkv_score_select(hardkv_ctx *, const hardkv_state *, const void *q, float p, hardkv_stream);
/* Logits Calibration, solve-T: Algorithm 2 "Binary Search on T" (L625-648) for Problem 1 (L108-110), run at a
 * request's first compression (L607).  Needs state->logits of a preceding hardkv_score.  Per (b, KV head):
 * k = Num_Selected_TopP(S, p) with S the raw attention scores (group mean of softmax(z), T = 1, no k_cap clamp);
 * then T_mid = (T_min + T_max) / 2, S_hat = calibrated metric at T_mid, M_k = integer mass of the k largest
 * probabilities over the total; M_k(S) < M_k(S_hat) raises T_min, else lowers T_max; stops when
 * |M_k(S) - M_k(S_hat)| <= eps, T_min >= T_max or after max_iter rounds.  Writes the last T_mid to
 * state->temperature[b][h] (ACCUM heads and empty pools are left unchanged); state->probs is used as scratch. */
hardkv_status hardkv_solve_temperature(hardkv_ctx *, const hardkv_state *, float p, float t_min, float t_max,
                                       float eps, int32_t max_iter, hardkv_stream);
/* Top-p nucleus (L108) on state->probs as given: integer mass w_i = rn(P_i 2^32),
 * order (P bits desc, position asc), minimal prefix with mass >= ceil(p * sum w),
 * clamped to k_cap (L233).  Writes sel_idx, sel_count, sel_table, (sel_mask), votes += 1.
 * probs must be probabilities (0 <= P <= 1; larger values are treated as 1). */
hardkv_status hardkv_topp_select(hardkv_ctx *, const hardkv_state *, float p, hardkv_stream);
/* Rewrite Cache (L172): gather the selected rows into the contiguous selected tier. */
hardkv_status hardkv_rewrite(hardkv_ctx *, const hardkv_state *, hardkv_stream);
/* Split-K decode attention over dense + selected + condensed tiers merged by Eq. 6 (L748-762). */
hardkv_status hardkv_decode_attn(hardkv_ctx *, const hardkv_state *, const void *q, float *out,
                                 float *lse /* nullable */, hardkv_stream);
/* hardkv_decode_attn for callers that cannot allocate device memory at all (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): no hardkv_ctx and no workspace.  The split-K partial states and the
 * arrival counters of the attention kernel live in ONE file-scope static __device__ array of the library,
 * HARDKV_NOALLOC_SCRATCH_BYTES (4 MiB) large, which every GPU that loads the library holds until the process exits.
 * Same kernel, same arithmetic and same results as hardkv_decode_attn on the same state.  Calls no cudaMalloc / cudaFree
 * or any allocating routine; the only other stream work is one memset of the arrival counters.
 *  - cfg is validated like hardkv_create's; a problem whose scratch
 *        4096 + batch * num_kv_heads * ceil((sink + recent + reuse_max + k_cap + cond_cap) / 128) * G * (head_dim + 2) * 4
 *    bytes exceeds the array, or with more than 1024 (sequence, KV head) units, is refused with
 *    HARDKV_ERR_NOALLOC_LIMIT before anything is launched.
 *  - All calls on a device share the array and it keeps the previous call's contents (the counters are cleared on the
 *    stream at every call; the partial states are rewritten before they are read).  Calls that can overlap on the GPU
 *    (different streams, or graphs replayed concurrently) RACE on it: serialise them, or use hardkv_decode_attn with
 *    one workspace per ctx.
 *  - The array's device address is looked up once per device (cudaGetSymbolAddress, with that device current) at the
 *    first call on that device. */
#define HARDKV_NOALLOC_SCRATCH_BYTES (4u << 20)
hardkv_status hardkv_decode_attn_noalloc(const hardkv_config *cfg, const hardkv_state *, const void *q, float *out,
                                         float *lse /* nullable */, hardkv_stream);
/* Steps 3 + 4 fused: the selected rows are gathered from the base pool through sel_idx, written
 * through to the selected tier (L172) and attended while they are in flight, so each selected
 * row is read once; same results as hardkv_rewrite followed by hardkv_decode_attn. */
hardkv_status hardkv_rewrite_attend(hardkv_ctx *, const hardkv_state *, const void *q, float *out,
                                    float *lse /* nullable */, hardkv_stream);
/* HA-Sparse / "Sparse Loading" (L178, L191): attention over dense + selected + condensed where the selected rows
 * are gathered from the base pool through sel_idx; the selected tier is neither read nor written (no rewrite, no
 * memory movement; the gather is the "redundant, irregular" load the paper trades against it).  Same result as
 * hardkv_rewrite followed by hardkv_decode_attn. */
hardkv_status hardkv_sparse_attend(hardkv_ctx *, const hardkv_state *, const void *q, float *out,
                                   float *lse /* nullable */, hardkv_stream);
/* do_select of hardkv_decode_step: which of the paper's regimes the step runs (L191-197, L274). */
enum {
  HARDKV_STEP_REUSE_TIER = 0,     /* between two compressions, HA-Max: attend over the selected tier as rewritten  */
  HARDKV_STEP_SELECT_REWRITE = 1, /* compression step, HA-Max: score, calibrate + Top-p, rewrite fused with attention */
  HARDKV_STEP_SELECT_SPARSE = 2,  /* compression step, HA-Sparse: score, calibrate + Top-p, attention through sel_idx */
  HARDKV_STEP_REUSE_SPARSE = 3    /* between two compressions, HA-Sparse: attention through the previous sel_idx      */
};
/* The whole step on one stream.  Compression steps (do_select 1, 2): append, retire, score, calibrate + Top-p, then
 * rewrite fused with attention (selected rows are read once) or the HA-Sparse attention.  Steps between two
 * compressions (do_select 0, 3; L274): append only -- the token joins the dense tier, which grows from dense_lo (L78
 * steps 1-2), nothing retires -- then attention over dense + the tier / indices of the last compression + condensed:
 * every live token exactly once.  At most cfg.reuse_max such steps may follow one compression (err_flag = 2 beyond). */
hardkv_status hardkv_decode_step(hardkv_ctx *, const hardkv_state *, const void *q, const void *k_new,
                                 const void *v_new, float p, int32_t do_select, float *out,
                                 float *lse /* nullable */, hardkv_stream);

/* hardkv_decode_step with HOST buffers for the per-step tensors (end-to-end entry): q_host
 * [B][Hq][d], k_new_host / v_new_host [B][Hkv][d] in kv_dtype and out_host [B][Hq][d] f32 are
 * HOST pointers (pinned memory for truly asynchronous copies; pageable works, slower).  The
 * call enqueues H2D copies into staging buffers inside the workspace (ONE copy when the three
 * inputs are packed back to back, k_new_host == q_host + bytes(q), v_new_host == k_new_host +
 * bytes(k_new)), then the step, all on `stream`.  When out_host is pinned (mapped) host memory
 * the attention kernel stores the result straight into it and no D2H copy is enqueued; pageable
 * out_host gets one D2H copy.  It does not synchronise -- out_host is valid after the caller
 * synchronises the stream.  The host input buffers must stay untouched until then. */
hardkv_status hardkv_decode_step_host(hardkv_ctx *, const hardkv_state *, const void *q_host,
                                      const void *k_new_host, const void *v_new_host, float p,
                                      int32_t do_select, float *out_host, hardkv_stream);
/* Number of kernels this ctx has launched since hardkv_create (host counter; memcpys excluded). */
int64_t hardkv_launch_count(const hardkv_ctx *ctx);
/* Measurement helper, no ctx: one read-only pass over buf (DEVICE memory, 16-byte aligned, `bytes` of it) with plain
 * 16-byte grid-stride loads, 8 in flight per thread.  Timed by the caller, bytes / time is the read bandwidth a
 * streaming kernel can hope for on this GPU (bench.py --read-peak), next to the copy peak the roofline is quoted on. */
hardkv_status hardkv_probe_read_stream(const void *buf, size_t bytes, hardkv_stream);

#ifdef __cplusplus
}
#endif
#endif
