// hardkv.cu -- C ABI of libhardkv.so (include/hardkv.h): argument checks, kernel dispatch on
// (kv_dtype, head_dim, G), stream-ordered launches only.  No allocation, no synchronisation.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>

#include <mutex>

#include "common.cuh"
#include "fast_kernels.cuh"
#include "score_tma.cuh"
#include "select_kernel.cuh"
#include "stage_kernels.cuh"
#include "attend_mma.cuh"
#include "metric_kernels.cuh"
#include "qcache_kernels.cuh"
#include "qcache_umma.cuh"
#include "score_select.cuh"

using namespace hardkv;

struct hardkv_ctx {
  hardkv_config cfg;
  Params base;      // config-derived fields + workspace pointers; `st` is filled per call
  int variant;
  int overlap;                   // 1 (default): the attention of a compression step starts while the select kernel runs
  int fused_ok;                  // the fused score -> select kernel applies to this config (score_select.cuh)
  int overlap_ok;                // the co-resident score || select pair (variant 4) applies to this config
  cudaStream_t aux;              // hardkv_decode_step: the branch the append / retire kernel runs on beside the score kernel
  cudaEvent_t ev_fork, ev_join;  // (fork / join by events: capturable; host-side driver objects, no device memory)
  unsigned long long *timing;    // hardkv_set_timing: per-launch (first CTA start, last CTA end), or NULL
  int timing_cap, timing_next;
  int pdl;                       // 1: launches carry the programmatic-stream-serialization attribute (hardkv_set_pdl)
  int num_sms;
  size_t ws_bytes;
  int64_t launches;              // kernels launched through this ctx (hardkv_launch_count)
  char *stage_q, *stage_k, *stage_v;  // device staging of hardkv_decode_step_host (inside the workspace)
  float *stage_out;
};

namespace {

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct WsLayout { size_t part, arrive, ss, ovl, stats, stage_q, stage_k, stage_v, stage_out, pooled, qc_stats, qc_final, total; };

size_t esize_of(const hardkv_config &c) { return c.kv_dtype == HARDKV_F32 ? 4 : 2; }

int att_chunks_of(const hardkv_config &c) {
  return (c.sink + c.recent + c.reuse_max + c.k_cap + c.cond_cap + ATT_CHUNK - 1) / ATT_CHUNK;
}

int score_chunks_of(const hardkv_config &c) {
  return (c.max_ctx / PAGE + SCORE_PAGES_PER_CTA - 1) / SCORE_PAGES_PER_CTA;
}

WsLayout ws_layout(const hardkv_config &c) {
  const size_t units = (size_t)c.batch * c.num_kv_heads;
  const int G = c.num_q_heads / c.num_kv_heads;
  WsLayout w;
  size_t off = 0;
  w.arrive = off; off += align256(units * sizeof(int32_t));
  w.ss = off;     off += align256((units + 1) * sizeof(int32_t));
  w.ovl = off;    off += align256((3 * units + 1 + 3 * (size_t)c.batch) * sizeof(int32_t));   // sel_flag[units] | unit_order[units] | epoch | score_flag[units] | sh_scal[3][B]
  w.part = off;   off += align256(units * att_chunks_of(c) * G * (c.head_dim + 2) * sizeof(float));
  w.stats = off;  off += align256(units * score_chunks_of(c) * 8 * sizeof(float2));
  const size_t qb = (size_t)c.batch * c.num_q_heads * c.head_dim, kb = units * c.head_dim;
  // staging of the host entry: q | k_new | v_new back to back (rows are >= 128 B, so every part stays 16-byte aligned):
  // packed host buffers arrive with ONE host-to-device copy
  w.stage_q = off;   off += qb * esize_of(c);
  w.stage_k = off;   off += kb * esize_of(c);
  w.stage_v = off;   off += align256(kb * esize_of(c));
  off = align256(off);
  w.stage_out = off; off += align256(qb * sizeof(float));
  w.pooled = off;    off += c.pool_kernel > 1 ? align256((size_t)c.batch * c.num_q_heads * c.max_ctx * sizeof(float)) : 0;
  // query-cache metric: only configs that declare an accumulation window can hold SCORE_ACCUM_QCACHE heads
  w.qc_stats = off;  off += c.accum_window > 0 ? align256(units * score_chunks_of(c) * QC_ROWS * sizeof(float2)) : 0;
  w.qc_final = off;  off += c.accum_window > 0 ? align256(units * QC_ROWS * sizeof(float2)) : 0;
  w.total = off;
  return w;
}

// The fused score -> select kernel holds a whole unit's probability slice in one 1024-thread CTA.
int ss_slice_cap_of(const hardkv_config &c) {
  const int max_pool = c.max_ctx - c.recent > 0 ? c.max_ctx - c.recent : 1;
  return sel_slice_len(max_pool + 31, 1, SS_THREADS);
}
bool fused_eligible(const hardkv_config &c) {
  const int units = c.batch * c.num_kv_heads;
  return c.kv_dtype == HARDKV_BF16 && c.pool_kernel <= 1 && units <= SS_MAX_UNITS &&
         score_select_smem(c.head_dim, ss_slice_cap_of(c), units, c.batch) <= 227u * 1024u;
}

size_t select_smem_bytes(const Params &P) { return (size_t)P.sel_slice_cap * 4 + sizeof(SelShared); }

// Cluster size of the select kernel, from measurements on B200: the kernel is latency bound and
// every extra CTA of a cluster adds DSMEM-merge and barrier latency, so the smallest cluster that keeps a CTA's
// slice near 16 k tokens (~32 per thread) wins (config 2: C = 2 < 1 < 4 < 8; config 3: 1 < 2 < 4; config 4: 4 < 8 < 2);
// with only a few units the clusters are widened to spread them over the chip (config 1: 8 < 2 < 1).
// force_c / force_nt (0 = automatic) come from hardkv_set_select_geometry: A/B measurements and the tests that run
// the kernel at every cluster size.
void select_geometry(const hardkv_config &c, int force_c, int force_nt, int *cluster, int *slice_cap, int *threads) {
  const int units = c.batch * c.num_kv_heads;
  const int max_pool = c.max_ctx - c.recent > 0 ? c.max_ctx - c.recent : 1;
  int C = 1, nt = SEL_NT;
  while (C < SEL_MAXC && sel_slice_len(max_pool + 31, C, SEL_NT) > 17408) C <<= 1;
  while (C < SEL_MAXC && units * C * 2 <= 148) C <<= 1;
  // a unit that would need a cluster of two 512-thread CTAs runs faster as ONE 1024-thread CTA (one per SM): the same
  // threads per unit and no cluster barriers (config 2: 229.0 -> 226.4 us per step).  Wider clusters stay on 512-thread
  // CTAs: two 1024-thread CTAs per unit measured slower than four 512-thread ones (config 4: 108.7 vs 104 us).
  if (C == 2 && units <= 148 && units * 2 > 148 && sel_slice_len(max_pool + 31, 1, SEL_NT_BIG) <= 34816) { C = 1; nt = SEL_NT_BIG; }
  if (force_c == 1 || force_c == 2 || force_c == 4 || force_c == 8) C = force_c;
  if (force_nt == SEL_NT || force_nt == SEL_NT_BIG) nt = force_nt;
  while (C < SEL_MAXC && (size_t)sel_slice_len(max_pool + 31, C, nt) * 4 + sizeof(SelShared) > 227u * 1024u) C <<= 1;
  *cluster = C;
  *slice_cap = sel_slice_len(max_pool + 31, C, nt);
  *threads = nt;
}

// Opt in to the large dynamic shared memory of the select kernel (host-side attribute, no stream work); the attribute
// is per function, so it is raised to the largest request seen in this process.
bool raise_select_smem(const Params &P) {
  static size_t sel_smem_max = 0;
  if (select_smem_bytes(P) > sel_smem_max) sel_smem_max = select_smem_bytes(P);
  const int smx = (int)sel_smem_max;
  const cudaFuncAttribute fa = cudaFuncAttributeMaxDynamicSharedMemorySize;
  bool okk = true;
#define HK_SELATTR(CAL, GM)                                                                              \
  okk = okk && cudaFuncSetAttribute(select_kernel<CAL, GM, SEL_NT>, fa, smx) == cudaSuccess &&          \
        cudaFuncSetAttribute(select_kernel<CAL, GM, SEL_NT_BIG>, fa, smx) == cudaSuccess
  HK_SELATTR(0, 4); HK_SELATTR(1, 4); HK_SELATTR(2, 4); HK_SELATTR(0, 8); HK_SELATTR(1, 8); HK_SELATTR(2, 8);
#undef HK_SELATTR
  return okk;
}

hardkv_status check_config(const hardkv_config *c) {
  if (!c) return HARDKV_ERR_INVALID_ARG;
  if (c->batch <= 0 || c->num_q_heads <= 0 || c->num_kv_heads <= 0 || c->head_dim <= 0) return HARDKV_ERR_INVALID_ARG;
  if (c->num_q_heads % c->num_kv_heads) return HARDKV_ERR_INVALID_ARG;
  if (c->max_ctx <= 0 || c->k_cap <= 0 || c->sink < 0 || c->recent < 0 || c->cond_cap < 0 || c->reuse_max < 0)
    return HARDKV_ERR_INVALID_ARG;
  if (c->page_size != PAGE) return HARDKV_ERR_UNSUPPORTED;
  if (c->max_ctx % PAGE || c->k_cap % PAGE) return HARDKV_ERR_INVALID_ARG;
  if (c->accum_window > 0 && c->accum_window * (c->num_q_heads / c->num_kv_heads) > QC_ROWS) return HARDKV_ERR_UNSUPPORTED;
  if (c->pool_kernel < 0 || c->pool_kernel > 63 || (c->pool_kernel > 1 && c->pool_kernel % 2 == 0)) return HARDKV_ERR_INVALID_ARG;
  const int G = c->num_q_heads / c->num_kv_heads;
  const bool gok = G == 1 || G == 2 || G == 4 || G == 5 || G == 7 || G == 8;
  const bool tok = (c->kv_dtype == HARDKV_F32 && c->head_dim == 64) ||
                   (c->kv_dtype == HARDKV_BF16 && (c->head_dim == 64 || c->head_dim == 128));
  if (!gok || !tok) return HARDKV_ERR_UNSUPPORTED;
  int cl, cap, nt;
  select_geometry(*c, 0, 0, &cl, &cap, &nt);
  if ((size_t)cap * 4 + sizeof(SelShared) > 227u * 1024u) return HARDKV_ERR_UNSUPPORTED;  // pool slice must fit one SM
  return HARDKV_OK;
}

hardkv_status launch_status() { return cudaPeekAtLastError() == cudaSuccess ? HARDKV_OK : HARDKV_ERR_CUDA; }

bool state_ok(const hardkv_ctx *ctx, const hardkv_state *s) {
  if (!ctx || !s) return false;
  return s->k_pool && s->v_pool && s->base_table && s->sel_k_pool && s->sel_v_pool && s->sel_pages &&
         s->cond_count && s->ctx_len && s->c_lo && s->l_lower && s->l_upper && s->votes && s->temperature &&
         s->score_mode && s->sel_idx && s->sel_count && s->sel_table && s->logits && s->probs && s->err_flag && s->dense_lo &&
         (ctx->cfg.cond_cap == 0 || (s->cond_k && s->cond_v && s->cond_pos && s->cond_votes));
}

Params params_of(const hardkv_ctx *ctx, const hardkv_state *s) {
  Params P = ctx->base;
  P.st = *s;
  return P;
}

// Params of ONE launch: takes the next timing slot when hardkv_set_timing is active.
Params launch_params(hardkv_ctx *ctx, const Params &P0) {
  Params P = P0;
  P.timing = nullptr;
  if (ctx->timing && ctx->timing_next < ctx->timing_cap) {
    P.timing = ctx->timing;
    P.timing_slot = ctx->timing_next++;
  }
  return P;
}

// Dispatch on (dtype, head_dim) and on G where the kernel keeps per-head registers.
#define HK_DISPATCH_TD(cfg, ...)                                                                   \
  do {                                                                                             \
    if ((cfg).kv_dtype == HARDKV_F32) { using T = float; constexpr int D = 64; __VA_ARGS__; }      \
    else if ((cfg).head_dim == 128) { using T = bf16_t; constexpr int D = 128; __VA_ARGS__; }      \
    else { using T = bf16_t; constexpr int D = 64; __VA_ARGS__; }                                  \
  } while (0)

#define HK_DISPATCH_G(Gv, ...)                                                                     \
  do {                                                                                             \
    switch (Gv) {                                                                                  \
      case 1: { constexpr int G = 1; __VA_ARGS__; } break;                                         \
      case 2: { constexpr int G = 2; __VA_ARGS__; } break;                                         \
      case 4: { constexpr int G = 4; __VA_ARGS__; } break;                                         \
      case 5: { constexpr int G = 5; __VA_ARGS__; } break;                                         \
      case 7: { constexpr int G = 7; __VA_ARGS__; } break;                                         \
      default: { constexpr int G = 8; __VA_ARGS__; } break;                                        \
    }                                                                                              \
  } while (0)

// Launch with the programmatic-stream-serialization attribute (PDL, see pdl_wait_then_trigger in common.cuh); the
// kernels wait for their predecessor at the top, so ordering and visibility are those of a plain stream launch.
// Off by default (hardkv_set_pdl turns it on): measured on B200 it shortens eager launch loops (config 2 amortised
// regime 59.3 -> 56.1 us, host entry 295.7 -> 293.7 us) but lengthens the captured graph of the headline step
// (234.5 -> 239.8 us): the graph already has no launch gap, and early-resident successors take SM slots from the tail.
template <typename... KArgs, typename... Args>
void launch_pdl(const hardkv_ctx *ctx, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                Args... args) {
  cudaLaunchConfig_t lc = {};
  lc.gridDim = grid; lc.blockDim = block; lc.dynamicSmemBytes = smem; lc.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at;
  lc.numAttrs = ctx->pdl ? 1 : 0;
  cudaLaunchKernelEx(&lc, kernel, KArgs(args)...);
}

// bf16 tensor-core paths (variant 1); fp32 K/V and variant 0 run the generic FMA kernels
bool fast_path(const hardkv_ctx *ctx) { return ctx->variant >= 1 && ctx->cfg.kv_dtype == HARDKV_BF16; }

void launch_append(hardkv_ctx *ctx, const Params &P0, const void *k_new, const void *v_new, const void *q,
                   int do_retire, cudaStream_t st) {
  const Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  // one CTA per sequence + one for the step counter and the unit order of the overlapped attention
  HK_DISPATCH_TD(ctx->cfg, (launch_pdl(ctx, append_retire_kernel<T, D>, dim3(P.B + 1), dim3(256), 0, st, P, k_new, v_new, q,
                                       do_retire)));
}

void launch_score(hardkv_ctx *ctx, const Params &P0, const void *q, cudaStream_t st) {
  const Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  dim3 grid(P.score_chunks, P.B * P.Hkv);
  if (fast_path(ctx) && ctx->variant == 2) {   // TMA-staged persistent variant (A/B: see DESIGN.md)
    const size_t smem = score_tma_smem(P.d, P.B * P.Hkv, P.B);
    if (P.d == 128) score_tma_kernel<128, false><<<ctx->num_sms, SCORE_TMA_THREADS, smem, st>>>(P, q);
    else score_tma_kernel<64, false><<<ctx->num_sms, SCORE_TMA_THREADS, smem, st>>>(P, q);
    return;
  }
  if (fast_path(ctx)) {
    // d = 128: one page in flight per warp at 64 registers, four CTAs per SM -- the same 128 KiB in flight per SM as two
    // pages at two CTAs, in 32 warps instead of 16 (98.5 vs 100.7 us on config 2, probe in profiles/r2_probes.md)
    if (P.d == 128) launch_pdl(ctx, score_mma_kernel<128, 1, 4>, grid, dim3(256), 0, st, P, q);
    else launch_pdl(ctx, score_mma_kernel<64, 2, 2>, grid, dim3(256), 0, st, P, q);
    return;
  }
  HK_DISPATCH_TD(ctx->cfg, HK_DISPATCH_G(P.G, (score_generic_kernel<T, D, G><<<grid, 256, 0, st>>>(P, q))));
}

// calibrate: 0 = select on probs as given, 1 = logits -> probs with in-kernel statistics,
// 2 = logits -> probs with the chunk statistics the bf16 score kernel left in the workspace
void launch_select(hardkv_ctx *ctx, const Params &P0, float p, int calibrate, cudaStream_t st) {
  const Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3(P.B * P.Hkv * P.sel_cluster);
  lc.blockDim = dim3(P.sel_nt);
  lc.dynamicSmemBytes = select_smem_bytes(P);
  lc.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = P.sel_cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at;
  lc.numAttrs = ctx->pdl ? 2 : 1;
#define HK_SEL(CAL, GM)                                                                 \
  do {                                                                                  \
    if (P.sel_nt == SEL_NT_BIG) cudaLaunchKernelEx(&lc, select_kernel<CAL, GM, SEL_NT_BIG>, P, p); \
    else cudaLaunchKernelEx(&lc, select_kernel<CAL, GM, SEL_NT>, P, p);                 \
  } while (0)
  if (P.G <= 4) {
    if (calibrate == 2) HK_SEL(2, 4);
    else if (calibrate == 1) HK_SEL(1, 4);
    else HK_SEL(0, 4);
  } else {
    if (calibrate == 2) HK_SEL(2, 8);
    else if (calibrate == 1) HK_SEL(1, 8);
    else HK_SEL(0, 8);
  }
#undef HK_SEL
}

// Geometry of the select kernel when it runs beside the publishing score kernel (variant 4): 512-thread CTAs, the
// smallest cluster whose slice + scratch fit in the shared memory a score CTA leaves free on its SM.
bool overlap_geometry(const hardkv_config &c, int *cluster, int *slice_cap) {
  const int units = c.batch * c.num_kv_heads;
  const int max_pool = c.max_ctx - c.recent > 0 ? c.max_ctx - c.recent : 1;
  const size_t room = 227u * 1024u - score_tma_smem(c.head_dim, units, c.batch) - 2048 - 1024;  // static smem, per-CTA reserve
  for (int C = 1; C <= SEL_MAXC; C <<= 1) {
    const int cap = sel_slice_len(max_pool + 31, C, SEL_NT);
    if ((size_t)cap * 4 + sizeof(SelShared) <= room) { *cluster = C; *slice_cap = cap; return true; }
  }
  return false;
}
bool overlap_eligible(const hardkv_config &c) {
  int cl, cap;
  return c.kv_dtype == HARDKV_BF16 && c.pool_kernel <= 1 && score_tma_smem(c.head_dim, c.batch * c.num_kv_heads, c.batch) < 200u * 1024u &&
         overlap_geometry(c, &cl, &cap);
}

// stages 1 and 2a-2c as two co-resident kernels (variant 4): the persistent, publishing score kernel and, launched
// programmatically behind it, the select kernel that takes every unit as soon as its last chunk is scanned
void launch_score_select_overlapped(hardkv_ctx *ctx, const Params &P0, const void *q, float p, cudaStream_t st) {
  {
    const Params P = launch_params(ctx, P0);
    ctx->launches += 1;
    const size_t smem = score_tma_smem(P.d, P.B * P.Hkv, P.B);
    if (P.d == 128) score_tma_kernel<128, true><<<ctx->num_sms, SCORE_TMA_THREADS, smem, st>>>(P, q);
    else score_tma_kernel<64, true><<<ctx->num_sms, SCORE_TMA_THREADS, smem, st>>>(P, q);
  }
  Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  overlap_geometry(ctx->cfg, &P.sel_cluster, &P.sel_slice_cap);
  P.sel_nt = SEL_NT;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3(P.B * P.Hkv * P.sel_cluster);
  lc.blockDim = dim3(SEL_NT);
  lc.dynamicSmemBytes = select_smem_bytes(P);
  lc.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = P.sel_cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = at;
  lc.numAttrs = 2;
  if (P.G <= 4) cudaLaunchKernelEx(&lc, select_overlap_kernel<4>, P, p);
  else cudaLaunchKernelEx(&lc, select_overlap_kernel<8>, P, p);
}

// stages 1 + 2a-2c as one persistent kernel, one CTA per SM (variant 3)
void launch_score_select(hardkv_ctx *ctx, const Params &P0, const void *q, float p, cudaStream_t st) {
  const Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  const size_t smem = score_select_smem(P.d, P.ss_slice_cap, P.B * P.Hkv, P.B);
  const dim3 grid(ctx->num_sms), block(SS_THREADS);
  if (P.d == 128) {
    if (P.G <= 4) launch_pdl(ctx, score_select_kernel<128, 4>, grid, block, smem, st, P, q, p);
    else launch_pdl(ctx, score_select_kernel<128, 8>, grid, block, smem, st, P, q, p);
  } else {
    if (P.G <= 4) launch_pdl(ctx, score_select_kernel<64, 4>, grid, block, smem, st, P, q, p);
    else launch_pdl(ctx, score_select_kernel<64, 8>, grid, block, smem, st, P, q, p);
  }
}

// accumulated attention from the query cache (L448; reading C18): two passes over the pool + a reduction, launched
// only when the caller's state holds a query cache (heads in other modes exit at once)
void launch_qcache_metric(hardkv_ctx *ctx, const Params &P0, cudaStream_t st) {
  if (!P0.st.qcache || P0.accum_window <= 0 || ctx->cfg.kv_dtype != HARDKV_BF16) return;
  const dim3 grid(P0.score_chunks, P0.B * P0.Hkv);
  const size_t rowb = (size_t)P0.d * 2;
  const size_t sm1 = QC_ROWS * rowb + 8 * QC_ROWS * sizeof(float2), sm2 = QC_ROWS * rowb + QC_ROWS * sizeof(float2);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(qcache_pass_kernel<128, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(QC_ROWS * 256 + 8 * QC_ROWS * 8));
    cudaFuncSetAttribute(qcache_pass_kernel<128, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(QC_ROWS * 256 + 8 * QC_ROWS * 8));
    cudaFuncSetAttribute(qcache_pass_kernel<64, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(QC_ROWS * 256 + 8 * QC_ROWS * 8));
    cudaFuncSetAttribute(qcache_pass_kernel<64, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(QC_ROWS * 256 + 8 * QC_ROWS * 8));
    attr_set = true;
  }
  ctx->launches += 3;
  // tcgen05 / TMEM kernels (qcache_umma.cuh); variant 0 keeps the mma.sync kernels for A/B
  const bool umma = ctx->variant != 0 && P0.B * P0.Hkv <= QU_MAX_UNITS;
  const dim3 grid_u(ctx->num_sms);
  const size_t smu = qcache_umma_smem(P0.d, qcache_umma_rows(P0.accum_window, P0.G));
  static bool attr_u = false;
  if (umma && !attr_u) {
    const int mx = (int)(qcache_umma_smem(128, 256) < 216u * 1024u ? qcache_umma_smem(128, 256) : 216u * 1024u);
    cudaFuncSetAttribute(qcache_umma_kernel<128, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
    cudaFuncSetAttribute(qcache_umma_kernel<128, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
    cudaFuncSetAttribute(qcache_umma_kernel<64, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
    cudaFuncSetAttribute(qcache_umma_kernel<64, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
    attr_u = true;
  }
  {
    const Params P = launch_params(ctx, P0);
    if (umma) {
      if (P.d == 128) qcache_umma_kernel<128, 1><<<grid_u, QU_THREADS, smu, st>>>(P);
      else qcache_umma_kernel<64, 1><<<grid_u, QU_THREADS, smu, st>>>(P);
    } else if (P.d == 128) qcache_pass_kernel<128, 1><<<grid, 256, sm1, st>>>(P);
    else qcache_pass_kernel<64, 1><<<grid, 256, sm1, st>>>(P);
  }
  {
    const Params P = launch_params(ctx, P0);
    qcache_reduce_kernel<<<P.B * P.Hkv, QC_ROWS, 0, st>>>(P);
  }
  {
    const Params P = launch_params(ctx, P0);
    if (umma) {
      if (P.d == 128) qcache_umma_kernel<128, 2><<<grid_u, QU_THREADS, smu, st>>>(P);
      else qcache_umma_kernel<64, 2><<<grid_u, QU_THREADS, smu, st>>>(P);
    } else if (P.d == 128) qcache_pass_kernel<128, 2><<<grid, 256, sm2, st>>>(P);
    else qcache_pass_kernel<64, 2><<<grid, 256, sm2, st>>>(P);
  }
}

void launch_qcache_push(hardkv_ctx *ctx, const Params &P, const void *q, cudaStream_t st) {
  if (!P.st.qcache || P.accum_window <= 0) return;
  ctx->launches += 1;
  qcache_push_kernel<<<P.B, 256, 0, st>>>(P, q);
}

// SNAPKV metric transform (L278): only configs that declare a pooling window pay for the launch
void launch_pool(hardkv_ctx *ctx, const Params &P0, cudaStream_t st) {
  if (P0.pool_kernel <= 1) return;
  const Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  dim3 grid((P.max_ctx + POOL_TOK - 1) / POOL_TOK, P.B * P.Hkv);
  maxpool_kernel<<<grid, 256, 0, st>>>(P);
}

void launch_rewrite(hardkv_ctx *ctx, const Params &P, cudaStream_t st) {
  ctx->launches += 1;
  dim3 grid((P.k_cap + RW_ROWS_PER_CTA - 1) / RW_ROWS_PER_CTA, P.B * P.Hkv);
  HK_DISPATCH_TD(ctx->cfg, (rewrite_kernel<T, D><<<grid, 256, 0, st>>>(P)));
}

// overlap = 1: the launch directly follows the select kernel in the stream and may start while it runs (programmatic
// dependent launch): its CTAs take units in the order their selections finish and wait per unit (wait_unit_selected)
void launch_attend(hardkv_ctx *ctx, const Params &P0, const void *q, float *out, float *lse, int mode,
                   cudaStream_t st, int overlap = 0) {
  Params P = launch_params(ctx, P0);
  ctx->launches += 1;
  if (fast_path(ctx) && overlap) {
    P.wait_select = overlap;
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((P.att_chunks * ATT_CHUNK + ATT_MMA_CHUNK - 1) / ATT_MMA_CHUNK, P.B * P.Hkv);
    lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = at; lc.numAttrs = 1;
    if (P.d == 128) {
      if (mode == ATT_REWRITE) cudaLaunchKernelEx(&lc, attend_mma_kernel<128, ATT_REWRITE>, P, q, out, lse);
      else cudaLaunchKernelEx(&lc, attend_mma_kernel<128, ATT_SPARSE>, P, q, out, lse);
    } else {
      if (mode == ATT_REWRITE) cudaLaunchKernelEx(&lc, attend_mma_kernel<64, ATT_REWRITE>, P, q, out, lse);
      else cudaLaunchKernelEx(&lc, attend_mma_kernel<64, ATT_SPARSE>, P, q, out, lse);
    }
    return;
  }
  if (fast_path(ctx)) {
    dim3 gm((P.att_chunks * ATT_CHUNK + ATT_MMA_CHUNK - 1) / ATT_MMA_CHUNK, P.B * P.Hkv);
    const size_t sm = 0;
    if (P.d == 128) {
      if (mode == ATT_REWRITE) launch_pdl(ctx, attend_mma_kernel<128, ATT_REWRITE>, gm, dim3(256), sm, st, P, q, out, lse);
      else if (mode == ATT_SPARSE) launch_pdl(ctx, attend_mma_kernel<128, ATT_SPARSE>, gm, dim3(256), sm, st, P, q, out, lse);
      else launch_pdl(ctx, attend_mma_kernel<128, ATT_TIER>, gm, dim3(256), sm, st, P, q, out, lse);
    } else {
      if (mode == ATT_REWRITE) launch_pdl(ctx, attend_mma_kernel<64, ATT_REWRITE>, gm, dim3(256), sm, st, P, q, out, lse);
      else if (mode == ATT_SPARSE) launch_pdl(ctx, attend_mma_kernel<64, ATT_SPARSE>, gm, dim3(256), sm, st, P, q, out, lse);
      else launch_pdl(ctx, attend_mma_kernel<64, ATT_TIER>, gm, dim3(256), sm, st, P, q, out, lse);
    }
    return;
  }
  dim3 grid(P.att_chunks, P.B * P.Hkv);
  if (mode == ATT_REWRITE)
    HK_DISPATCH_TD(ctx->cfg, HK_DISPATCH_G(P.G, (attend_generic_kernel<T, D, G, ATT_REWRITE><<<grid, 256, 0, st>>>(P, q, out, lse))));
  else if (mode == ATT_SPARSE)
    HK_DISPATCH_TD(ctx->cfg, HK_DISPATCH_G(P.G, (attend_generic_kernel<T, D, G, ATT_SPARSE><<<grid, 256, 0, st>>>(P, q, out, lse))));
  else
    HK_DISPATCH_TD(ctx->cfg, HK_DISPATCH_G(P.G, (attend_generic_kernel<T, D, G, ATT_TIER><<<grid, 256, 0, st>>>(P, q, out, lse))));
}

// Read-only streaming probe (hardkv_probe_read_stream): what a plain 16-byte grid-stride read reaches on this GPU,
// the reference the K scan is compared with beside the copy peak of MEASURED_PEAKS.json.
__device__ unsigned int g_probe_sink;
__global__ void __launch_bounds__(256) read_stream_kernel(const uint4 *p, size_t n) {
  unsigned int acc = 0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  for (; i + 7 * stride < n; i += 8 * stride) {
    uint4 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = ldg_nc(p + i + u * stride);
#pragma unroll
    for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
  }
  for (; i < n; i += stride) { const uint4 v = ldg_nc(p + i); acc ^= v.x ^ v.y ^ v.z ^ v.w; }
  if (acc == 0x9e3779b9u) g_probe_sink = acc;   // keeps the loads alive; practically never taken
}

}  // namespace

// ---- scratch of hardkv_decode_attn_noalloc: [0, 4096) arrival counters of up to 1024 units | split-K partial states.
// In HOST code this name is only a stand-in for the symbol, not a device address: the address a kernel may be given
// comes from cudaGetSymbolAddress (noalloc_scratch below), once per device.
static __device__ __align__(256) unsigned char g_noalloc_scratch[HARDKV_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr size_t NOALLOC_COUNTER_BYTES = 4096;
constexpr int NOALLOC_MAX_UNITS = (int)(NOALLOC_COUNTER_BYTES / sizeof(int32_t));
constexpr int NOALLOC_MAX_DEVICES = 64;

// Device address of g_noalloc_scratch on the CURRENT device, looked up once per device.
unsigned char *noalloc_scratch(cudaError_t *err) {
  static std::mutex mu;
  static unsigned char *ptr[NOALLOC_MAX_DEVICES] = {};
  int dev = -1;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { *err = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    void *p = nullptr;
    *err = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (*err != cudaSuccess || !p) { if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol; return nullptr; }
    ptr[dev] = static_cast<unsigned char *>(p);
  }
  return ptr[dev];
}
}  // namespace

extern "C" {

const char *hardkv_status_string(hardkv_status s) {
  switch (s) {
    case HARDKV_OK: return "ok";
    case HARDKV_ERR_INVALID_ARG: return "invalid argument";
    case HARDKV_ERR_UNSUPPORTED: return "unsupported (kv_dtype, head_dim, G, page_size)";
    case HARDKV_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case HARDKV_ERR_CUDA: return "CUDA launch error";
    case HARDKV_ERR_NOALLOC_LIMIT: return "problem exceeds the static scratch of the no-allocation entry point (HARDKV_NOALLOC_SCRATCH_BYTES)";
  }
  return "unknown status";
}

hardkv_status hardkv_workspace_bytes(const hardkv_config *cfg, size_t *bytes) {
  if (!bytes) return HARDKV_ERR_INVALID_ARG;
  hardkv_status s = check_config(cfg);
  if (s != HARDKV_OK) return s;
  *bytes = ws_layout(*cfg).total;
  return HARDKV_OK;
}

hardkv_status hardkv_create(const hardkv_config *cfg, void *workspace, size_t bytes, hardkv_ctx **out) {
  if (!out) return HARDKV_ERR_INVALID_ARG;
  *out = nullptr;
  hardkv_status s = check_config(cfg);
  if (s != HARDKV_OK) return s;
  const WsLayout w = ws_layout(*cfg);
  if (!workspace || ((uintptr_t)workspace & 255) || bytes < w.total) return HARDKV_ERR_WORKSPACE;
  hardkv_ctx *ctx = new (std::nothrow) hardkv_ctx;
  if (!ctx) return HARDKV_ERR_INVALID_ARG;
  memset(ctx, 0, sizeof(*ctx));
  ctx->cfg = *cfg;
  ctx->variant = 1;
  ctx->overlap = 1;
  ctx->ws_bytes = w.total;
  Params &P = ctx->base;
  P.B = cfg->batch; P.Hq = cfg->num_q_heads; P.Hkv = cfg->num_kv_heads; P.G = P.Hq / P.Hkv;
  P.d = cfg->head_dim; P.max_ctx = cfg->max_ctx; P.sink = cfg->sink; P.recent = cfg->recent;
  P.k_cap = cfg->k_cap; P.cond_cap = cfg->cond_cap; P.accum_window = cfg->accum_window; P.reuse_max = cfg->reuse_max;
  P.ppu = cfg->max_ctx / PAGE; P.spu = cfg->k_cap / PAGE;
  P.att_chunks = att_chunks_of(*cfg);
  P.sm_scale = cfg->sm_scale > 0.f ? cfg->sm_scale : 1.0f / sqrtf((float)cfg->head_dim);
  char *base = reinterpret_cast<char *>(workspace);
  P.att_arrive = reinterpret_cast<int32_t *>(base + w.arrive);
  P.ss_arrive = reinterpret_cast<int32_t *>(base + w.ss);
  P.ss_next = P.ss_arrive + (size_t)cfg->batch * cfg->num_kv_heads;
  P.ss_slice_cap = ss_slice_cap_of(*cfg);
  P.sel_flag = reinterpret_cast<int32_t *>(base + w.ovl);
  P.unit_order = P.sel_flag + (size_t)cfg->batch * cfg->num_kv_heads;
  P.epoch = P.unit_order + (size_t)cfg->batch * cfg->num_kv_heads;
  P.score_flag = P.epoch + 1;
  P.sh_scal = P.score_flag + (size_t)cfg->batch * cfg->num_kv_heads;
  P.wait_select = 0;
  P.part = reinterpret_cast<float *>(base + w.part);
  P.score_stats = reinterpret_cast<float2 *>(base + w.stats);
  P.score_chunks = score_chunks_of(*cfg);
  P.pool_kernel = cfg->pool_kernel;
  P.cond_merge = cfg->cond_merge != 0;
  P.pooled = cfg->pool_kernel > 1 ? reinterpret_cast<float *>(base + w.pooled) : nullptr;
  P.qc_stats = cfg->accum_window > 0 ? reinterpret_cast<float2 *>(base + w.qc_stats) : nullptr;
  P.qc_final = cfg->accum_window > 0 ? reinterpret_cast<float2 *>(base + w.qc_final) : nullptr;
  P.st_esize = (int)esize_of(*cfg);
  ctx->stage_q = base + w.stage_q; ctx->stage_k = base + w.stage_k; ctx->stage_v = base + w.stage_v;
  ctx->stage_out = reinterpret_cast<float *>(base + w.stage_out);
  select_geometry(*cfg, 0, 0, &P.sel_cluster, &P.sel_slice_cap, &P.sel_nt);
  int dev = 0, nsm = 148;
  cudaGetDevice(&dev);
  if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) nsm = 148;
  ctx->num_sms = nsm;
  if (cfg->kv_dtype == HARDKV_BF16) {
    const int ssm = (int)score_tma_smem(cfg->head_dim, cfg->batch * cfg->num_kv_heads, cfg->batch);
    static int score_smem_max = 0;
    if (ssm > score_smem_max) score_smem_max = ssm;
    cudaFuncSetAttribute(score_tma_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_smem_max);
    cudaFuncSetAttribute(score_tma_kernel<64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_smem_max);
    cudaFuncSetAttribute(score_tma_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_smem_max);
    cudaFuncSetAttribute(score_tma_kernel<64, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_smem_max);
    // the publishing kernel shares its SM with a select CTA: all of the SM's on-chip memory as shared memory
    cudaFuncSetAttribute(score_tma_kernel<128, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(score_tma_kernel<64, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  }
  ctx->overlap_ok = overlap_eligible(*cfg) ? 1 : 0;
  if (ctx->overlap_ok) {
    static int so_smem_max = 0;
    int cl, cap;
    overlap_geometry(*cfg, &cl, &cap);
    const int need = (int)((size_t)cap * 4 + sizeof(SelShared));
    if (need > so_smem_max) so_smem_max = need;
    const cudaFuncAttribute fa = cudaFuncAttributeMaxDynamicSharedMemorySize;
    if (cudaFuncSetAttribute(select_overlap_kernel<4>, fa, so_smem_max) != cudaSuccess ||
        cudaFuncSetAttribute(select_overlap_kernel<8>, fa, so_smem_max) != cudaSuccess ||
        cudaFuncSetAttribute(select_overlap_kernel<4>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared) != cudaSuccess ||
        cudaFuncSetAttribute(select_overlap_kernel<8>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared) != cudaSuccess) {
      cudaGetLastError();
      ctx->overlap_ok = 0;
    }
  }
  if (!raise_select_smem(P)) {
    cudaGetLastError();
    delete ctx;
    return HARDKV_ERR_CUDA;
  }
  ctx->fused_ok = fused_eligible(*cfg) ? 1 : 0;
  if (ctx->fused_ok) {
    static int ss_smem_max = 0;
    const int need = (int)score_select_smem(cfg->head_dim, P.ss_slice_cap, cfg->batch * cfg->num_kv_heads, cfg->batch);
    if (need > ss_smem_max) ss_smem_max = need;
    const cudaFuncAttribute fa = cudaFuncAttributeMaxDynamicSharedMemorySize;
    if (cudaFuncSetAttribute(score_select_kernel<128, 4>, fa, ss_smem_max) != cudaSuccess ||
        cudaFuncSetAttribute(score_select_kernel<128, 8>, fa, ss_smem_max) != cudaSuccess ||
        cudaFuncSetAttribute(score_select_kernel<64, 4>, fa, ss_smem_max) != cudaSuccess ||
        cudaFuncSetAttribute(score_select_kernel<64, 8>, fa, ss_smem_max) != cudaSuccess) {
      cudaGetLastError();
      ctx->fused_ok = 0;
    }
  }
  // the side branch of hardkv_decode_step (without these driver objects the step runs in plain stream order)
  {
    int lo_p = 0, hi_p = 0;
    cudaDeviceGetStreamPriorityRange(&lo_p, &hi_p);
    if (cudaStreamCreateWithPriority(&ctx->aux, cudaStreamNonBlocking, hi_p) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError();
      if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
      if (ctx->aux) cudaStreamDestroy(ctx->aux);
      ctx->aux = nullptr; ctx->ev_fork = nullptr; ctx->ev_join = nullptr;
    }
  }
  *out = ctx;
  return HARDKV_OK;
}

void hardkv_destroy(hardkv_ctx *ctx) {
  if (!ctx) return;
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
  if (ctx->aux) cudaStreamDestroy(ctx->aux);
  delete ctx;
}

hardkv_status hardkv_set_variant(hardkv_ctx *ctx, int32_t variant) {
  if (!ctx || variant < 0 || variant > 4) return HARDKV_ERR_INVALID_ARG;
  if (variant == 3 && !ctx->fused_ok) return HARDKV_ERR_UNSUPPORTED;
  if (variant == 4 && !ctx->overlap_ok) return HARDKV_ERR_UNSUPPORTED;
  ctx->variant = variant;
  return HARDKV_OK;
}

hardkv_status hardkv_set_select_geometry(hardkv_ctx *ctx, int32_t cluster, int32_t threads) {
  if (!ctx) return HARDKV_ERR_INVALID_ARG;
  if (cluster != 0 && cluster != 1 && cluster != 2 && cluster != 4 && cluster != 8) return HARDKV_ERR_INVALID_ARG;
  if (threads != 0 && threads != SEL_NT && threads != SEL_NT_BIG) return HARDKV_ERR_INVALID_ARG;
  int cl, cap, nt;
  select_geometry(ctx->cfg, cluster, threads, &cl, &cap, &nt);
  if ((size_t)cap * 4 + sizeof(SelShared) > 227u * 1024u) return HARDKV_ERR_UNSUPPORTED;
  ctx->base.sel_cluster = cl; ctx->base.sel_slice_cap = cap; ctx->base.sel_nt = nt;
  return raise_select_smem(ctx->base) ? HARDKV_OK : HARDKV_ERR_CUDA;
}

hardkv_status hardkv_set_overlap(hardkv_ctx *ctx, int32_t on) {
  if (!ctx || (on != 0 && on != 1)) return HARDKV_ERR_INVALID_ARG;
  ctx->overlap = on;
  return HARDKV_OK;
}

hardkv_status hardkv_set_timing(hardkv_ctx *ctx, unsigned long long *slots, int32_t capacity) {
  if (!ctx || capacity < 0 || (slots && capacity == 0)) return HARDKV_ERR_INVALID_ARG;
  ctx->timing = slots;
  ctx->timing_cap = slots ? capacity : 0;
  ctx->timing_next = 0;
  return HARDKV_OK;
}

hardkv_status hardkv_set_pdl(hardkv_ctx *ctx, int32_t on) {
  if (!ctx || (on != 0 && on != 1)) return HARDKV_ERR_INVALID_ARG;
  ctx->pdl = on;
  return HARDKV_OK;
}

hardkv_status hardkv_append_kv(hardkv_ctx *ctx, const hardkv_state *s, const void *k_new, const void *v_new,
                               hardkv_stream st) {
  if (!state_ok(ctx, s) || !k_new || !v_new) return HARDKV_ERR_INVALID_ARG;
  launch_append(ctx, params_of(ctx, s), k_new, v_new, nullptr, 1, st);
  return launch_status();
}

hardkv_status hardkv_append_kv_merge(hardkv_ctx *ctx, const hardkv_state *s, const void *k_new, const void *v_new,
                                     const void *q, hardkv_stream st) {
  if (!state_ok(ctx, s) || !k_new || !v_new || !q) return HARDKV_ERR_INVALID_ARG;
  launch_append(ctx, params_of(ctx, s), k_new, v_new, q, 1, st);
  return launch_status();
}

hardkv_status hardkv_score(hardkv_ctx *ctx, const hardkv_state *s, const void *q, hardkv_stream st) {
  if (!state_ok(ctx, s) || !q) return HARDKV_ERR_INVALID_ARG;
  launch_score(ctx, params_of(ctx, s), q, st);
  return launch_status();
}

static bool accum_ok(const hardkv_ctx *ctx, const hardkv_state *s) {
  // ACCUM / ACCUM_QCACHE heads need their state; score_mode lives on the device, so require one complete set of
  // buffers (the ring of rows or the query cache) whenever the config declares a window.
  return ctx->cfg.accum_window <= 0 || (s->acc && s->ring && s->ring_slot) || (s->qcache && s->qc_count && s->qc_slot);
}

hardkv_status hardkv_calibrate_topp(hardkv_ctx *ctx, const hardkv_state *s, float p, hardkv_stream st) {
  if (!state_ok(ctx, s) || !(p > 0.f) || !accum_ok(ctx, s)) return HARDKV_ERR_INVALID_ARG;
  launch_pool(ctx, params_of(ctx, s), st);
  launch_qcache_metric(ctx, params_of(ctx, s), st);
  launch_select(ctx, params_of(ctx, s), p, 1, st);
  return launch_status();
}

hardkv_status hardkv_qcache_push(hardkv_ctx *ctx, const hardkv_state *s, const void *q, hardkv_stream st) {
  if (!state_ok(ctx, s) || !q || !s->qcache || !s->qc_count || !s->qc_slot || ctx->cfg.accum_window <= 0)
    return HARDKV_ERR_INVALID_ARG;
  launch_qcache_push(ctx, params_of(ctx, s), q, st);
  return launch_status();
}

hardkv_status hardkv_score_select(hardkv_ctx *ctx, const hardkv_state *s, const void *q, float p, hardkv_stream st) {
  if (!state_ok(ctx, s) || !q || !(p > 0.f) || !accum_ok(ctx, s)) return HARDKV_ERR_INVALID_ARG;
  const Params P = params_of(ctx, s);
  if (ctx->variant == 3 && !P.st.qcache) {
    launch_score_select(ctx, P, q, p, st);
  } else {   // variant 4 needs the unit order of a preceding append in the same call: here its two kernels run back to back
    launch_score(ctx, P, q, st);
    launch_pool(ctx, P, st);
    launch_qcache_metric(ctx, P, st);
    launch_select(ctx, P, p, (fast_path(ctx) && P.pool_kernel <= 1) ? 2 : 1, st);
  }
  return launch_status();
}

hardkv_status hardkv_solve_temperature(hardkv_ctx *ctx, const hardkv_state *s, float p, float t_min, float t_max,
                                       float eps, int32_t max_iter, hardkv_stream st) {
  if (!state_ok(ctx, s) || !(p > 0.f) || !(t_min > 0.f) || !(t_max > t_min) || !(eps >= 0.f) || max_iter < 1)
    return HARDKV_ERR_INVALID_ARG;
  const Params P = params_of(ctx, s);
  launch_pool(ctx, P, st);
  ctx->launches += 1;
  solve_temperature_kernel<<<P.B * P.Hkv, SOLVE_NT, 0, st>>>(P, p, t_min, t_max, eps, max_iter);
  return launch_status();
}

hardkv_status hardkv_topp_select(hardkv_ctx *ctx, const hardkv_state *s, float p, hardkv_stream st) {
  if (!state_ok(ctx, s) || !(p > 0.f)) return HARDKV_ERR_INVALID_ARG;
  launch_select(ctx, params_of(ctx, s), p, 0, st);
  return launch_status();
}

hardkv_status hardkv_rewrite(hardkv_ctx *ctx, const hardkv_state *s, hardkv_stream st) {
  if (!state_ok(ctx, s)) return HARDKV_ERR_INVALID_ARG;
  launch_rewrite(ctx, params_of(ctx, s), st);
  return launch_status();
}

hardkv_status hardkv_decode_attn(hardkv_ctx *ctx, const hardkv_state *s, const void *q, float *out, float *lse,
                                 hardkv_stream st) {
  if (!state_ok(ctx, s) || !q || !out) return HARDKV_ERR_INVALID_ARG;
  launch_attend(ctx, params_of(ctx, s), q, out, lse, ATT_TIER, st);
  return launch_status();
}

hardkv_status hardkv_rewrite_attend(hardkv_ctx *ctx, const hardkv_state *s, const void *q, float *out, float *lse,
                                    hardkv_stream st) {
  if (!state_ok(ctx, s) || !q || !out) return HARDKV_ERR_INVALID_ARG;
  launch_attend(ctx, params_of(ctx, s), q, out, lse, ATT_REWRITE, st);
  return launch_status();
}

hardkv_status hardkv_sparse_attend(hardkv_ctx *ctx, const hardkv_state *s, const void *q, float *out, float *lse,
                                   hardkv_stream st) {
  if (!state_ok(ctx, s) || !q || !out) return HARDKV_ERR_INVALID_ARG;
  launch_attend(ctx, params_of(ctx, s), q, out, lse, ATT_SPARSE, st);
  return launch_status();
}

hardkv_status hardkv_decode_attn_noalloc(const hardkv_config *cfg, const hardkv_state *s, const void *q, float *out,
                                         float *lse, hardkv_stream st) {
  const hardkv_status cs = check_config(cfg);
  if (cs != HARDKV_OK) return cs;
  // size limit first: nothing is touched or launched for a problem that does not fit the static array
  const size_t units = (size_t)cfg->batch * cfg->num_kv_heads;
  const int G = cfg->num_q_heads / cfg->num_kv_heads;
  const size_t part_bytes = units * att_chunks_of(*cfg) * G * (cfg->head_dim + 2) * sizeof(float);
  if (units > (size_t)NOALLOC_MAX_UNITS || NOALLOC_COUNTER_BYTES + part_bytes > (size_t)HARDKV_NOALLOC_SCRATCH_BYTES)
    return HARDKV_ERR_NOALLOC_LIMIT;
  if (!s || !q || !out) return HARDKV_ERR_INVALID_ARG;
  if (!(s->k_pool && s->v_pool && s->base_table && s->sel_k_pool && s->sel_v_pool && s->sel_pages && s->sel_count &&
        s->cond_count && s->ctx_len && s->dense_lo && s->err_flag &&
        (cfg->cond_cap == 0 || (s->cond_k && s->cond_v))))
    return HARDKV_ERR_INVALID_ARG;
  cudaError_t ce;
  unsigned char *scratch = noalloc_scratch(&ce);
  if (!scratch) { cudaGetLastError(); return HARDKV_ERR_CUDA; }
  Params P;
  memset(&P, 0, sizeof(P));
  P.B = cfg->batch; P.Hq = cfg->num_q_heads; P.Hkv = cfg->num_kv_heads; P.G = G;
  P.d = cfg->head_dim; P.max_ctx = cfg->max_ctx; P.sink = cfg->sink; P.recent = cfg->recent;
  P.k_cap = cfg->k_cap; P.cond_cap = cfg->cond_cap; P.accum_window = cfg->accum_window; P.reuse_max = cfg->reuse_max;
  P.ppu = cfg->max_ctx / PAGE; P.spu = cfg->k_cap / PAGE;
  P.att_chunks = att_chunks_of(*cfg);
  P.sm_scale = cfg->sm_scale > 0.f ? cfg->sm_scale : 1.0f / sqrtf((float)cfg->head_dim);
  P.st = *s;
  P.st_esize = (int)esize_of(*cfg);
  P.att_arrive = reinterpret_cast<int32_t *>(scratch);
  P.part = reinterpret_cast<float *>(scratch + NOALLOC_COUNTER_BYTES);
  // the array keeps whatever the last call (or a launch that failed midway) left: the counters must start at zero
  if (cudaMemsetAsync(P.att_arrive, 0, units * sizeof(int32_t), st) != cudaSuccess) { cudaGetLastError(); return HARDKV_ERR_CUDA; }
  if (cfg->kv_dtype == HARDKV_BF16) {
    const dim3 gm((P.att_chunks * ATT_CHUNK + ATT_MMA_CHUNK - 1) / ATT_MMA_CHUNK, P.B * P.Hkv);
    if (P.d == 128) attend_mma_kernel<128, ATT_TIER><<<gm, 256, 0, st>>>(P, q, out, lse);
    else attend_mma_kernel<64, ATT_TIER><<<gm, 256, 0, st>>>(P, q, out, lse);
  } else {
    const dim3 grid(P.att_chunks, P.B * P.Hkv);
    HK_DISPATCH_TD(*cfg, HK_DISPATCH_G(P.G, (attend_generic_kernel<T, D, G, ATT_TIER><<<grid, 256, 0, st>>>(P, q, out, lse))));
  }
  return launch_status();
}

int64_t hardkv_launch_count(const hardkv_ctx *ctx) { return ctx ? ctx->launches : -1; }

hardkv_status hardkv_probe_read_stream(const void *buf, size_t bytes, hardkv_stream st) {
  if (!buf || bytes < 16 || ((uintptr_t)buf & 15)) return HARDKV_ERR_INVALID_ARG;
  int dev = 0, nsm = 148;
  cudaGetDevice(&dev);
  if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) nsm = 148;
  read_stream_kernel<<<nsm * 4, 256, 0, st>>>(static_cast<const uint4 *>(buf), bytes / 16);
  return launch_status();
}

hardkv_status hardkv_decode_step(hardkv_ctx *ctx, const hardkv_state *s, const void *q, const void *k_new,
                                 const void *v_new, float p, int32_t do_select, float *out, float *lse,
                                 hardkv_stream st) {
  if (!state_ok(ctx, s) || !q || !k_new || !v_new || !out || !(p > 0.f) || !accum_ok(ctx, s))
    return HARDKV_ERR_INVALID_ARG;
  const Params P = params_of(ctx, s);
  if (do_select < 0 || do_select > 3) return HARDKV_ERR_INVALID_ARG;
  const bool compress = do_select == HARDKV_STEP_SELECT_REWRITE || do_select == HARDKV_STEP_SELECT_SPARSE;
  // The score kernel needs from the append / retire kernel only the two scalars n + 1 and the new c_lo, which it can
  // compute itself (pool_bounds, pre_append), and never reads the appended row (it lies in the recent window, outside
  // the pool, for W >= 1): on a compression step the append kernel runs on a forked branch BESIDE the score kernel and
  // joins before the select kernel, which needs its step counter, unit order and re-armed counters.  While the score
  // kernel reads the per-sequence scalars nobody may overwrite them: the forked append kernel leaves them in the
  // workspace (sh_scal), the kernels after the join read them there, the attention kernel writes them back in place.
  const bool fork = compress && ctx->overlap && ctx->aux && fast_path(ctx) && (ctx->variant == 1 || ctx->variant == 2) &&
                    ctx->cfg.recent >= 1;
  Params Pj = P;                 // launches after the join
  if (fork) {
    Params Pa = P;
    Pa.defer_commit = 1;
    Pj.use_shadow = 1;
    cudaEventRecord(ctx->ev_fork, st);
    cudaStreamWaitEvent(ctx->aux, ctx->ev_fork, 0);
    launch_append(ctx, Pa, k_new, v_new, q, 1, ctx->aux);
    cudaEventRecord(ctx->ev_join, ctx->aux);
  } else {
    launch_append(ctx, P, k_new, v_new, q, compress ? 1 : 0, st);   // between compressions: Step 1 only (L78, L274)
  }
  launch_qcache_push(ctx, P, q, st);                              // the query window slides on every step (L448)
  // variant 4 overlaps the two kernels through the unit order the append kernel of THIS call has just written
  const bool ss_overlap = compress && ctx->variant == 4 && !P.st.qcache;
  if (compress && ctx->variant == 3 && !P.st.qcache) {
    launch_score_select(ctx, P, q, p, st);
  } else if (ss_overlap) {
    launch_score_select_overlapped(ctx, P, q, p, st);
  } else if (compress) {
    if (fork) {
      Params Ps = P;
      Ps.pre_append = 1;
      launch_score(ctx, Ps, q, st);
      cudaStreamWaitEvent(st, ctx->ev_join, 0);
    } else {
      launch_score(ctx, P, q, st);
    }
    launch_pool(ctx, Pj, st);
    launch_qcache_metric(ctx, Pj, st);
    // the score kernel's chunk statistics describe the raw logits: configs with pooled heads take them in-kernel
    launch_select(ctx, Pj, p, (fast_path(ctx) && P.pool_kernel <= 1) ? 2 : 1, st);
  }
  // the select kernel (variants 1, 2: the last launch above) is followed by the attention of the same units: overlap them
  const int overlap = ss_overlap ? 2 : (compress && ctx->overlap && fast_path(ctx) && ctx->variant != 3);
  launch_attend(ctx, Pj, q, out, lse, do_select == HARDKV_STEP_SELECT_REWRITE ? ATT_REWRITE
                                     : (do_select == HARDKV_STEP_REUSE_TIER ? ATT_TIER : ATT_SPARSE), st, overlap);
  return launch_status();
}

hardkv_status hardkv_decode_step_host(hardkv_ctx *ctx, const hardkv_state *s, const void *q_host,
                                      const void *k_new_host, const void *v_new_host, float p, int32_t do_select,
                                      float *out_host, hardkv_stream st) {
  if (!ctx || !q_host || !k_new_host || !v_new_host || !out_host) return HARDKV_ERR_INVALID_ARG;
  const hardkv_config &c = ctx->cfg;
  const size_t qe = (size_t)c.batch * c.num_q_heads * c.head_dim, ke = (size_t)c.batch * c.num_kv_heads * c.head_dim;
  const size_t es = esize_of(c);
  const char *qh = static_cast<const char *>(q_host), *kh = static_cast<const char *>(k_new_host),
             *vh = static_cast<const char *>(v_new_host);
  if (kh == qh + qe * es && vh == kh + ke * es) {   // packed [q | k_new | v_new]: one copy into the contiguous staging
    if (cudaMemcpyAsync(ctx->stage_q, q_host, (qe + 2 * ke) * es, cudaMemcpyHostToDevice, st) != cudaSuccess)
      return HARDKV_ERR_CUDA;
  } else if (cudaMemcpyAsync(ctx->stage_q, q_host, qe * es, cudaMemcpyHostToDevice, st) != cudaSuccess ||
             cudaMemcpyAsync(ctx->stage_k, k_new_host, ke * es, cudaMemcpyHostToDevice, st) != cudaSuccess ||
             cudaMemcpyAsync(ctx->stage_v, v_new_host, ke * es, cudaMemcpyHostToDevice, st) != cudaSuccess) {
    return HARDKV_ERR_CUDA;
  }
  // out_host in pinned (mapped) host memory: the merging CTAs of the attention kernel store the result straight into it
  // -- no device-to-host copy node; pageable memory goes through the staging buffer and one copy.
  float *out_dev = nullptr;
  cudaPointerAttributes pa;
  if (cudaPointerGetAttributes(&pa, out_host) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer)
    out_dev = static_cast<float *>(pa.devicePointer);
  else
    cudaGetLastError();
  hardkv_status r = hardkv_decode_step(ctx, s, ctx->stage_q, ctx->stage_k, ctx->stage_v, p, do_select,
                                       out_dev ? out_dev : ctx->stage_out, nullptr, st);
  if (r != HARDKV_OK) return r;
  if (!out_dev && cudaMemcpyAsync(out_host, ctx->stage_out, qe * sizeof(float), cudaMemcpyDeviceToHost, st) != cudaSuccess)
    return HARDKV_ERR_CUDA;
  return HARDKV_OK;
}

}  // extern "C"
