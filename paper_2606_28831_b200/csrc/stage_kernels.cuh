// stage_kernels.cuh -- append/retire, generic score, rewrite and split-K attention kernels.
// Generic = fp32 FMA arithmetic for every (dtype, head_dim, G); the bf16 tensor-core paths
// live in fast_kernels.cuh.  Citations are PAPER.md lines.
#pragma once
#include "common.cuh"

namespace hardkv {

// =============================================================================================
// Step 1 + Step 4 of L78: append the new (k, v) row; retire the oldest pool tokens into the
// constant-size condensed tier (L76), ranked on Cautious-Update votes (L86).
// One CTA per sequence, one warp per KV head (ctx_len / c_lo are per sequence: they are read by
// every warp before the barrier and written by thread 0 after it).
// do_retire = 0 is the step between two compressions (L274): Step 1 only -- the token joins the dense tier, nothing
// retires and the dense anchor stays (L78 steps 1-2); do_retire = 1 is the bookkeeping of a compression step.
// =============================================================================================
template <typename T, int D>
__global__ void __launch_bounds__(256) append_retire_kernel(Params P, const void *k_new, const void *v_new, const void *q_,
                                                            int do_retire) {
  pdl_wait_then_trigger();
  KernelClock kclock(P);
  constexpr int ROWB = D * sizeof(T);
  constexpr int LPR = ROWB / 16;  // 16-byte vectors per row
  constexpr int EPL = Elem<T>::EPL;
  __shared__ float s_qbar[8][D];  // per warp: group mean of the step's queries (merging only)
  const bool merging = P.cond_merge && q_ != nullptr && P.cond_cap > 0;
  if ((int)blockIdx.x == P.B) {
    // ---- one extra CTA: the step counter, and unit_order = the units by increasing pool length AFTER this step's
    //      append / retirement (arithmetic on the old scalars, so this CTA does not wait for the others): the order in
    //      which the selections of this step finish, which is the order the overlapped attention kernel takes them in ----
    __shared__ int s_len[1024];
    if (threadIdx.x == 0) *P.epoch += 1;
    const int units = P.B * P.Hkv;
    auto len_of = [&](int v) {
      const int bb = v / P.Hkv, n1_ = P.st.ctx_len[bb] + 1;
      int c = P.st.c_lo[bb];
      if (do_retire && n1_ - P.recent - c > P.st.l_upper[bb]) c = n1_ - P.recent - P.st.l_upper[bb];
      return max(n1_ - P.recent - c, 0);
    };
    const bool cached = units <= 1024;
    if (cached) {
      for (int u = threadIdx.x; u < units; u += blockDim.x) s_len[u] = len_of(u);
      __syncthreads();
    }
    for (int u = threadIdx.x; u < units; u += blockDim.x) {
      const int len = cached ? s_len[u] : len_of(u);
      int r = 0;
      for (int v = 0; v < units; ++v) {
        const int lv = cached ? s_len[v] : len_of(v);
        r += (lv < len) || (lv == len && v < u);
      }
      P.unit_order[r] = u;
    }
    return;
  }
  const int b = blockIdx.x, lane = threadIdx.x & 31;
  const int n = P.st.ctx_len[b];
  const int clo0 = P.st.c_lo[b];
  const int lup = P.st.l_upper[b];
  if (n >= P.max_ctx) {  // device-detected inconsistency: flag and leave the sequence untouched
    if (threadIdx.x == 0) {
      atomicExch(P.st.err_flag, 1);
      if (P.defer_commit) { P.sh_scal[b] = n; P.sh_scal[P.B + b] = clo0; P.sh_scal[2 * P.B + b] = P.st.dense_lo[b]; }
    }
    return;
  }
  const int n1 = n + 1;
  int clo = clo0;
  for (int h = threadIdx.x >> 5; h < P.Hkv; h += blockDim.x >> 5) {
    const int unit = b * P.Hkv + h;
    const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
    // the kernel is a chain of dependent loads (latency bound): everything the retirement needs that does not depend
    // on the append is loaded before the append's stores, so the loads overlap instead of queueing behind them
    int cnt = P.st.cond_count[unit];
    // Step 1: "linearly append KV pairs to the Tier 1 Dense Cache" (L78)
    {
      char *dk = const_cast<char *>(paged_row<T, D>(P.st.k_pool, tab, n));
      char *dv = const_cast<char *>(paged_row<T, D>(P.st.v_pool, tab, n));
      const char *sk = reinterpret_cast<const char *>(k_new) + (size_t)unit * ROWB;
      const char *sv = reinterpret_cast<const char *>(v_new) + (size_t)unit * ROWB;
      for (int c = lane; c < LPR; c += 32) {
        stg(dk + c * 16, ldg_ca(sk + c * 16));
        stg(dv + c * 16, ldg_ca(sv + c * 16));
      }
    }
    // Step 4: while the pool exceeds l_upper its oldest token t = c_lo retires.
    int32_t *cpos = P.st.cond_pos + (size_t)unit * P.cond_cap;
    int32_t *cvot = P.st.cond_votes + (size_t)unit * P.cond_cap;
    const int32_t *votes = P.st.votes + (size_t)unit * P.max_ctx;
    clo = clo0;
    bool qbar_ready = false;
    while (do_retire && n1 - P.recent - clo > lup) {
      const int t = clo;
      int slot = -1;
      const bool full = cnt >= P.cond_cap && P.cond_cap > 0;   // a full tier produces an evictee (merging, reading C17)
      const int votes_t = votes[t];                             // in flight together with the scan below
      const char *sk = paged_row<T, D>(P.st.k_pool, tab, t);
      const char *sv = paged_row<T, D>(P.st.v_pool, tab, t);
      if (cnt < P.cond_cap) {
        slot = cnt++;
      } else if (P.cond_cap > 0) {
        // resident with the lexicographically smallest (votes, pos): 8 slots per lane loaded as one batch
        unsigned long long best = ~0ull;
        int best_slot = 0;
        for (int j0 = 0; j0 < P.cond_cap; j0 += 256) {
          int32_t kv[8], kp[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int j = j0 + lane + 32 * i;
            kv[i] = j < P.cond_cap ? cvot[j] : 0x7fffffff;
            kp[i] = j < P.cond_cap ? cpos[j] : 0x7fffffff;
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const unsigned long long key = ((unsigned long long)(uint32_t)kv[i] << 32) | (uint32_t)kp[i];
            if (key < best) { best = key; best_slot = j0 + lane + 32 * i; }
          }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
          unsigned long long ob = shfl_xor_u64(best, o);
          int os = __shfl_xor_sync(0xffffffffu, best_slot, o);
          if (ob < best) { best = ob; best_slot = os; }
        }
        if (votes_t >= (int32_t)(best >> 32)) slot = best_slot;  // newcomer wins ties (it is newer)
      }
      char *ck = reinterpret_cast<char *>(P.st.cond_k) + (size_t)unit * P.cond_cap * ROWB;
      char *cv = reinterpret_cast<char *>(P.st.cond_v) + (size_t)unit * P.cond_cap * ROWB;
      uint4 ek = make_uint4(0, 0, 0, 0), ev = ek;   // evictee pieces (lanes < LPR)
      if (merging && full && lane < LPR) {
        // the displaced resident (newcomer won) or the newcomer itself (it lost) is the evictee
        ek = slot >= 0 ? ldg_ca(ck + (size_t)slot * ROWB + lane * 16) : ldg_ca(sk + lane * 16);
        ev = slot >= 0 ? ldg_ca(cv + (size_t)slot * ROWB + lane * 16) : ldg_ca(sv + lane * 16);
      }
      if (slot >= 0) {
        char *dk = ck + (size_t)slot * ROWB;
        char *dv = cv + (size_t)slot * ROWB;
        for (int c = lane; c < LPR; c += 32) {
          stg(dk + c * 16, ldg_ca(sk + c * 16));
          stg(dv + c * 16, ldg_ca(sv + c * 16));
        }
        if (lane == 0) { cpos[slot] = t; cvot[slot] = votes_t; }
      }
      __syncwarp();
      if (merging && full) {
        // ---- LSE-preserving weighted merging (Appendix G Eq. 9, Thm G.1; reading C17): fold the evictee into
        //      the resident with the highest group-mean score under this step's queries ----
        const int w = threadIdx.x >> 5;
        if (!qbar_ready) {
          for (int e = lane; e < D; e += 32) {
            float acc = 0.f;
            for (int g = 0; g < P.G; ++g) {
              const T *qp = reinterpret_cast<const T *>(q_) + ((size_t)(b * P.Hq + h * P.G + g)) * D + e;
              float f;
              if (sizeof(T) == 4) f = *reinterpret_cast<const float *>(qp);
              else f = __uint_as_float((uint32_t)*reinterpret_cast<const uint16_t *>(qp) << 16);
              acc += f;
            }
            s_qbar[w][e] = acc / (float)P.G;
          }
          __syncwarp();
          qbar_ready = true;
        }
        float bx = -INFINITY;
        int br = 0x7fffffff;
        for (int r = lane; r < cnt; r += 32) {
          float dot = 0.f;
#pragma unroll 4
          for (int c = 0; c < LPR; ++c) {
            float f[EPL];
            Elem<T>::unpack(ldg_ca(ck + (size_t)r * ROWB + c * 16), f);
#pragma unroll
            for (int i = 0; i < EPL; ++i) dot = fmaf(f[i], s_qbar[w][c * EPL + i], dot);
          }
          const float x = P.sm_scale * dot;
          if (x > bx) { bx = x; br = r; }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
          const float ox = __shfl_xor_sync(0xffffffffu, bx, o);
          const int orr = __shfl_xor_sync(0xffffffffu, br, o);
          if (ox > bx || (ox == bx && orr < br)) { bx = ox; br = orr; }
        }
        float fe[EPL], fv[EPL];
        Elem<T>::unpack(ek, fe);
        Elem<T>::unpack(ev, fv);
        float de = 0.f;
        if (lane < LPR) {
#pragma unroll
          for (int i = 0; i < EPL; ++i) de = fmaf(fe[i], s_qbar[w][lane * EPL + i], de);
        }
        const float xe = P.sm_scale * warp_sum_f32(de);
        const float wa = 1.0f / (1.0f + expf(xe - bx)), we = 1.0f - wa;
        if (lane < LPR) {
          float fa[EPL], fb[EPL];
          Elem<T>::unpack(ldg_ca(ck + (size_t)br * ROWB + lane * 16), fa);
          Elem<T>::unpack(ldg_ca(cv + (size_t)br * ROWB + lane * 16), fb);
#pragma unroll
          for (int i = 0; i < EPL; ++i) { fa[i] = fmaf(wa, fa[i], we * fe[i]); fb[i] = fmaf(wa, fb[i], we * fv[i]); }
          stg(ck + (size_t)br * ROWB + lane * 16, Elem<T>::pack(fa));
          stg(cv + (size_t)br * ROWB + lane * 16, Elem<T>::pack(fb));
        }
        __syncwarp();
      }
      ++clo;
    }
    if (lane == 0) {
      P.st.cond_count[unit] = cnt;
      P.att_arrive[unit] = 0;   // re-arm the arrival counters of the kernels that follow (a launch that failed midway
      P.ss_arrive[unit] = 0;    // must not poison the next step)
      if (unit == 0) *P.ss_next = 0;
    }
  }
  // every warp computed the same final c_lo (or ran no head: recompute it arithmetically)
  __syncthreads();
  if (threadIdx.x == 0) {
    int c = clo0;
    if (do_retire && n1 - P.recent - c > lup) c = n1 - P.recent - lup;
    if (P.defer_commit) {      // forked beside the score kernel, which is reading the scalars: into the shadow (common.cuh)
      P.sh_scal[b] = n1;
      P.sh_scal[P.B + b] = c;
      P.sh_scal[2 * P.B + b] = do_retire ? max(min(P.sink, n1), n1 - P.recent) : P.st.dense_lo[b];
    } else {
      P.st.ctx_len[b] = n1;
      P.st.c_lo[b] = c;
      if (do_retire) P.st.dense_lo[b] = max(min(P.sink, n1), n1 - P.recent);   // re-anchor the dense tier (L71)
    }
  }
}

// =============================================================================================
// score (generic): z[g][i] = sm_scale * q_g . k_i over the pool (exponent of Eq. 4).
// A warp streams one 16-row page per iteration: each load instruction covers 512 contiguous
// bytes (32 lanes x 16 B); the LPR lanes that share a row reduce with xor-shuffles.
// =============================================================================================

template <typename T, int D, int G>
__global__ void __launch_bounds__(256) score_generic_kernel(Params P, const void *q_) {
  constexpr int EPL = Elem<T>::EPL, LPR = D / EPL, RPW = 32 / LPR, NIT = PAGE / RPW;
  const int unit = blockIdx.y, b = unit / P.Hkv, h = unit % P.Hkv;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  if (hi <= lo) return;
  const int first_page = lo >> 4, last_page = (hi - 1) >> 4;
  const int pg0 = blockIdx.x * SCORE_PAGES_PER_CTA;
  if (pg0 > last_page || pg0 + SCORE_PAGES_PER_CTA <= first_page) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int lr = lane % LPR, rw = lane / LPR;

  float qf[G][EPL];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const char *qp = reinterpret_cast<const char *>(q_) + ((size_t)(b * P.Hq + h * G + g) * D) * sizeof(T);
    Elem<T>::unpack(ldg_ca(qp + lr * 16), qf[g]);
  }
  const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
  float *lg = P.st.logits + ((size_t)(b * P.Hq + h * G)) * P.max_ctx;

  for (int pi = warp; pi < SCORE_PAGES_PER_CTA; pi += 8) {
    const int pg = pg0 + pi;
    if (pg < first_page || pg > last_page) continue;
    const char *src = reinterpret_cast<const char *>(P.st.k_pool) + (size_t)__ldg(tab + pg) * PAGE * D * sizeof(T);
    uint4 raw[NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) raw[it] = ldg_nc(src + (it * 32 + lane) * 16);
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      float kf[EPL];
      Elem<T>::unpack(raw[it], kf);
      float acc[G];
#pragma unroll
      for (int g = 0; g < G; ++g) {
        float a = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) a = fmaf(qf[g][e], kf[e], a);
        acc[g] = a;
      }
#pragma unroll
      for (int o = LPR / 2; o; o >>= 1)
#pragma unroll
        for (int g = 0; g < G; ++g) acc[g] += __shfl_xor_sync(0xffffffffu, acc[g], o);
      const int pos = pg * PAGE + it * RPW + rw;
      if (lr == 0 && pos >= lo && pos < hi) {
#pragma unroll
        for (int g = 0; g < G; ++g) lg[(size_t)g * P.max_ctx + pos] = acc[g] * P.sm_scale;
      }
    }
  }
}

// =============================================================================================
// Rewrite Cache (L172): "read the selected blocks and write them into a regularized, contiguous
// range".  Slot j of the selected tier <- base row sel_idx[j]; rows k .. 16*ceil(k/16)-1 zero.
// =============================================================================================
constexpr int RW_ROWS_PER_CTA = 64;

template <typename T, int D>
__global__ void __launch_bounds__(256) rewrite_kernel(Params P) {
  constexpr int ROWB = D * sizeof(T), LPR = ROWB / 16;
  constexpr int NV = RW_ROWS_PER_CTA * LPR / 256;  // vectors per thread
  const int unit = blockIdx.y;
  const int k = P.st.sel_count[unit];
  const int kend = (k + PAGE - 1) & ~(PAGE - 1);
  const int j0 = blockIdx.x * RW_ROWS_PER_CTA;
  if (j0 >= kend) return;
  const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
  const int32_t *stab = P.st.sel_pages + (size_t)unit * P.spu;
  const int32_t *idx = P.st.sel_idx + (size_t)unit * P.k_cap;
  uint4 kv[NV], vv[NV];
  size_t dst[NV];
  bool ok[NV];
#pragma unroll
  for (int u = 0; u < NV; ++u) {
    const int vec = threadIdx.x + u * 256;
    const int j = j0 + vec / LPR, c = vec % LPR;
    ok[u] = j < kend;
    kv[u] = make_uint4(0, 0, 0, 0);
    vv[u] = make_uint4(0, 0, 0, 0);
    dst[u] = 0;
    if (ok[u]) {
      dst[u] = ((size_t)__ldg(stab + (j >> 4)) * PAGE + (j & 15)) * ROWB + c * 16;
      if (j < k) {
        const int pos = __ldg(idx + j);
        kv[u] = ldg_nc(paged_row<T, D>(P.st.k_pool, tab, pos) + c * 16);
        vv[u] = ldg_nc(paged_row<T, D>(P.st.v_pool, tab, pos) + c * 16);
      }
    }
  }
#pragma unroll
  for (int u = 0; u < NV; ++u)
    if (ok[u]) {
      stg(reinterpret_cast<char *>(P.st.sel_k_pool) + dst[u], kv[u]);
      stg(reinterpret_cast<char *>(P.st.sel_v_pool) + dst[u], vv[u]);
    }
}

// =============================================================================================
// Split-K decode attention over the three tiers (L84; Appendix F Eq. 4-6).
// Virtual row space of a unit: [dense: sinks, recent | selected tier | condensed residents].
// A CTA takes ATT_CHUNK consecutive virtual rows, keeps a max-shifted state (m, l, acc) per
// query head, and writes it as a partial; the last CTA of the unit to arrive merges the
// partials with the operator of Eq. 6 (SE = l * e^m, o = acc / l).
// MODE: ATT_TIER reads the selected rows from the rewritten selected tier (HA-Max after a rewrite);
// ATT_REWRITE gathers them from the base pool through sel_idx and writes them through to the selected tier while
// they are in registers (rewrite + attend read each row once); ATT_SPARSE gathers them and writes nothing
// (HA-Sparse / "Sparse Loading": regular indices, no memory movement).
// =============================================================================================
constexpr int ATT_CHUNK = 128;
constexpr int ATT_TIER = 0, ATT_REWRITE = 1, ATT_SPARSE = 2;

template <typename T, int D, int G, int MODE>
__global__ void __launch_bounds__(256) attend_generic_kernel(Params P, const void *q_, float *out, float *lse) {
  constexpr int EPL = Elem<T>::EPL, LPR = D / EPL, ROWB = D * sizeof(T);
  constexpr int NGRP = 256 / LPR;  // row groups per CTA
  constexpr int UNR = 4;
  const int unit = blockIdx.y, b = unit / P.Hkv, h = unit % P.Hkv;
  const int n = P.st.ctx_len[b];
  int s_end, r_lo;
  if (!dense_bounds(P, b, n, s_end, r_lo)) {   // more reuse steps than cfg.reuse_max: flag, leave the unit untouched
    if (threadIdx.x == 0 && blockIdx.x == 0) atomicExch(P.st.err_flag, 2);
    return;
  }
  const int n_dense = s_end + (n - r_lo);
  const int k = P.st.sel_count[unit];
  const int cc = P.st.cond_count[unit];
  const int total = n_dense + k + cc;
  const int nchunks = (total + ATT_CHUNK - 1) / ATT_CHUNK;
  const int c = blockIdx.x;
  if (c >= nchunks) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int lr = lane % LPR, grp = tid / LPR;

  const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
  const int32_t *stab = P.st.sel_pages + (size_t)unit * P.spu;
  const int32_t *idx = P.st.sel_idx + (size_t)unit * P.k_cap;

  float qf[G][EPL];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const char *qp = reinterpret_cast<const char *>(q_) + ((size_t)(b * P.Hq + h * G + g) * D) * sizeof(T);
    Elem<T>::unpack(ldg_ca(qp + lr * 16), qf[g]);
  }
  float m[G], l[G], acc[G][EPL];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    m[g] = -INFINITY; l[g] = 0.f;
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[g][e] = 0.f;
  }

  const int v0 = c * ATT_CHUNK, v1 = min(total, v0 + ATT_CHUNK);
  for (int vb = v0 + grp; vb < v1; vb += NGRP * UNR) {
    uint4 kr[UNR], vr[UNR];
    bool ok[UNR];
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      const int v = vb + u * NGRP;
      ok[u] = v < v1;
      kr[u] = make_uint4(0, 0, 0, 0);
      vr[u] = make_uint4(0, 0, 0, 0);
      if (!ok[u]) continue;
      const char *kp, *vp;
      if (v < n_dense) {  // Tier 1: sinks + recent window, read in place
        const int pos = v < s_end ? v : r_lo + (v - s_end);
        kp = paged_row<T, D>(P.st.k_pool, tab, pos);
        vp = paged_row<T, D>(P.st.v_pool, tab, pos);
      } else if (v < n_dense + k) {  // Tier 2: selected rows
        const int j = v - n_dense;
        const size_t so = ((size_t)__ldg(stab + (j >> 4)) * PAGE + (j & 15)) * ROWB;
        if (MODE != ATT_TIER) {
          const int pos = __ldg(idx + j);
          kp = paged_row<T, D>(P.st.k_pool, tab, pos);
          vp = paged_row<T, D>(P.st.v_pool, tab, pos);
        } else {
          kp = reinterpret_cast<const char *>(P.st.sel_k_pool) + so;
          vp = reinterpret_cast<const char *>(P.st.sel_v_pool) + so;
        }
        kr[u] = ldg_nc(kp + lr * 16);
        vr[u] = ldg_nc(vp + lr * 16);
        if (MODE == ATT_REWRITE) {
          stg(reinterpret_cast<char *>(P.st.sel_k_pool) + so + lr * 16, kr[u]);
          stg(reinterpret_cast<char *>(P.st.sel_v_pool) + so + lr * 16, vr[u]);
        }
        continue;
      } else {  // Tier 3: condensed residents
        const size_t co = ((size_t)unit * P.cond_cap + (v - n_dense - k)) * ROWB;
        kp = reinterpret_cast<const char *>(P.st.cond_k) + co;
        vp = reinterpret_cast<const char *>(P.st.cond_v) + co;
      }
      kr[u] = ldg_nc(kp + lr * 16);
      vr[u] = ldg_nc(vp + lr * 16);
    }
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      if (!ok[u]) continue;  // uniform within a row group; groups of one warp may differ -> masks below
      float kf[EPL], vf[EPL];
      Elem<T>::unpack(kr[u], kf);
      Elem<T>::unpack(vr[u], vf);
      float s[G];
#pragma unroll
      for (int g = 0; g < G; ++g) {
        float a = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) a = fmaf(qf[g][e], kf[e], a);
        s[g] = a;
      }
      // reduce over the LPR lanes of this row group (lanes of other groups may be inactive)
      const unsigned gmask = LPR == 32 ? 0xffffffffu : (((1u << LPR) - 1u) << ((lane / LPR) * LPR));
#pragma unroll
      for (int o = LPR / 2; o; o >>= 1)
#pragma unroll
        for (int g = 0; g < G; ++g) s[g] += __shfl_xor_sync(gmask, s[g], o);
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const float x = s[g] * P.sm_scale;
        const float mn = fmaxf(m[g], x);
        const float corr = __expf(m[g] - mn);
        const float pw = __expf(x - mn);
        l[g] = l[g] * corr + pw;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[g][e] = fmaf(acc[g][e], corr, pw * vf[e]);
        m[g] = mn;
      }
    }
  }

  if (MODE == ATT_REWRITE && k > 0 && (n_dense + k - 1) >= v0 && (n_dense + k - 1) < v1) {
    // zero tail of the last valid page of the selected tier (DESIGN reading C9)
    const int kend = (k + PAGE - 1) & ~(PAGE - 1);
    for (int vec = tid; vec < (kend - k) * LPR; vec += 256) {
      const int j = k + vec / LPR, cch = vec % LPR;
      const size_t so = ((size_t)__ldg(stab + (j >> 4)) * PAGE + (j & 15)) * ROWB + cch * 16;
      stg(reinterpret_cast<char *>(P.st.sel_k_pool) + so, make_uint4(0, 0, 0, 0));
      stg(reinterpret_cast<char *>(P.st.sel_v_pool) + so, make_uint4(0, 0, 0, 0));
    }
  }

  // ---- combine the row groups of a warp (Eq. 6 in max-shifted form) ------------------------
#pragma unroll
  for (int o = LPR; o < 32; o <<= 1) {
#pragma unroll
    for (int g = 0; g < G; ++g) {
      const float om = __shfl_xor_sync(0xffffffffu, m[g], o);
      const float ol = __shfl_xor_sync(0xffffffffu, l[g], o);
      const float mn = fmaxf(m[g], om);
      const float ca = (m[g] == -INFINITY) ? 0.f : __expf(m[g] - mn);
      const float cb = (om == -INFINITY) ? 0.f : __expf(om - mn);
      l[g] = l[g] * ca + ol * cb;
#pragma unroll
      for (int e = 0; e < EPL; ++e) {
        const float oa = __shfl_xor_sync(0xffffffffu, acc[g][e], o);
        acc[g][e] = acc[g][e] * ca + oa * cb;
      }
      m[g] = mn;
    }
  }
  // ---- combine the 8 warps through shared memory ---------------------------------------------
  __shared__ float s_st[8][G][D + 2];
  __shared__ int s_last;
  if (lane < LPR) {
#pragma unroll
    for (int g = 0; g < G; ++g) {
#pragma unroll
      for (int e = 0; e < EPL; ++e) s_st[warp][g][2 + lr * EPL + e] = acc[g][e];
      if (lr == 0) { s_st[warp][g][0] = m[g]; s_st[warp][g][1] = l[g]; }
    }
  }
  __syncthreads();
  float *part = P.part + ((size_t)unit * P.att_chunks + c) * G * (D + 2);
  for (int it = tid; it < G * D; it += 256) {
    const int g = it / D, e = it % D;
    float M = -INFINITY;
#pragma unroll
    for (int w = 0; w < 8; ++w) M = fmaxf(M, s_st[w][g][0]);
    float L = 0.f, A = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const float mw = s_st[w][g][0];
      const float cw = (mw == -INFINITY) ? 0.f : __expf(mw - M);
      L += s_st[w][g][1] * cw;
      A += s_st[w][g][2 + e] * cw;
    }
    part[g * (D + 2) + 2 + e] = A;
    if (e == 0) { part[g * (D + 2)] = M; part[g * (D + 2) + 1] = L; }
  }
  // ---- last CTA of the unit merges all partials ------------------------------------------------
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    const int ticket = atomicAdd(P.att_arrive + unit, 1);
    s_last = (ticket == nchunks - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  const float *pu = P.part + (size_t)unit * P.att_chunks * G * (D + 2);
  for (int it = tid; it < G * D; it += 256) {
    const int g = it / D, e = it % D;
    float M = -INFINITY;
    for (int ch = 0; ch < nchunks; ++ch) M = fmaxf(M, __ldcg(pu + ((size_t)ch * G + g) * (D + 2)));
    float L = 0.f, A = 0.f;
    for (int ch = 0; ch < nchunks; ++ch) {
      const float *pp = pu + ((size_t)ch * G + g) * (D + 2);
      const float mw = __ldcg(pp);
      const float cw = (mw == -INFINITY) ? 0.f : __expf(mw - M);
      L += __ldcg(pp + 1) * cw;
      A += __ldcg(pp + 2 + e) * cw;
    }
    out[((size_t)(b * P.Hq + h * G + g)) * D + e] = A / L;
    if (e == 0 && lse) lse[b * P.Hq + h * G + g] = M + logf(L);
  }
  if (tid == 0) P.att_arrive[unit] = 0;  // restore for the next launch / graph replay
}

}  // namespace hardkv
