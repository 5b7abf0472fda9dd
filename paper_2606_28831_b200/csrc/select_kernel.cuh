// select_kernel.cuh -- Logits Calibration (apply-T) + Top-p nucleus + stream compaction.
// PAPER.md L106-128 (calibration), L108 (Top-p), L86 (votes), L207-209 / L439 (head-wise block
// table, packed mask); readings C2-C6, C9.
//
// One thread-block CLUSTER per (sequence, KV head); the C CTAs of a cluster split the pool into
// contiguous, 32-aligned position slices and keep their slice of the probability row (fp32 bit
// patterns) in shared memory for the whole kernel.  Cross-CTA exchange goes through distributed
// shared memory (DSMEM) and cluster barriers; nothing but the final results touches HBM.
//
// The nucleus is found without a sort: a most-significant-digit radix descent on the fp32 bit
// pattern of P (0 <= P <= 1: unsigned order == float order, 30 significant bits) with three digits of 10 bits.
// Each level builds a histogram of (count, integer mass) per digit with w_i = rn(P_i * 2^32)
// summed exactly (u32 shared atomics on count, w >> 12 and w & 4095): exact and order
// independent, so it reproduces a sorted-prefix definition bit for bit (reading C5).  The bins
// are merged across the cluster by their owner CTA, and every CTA then walks the merged bins from
// the top to the bin in which the mass reaches Theta = ceil(p * Wtot) (or the count reaches
// k_cap, reading C6).
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"

namespace hardkv {
namespace cg = cooperative_groups;

constexpr int SEL_NT = 512;         // threads of a CTA: 512 (2 CTAs / SM, clusters) or SEL_NT_BIG (1 CTA / SM, whole unit)
constexpr int SEL_NT_BIG = 1024;
constexpr int SEL_NW = SEL_NT_BIG / 32;   // capacity of the per-warp arrays in shared memory
constexpr int SEL_MAXC = 8;        // portable cluster size limit
constexpr int SEL_NB = 1024;       // bins per level: a probability is <= 1, so its fp32 pattern has 30 significant bits
constexpr uint32_t SEL_ONE = 0x3f800000u;   // bit pattern of 1.0f: larger inputs are treated as 1
constexpr int SEL_MSPLIT = 12;     // mass kept as (w >> 12, w & 4095) in two u32 counters
constexpr uint32_t SEL_INVALID = 0xffffffffu;  // slice entry outside the pool (never a probability)

struct SelShared {
  uint32_t h_cnt[SEL_NB], h_hi[SEL_NB], h_lo[SEL_NB];  // local histogram of the current level
  uint32_t m_cnt[SEL_NB / 2];                          // bins owned by this CTA, merged over the cluster
  unsigned long long m_mass[SEL_NB / 2];
  unsigned long long tot_mass[SEL_MAXC];               // per owner range: totals (written by the owner into every CTA)
  uint32_t tot_cnt[SEL_MAXC];
  float st_m[SEL_MAXC][8], st_s[SEL_MAXC][8];          // per CTA softmax statistics of the G query heads
  double acc_tot[SEL_MAXC];
  int c_gt[SEL_MAXC], c_tie[SEL_MAXC];
  float red_f[SEL_NW][8][2];
  double red_d[SEL_NW];
  unsigned long long red_u[SEL_NW];
  uint32_t red_c[SEL_NW];
  int w_gt[SEL_NW], w_tie[SEL_NW];
  // result of one level's walk (written by warp 0)
  int res_bin, res_bin_cnt, res_cum_cnt;
  unsigned long long res_cum_mass, res_theta;
};

__device__ __forceinline__ unsigned long long mass_of_bits(uint32_t bits) {
  // w = rn(P * 2^32): the product is exact in fp32 (power-of-two scale), conversion rounds to nearest even
  return __float2ull_rn(__uint_as_float(bits) * 4294967296.0f);
}

__device__ __forceinline__ void hist_add(SelShared &sh, int bin, uint32_t bits) {
  const unsigned long long w = mass_of_bits(bits);
  atomicAdd(&sh.h_cnt[bin], 1u);
  atomicAdd(&sh.h_hi[bin], (uint32_t)(w >> SEL_MSPLIT));
  atomicAdd(&sh.h_lo[bin], (uint32_t)(w & ((1u << SEL_MSPLIT) - 1u)));
}

// Per-CTA slice geometry: the cluster covers absolute positions [base, base + C*per), base = lo & ~31.
__host__ __device__ __forceinline__ int sel_slice_len(int span, int C, int nt) {
  const int per = (span + C - 1) / C;
  return (per + nt - 1) / nt * nt;
}

// Loads of data that another CTA of the SAME launch may have written (the fused score -> select kernel): L2-coherent
// ld.global.cg; otherwise the read-only path.
template <bool COHERENT> __device__ __forceinline__ float4 sel_ld4(const float4 *p) { return COHERENT ? __ldcg(p) : __ldg(p); }
template <bool COHERENT> __device__ __forceinline__ float sel_ld(const float *p) { return COHERENT ? __ldcg(p) : __ldg(p); }
template <bool COHERENT> __device__ __forceinline__ float2 sel_ld2(const float2 *p) { return COHERENT ? __ldcg(p) : __ldg(p); }

// Stages 2a-2c for ONE (sequence, KV head) unit, run by every thread of the CTA (and of its cluster when CLUSTERED).
// CALIBRATE: 1 = logits -> probs (2a) with in-kernel statistics, 2 = with the chunk statistics of the score kernel,
//            0 = select on state->probs as given.
// GMAX: compile-time bound of the GQA group (4 or 8) -- sizes the register arrays of the calibration.
// NT: threads per CTA (SEL_NT: two CTAs per SM; SEL_NT_BIG: one CTA per SM that holds a whole unit without a cluster).
// CLUSTERED: the unit is split over the P.sel_cluster CTAs of a thread-block cluster (DSMEM exchange); false = one CTA.
// COHERENT: logits / chunk statistics were written earlier in this same launch (score_select_kernel).
// pbits: this CTA's slice of the probability row, sh: its scratch, both in shared memory.
template <int CALIBRATE, int GMAX, int NT, bool CLUSTERED, bool COHERENT>
__device__ __forceinline__ void select_unit(const Params &P, float p, int unit, uint32_t *pbits, SelShared &sh) {
  constexpr int NW = NT / 32;
  cg::cluster_group cluster = cg::this_cluster();
  const int C = CLUSTERED ? P.sel_cluster : 1;
  const int rank = CLUSTERED ? (int)cluster.block_rank() : 0;
  const int b = unit / P.Hkv, h = unit % P.Hkv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  const int N = hi - lo;
  const int G = P.G;
  float *probs = P.st.probs + (size_t)unit * P.max_ctx;
  int32_t *sel_idx = P.st.sel_idx + (size_t)unit * P.k_cap;
  int32_t *sel_table = P.st.sel_table + (size_t)unit * P.spu;
  const bool want_mask = P.st.sel_mask != nullptr;
  uint8_t *mask = want_mask ? P.st.sel_mask + (size_t)unit * (P.max_ctx / 8) : nullptr;
  const int mask_bytes = P.max_ctx / 8;

  if (N <= 0) {  // empty pool: nothing selected (uniform over the cluster: no barrier is pending)
    for (int j = rank * NT + tid; j < P.k_cap; j += C * NT) sel_idx[j] = -1;
    for (int j = rank * NT + tid; j < P.spu; j += C * NT) sel_table[j] = -1;
    if (want_mask)
      for (int y = rank * NT + tid; y < mask_bytes; y += C * NT) mask[y] = 0;
    if (rank == 0 && tid == 0) P.st.sel_count[unit] = 0;
    __syncthreads();
    if (C > 1) cluster.sync();
    if (rank == 0 && tid == 0 && P.sel_flag) {
      __threadfence();
      *reinterpret_cast<volatile int32_t *>(P.sel_flag + unit) = *reinterpret_cast<volatile int32_t *>(P.epoch);
    }
    return;
  }

  const int base = lo & ~31;
  const int per = sel_slice_len(hi - base, C, NT);   // <= P.sel_slice_cap by construction of the cap
  const int s0 = base + rank * per;              // this CTA's slice: absolute positions [s0, s0 + per)
  const int wseg = per / NW;                 // positions per warp (multiple of 32)

  // split-phase cluster barrier: every CTA of the cluster must be running before its shared memory
  // is written by a peer; the wait sits in front of the first DSMEM access.
  if (C > 1) cluster.barrier_arrive();
  for (int d = tid; d < SEL_NB; d += NT) { sh.h_cnt[d] = 0; sh.h_hi[d] = 0; sh.h_lo[d] = 0; }

  // ---------------- 2a: calibration ------------------------------------------------------------
  // heads on the query-cache metric arrive with their probabilities in state->probs (qcache_kernels.cuh): select as given
  const bool given = CALIBRATE == 0 || P.st.score_mode[h] == HARDKV_SCORE_ACCUM_QCACHE;
  if (!given) {
    // softmax in the base-2 domain: exp(z/T - m) = 2^(z*c2 - m2), c2 = log2(e)/T (one FFMA + one MUFU.EX2)
    const float c2 = 1.4426950408889634f / P.st.temperature[unit];
    // SNAPKV heads calibrate the max-pooled copy of their logits (L278; metric_kernels.cuh), all others the raw logits
    const float *lg = ((P.pool_kernel > 1 && P.st.score_mode[h] == HARDKV_SCORE_SNAPKV) ? P.pooled : P.st.logits) +
                      ((size_t)(b * P.Hq + h * G)) * P.max_ctx;
    float mg[GMAX], rs[GMAX];
    if (CALIBRATE == 2) {
      // statistics were produced by the score kernel: one (m2, s) pair per query head and 512-token chunk
      if (C > 1) cluster.barrier_wait();
      const int ch0 = (lo >> 4) / SCORE_PAGES_PER_CTA, ch1 = ((hi - 1) >> 4) / SCORE_PAGES_PER_CTA;
      const float2 *sp = P.score_stats + ((size_t)unit * P.score_chunks) * 8;
      if (warp < G) {   // warp g reduces the chunk statistics of query head g (lanes over chunks)
        const int g = warp;
        float m = -INFINITY, sacc = 0.f;
        for (int c = ch0 + lane; c <= ch1; c += 32) m = fmaxf(m, sel_ld2<COHERENT>(&sp[(size_t)c * 8 + g]).x);
        m = warp_max_f32(m);
        for (int c = ch0 + lane; c <= ch1; c += 32) {
          const float2 v = sel_ld2<COHERENT>(&sp[(size_t)c * 8 + g]);
          sacc += v.y * fast_exp2(v.x - m);
        }
        sacc = warp_sum_f32(sacc);
        if (lane == 0) { sh.st_m[0][g] = m; sh.st_s[0][g] = 1.0f / (sacc * (float)G); }
      }
      __syncthreads();  // statistics published, histogram zeroed
#pragma unroll
      for (int g = 0; g < GMAX; ++g) {
        mg[g] = g < G ? sh.st_m[0][g] : -INFINITY;
        rs[g] = g < G ? sh.st_s[0][g] : 0.f;
      }
    } else {
      // per query head: max and sum of exp over the pool (softmax over the pool only, reading C3)
#pragma unroll
      for (int g = 0; g < GMAX; ++g) {
        if (g >= G) break;
        const float *row = lg + (size_t)g * P.max_ctx;
        float m = -INFINITY, sacc = 0.f;
        for (int i0 = tid; i0 < per; i0 += 4 * NT) {
          float x[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int pos = s0 + i0 + u * NT;
            x[u] = (i0 + u * NT < per && pos >= lo && pos < hi) ? sel_ld<COHERENT>(row + pos) * c2 : -INFINITY;
          }
          const float mn = fmaxf(fmaxf(fmaxf(x[0], x[1]), fmaxf(x[2], x[3])), m);
          if (mn != -INFINITY) {
            sacc = sacc * fast_exp2(m - mn) + fast_exp2(x[0] - mn) + fast_exp2(x[1] - mn) + fast_exp2(x[2] - mn) +
                   fast_exp2(x[3] - mn);
            m = mn;
          }
        }
        const float mw = warp_max_f32(m);
        sacc = warp_sum_f32(mw == -INFINITY ? 0.f : sacc * fast_exp2(m - mw));
        if (lane == 0) { sh.red_f[warp][g][0] = mw; sh.red_f[warp][g][1] = sacc; }
      }
      __syncthreads();
      if (C > 1) cluster.barrier_wait();
      if (tid < C * 8) {  // thread (c, g): publish this CTA's (m_g, s_g) into CTA c
        const int c = tid >> 3, g = tid & 7;
        float m = -INFINITY, sacc = 0.f;
        if (g < G) {
          for (int w = 0; w < NW; ++w) m = fmaxf(m, sh.red_f[w][g][0]);
          for (int w = 0; w < NW; ++w) {
            const float mw = sh.red_f[w][g][0];
            if (mw != -INFINITY) sacc += sh.red_f[w][g][1] * fast_exp2(mw - m);
          }
        }
        SelShared *dst = cluster.map_shared_rank(&sh, c);
        dst->st_m[rank][g] = m;
        dst->st_s[rank][g] = sacc;
      }
      cluster.sync();
#pragma unroll
      for (int g = 0; g < GMAX; ++g) {
        float m = -INFINITY, sacc = 0.f;
        if (g < G) {
          for (int c = 0; c < C; ++c) m = fmaxf(m, sh.st_m[c][g]);
          for (int c = 0; c < C; ++c) {
            const float mc = sh.st_m[c][g];
            if (mc != -INFINITY) sacc += sh.st_s[c][g] * fast_exp2(mc - m);
          }
        }
        mg[g] = m;
        rs[g] = 1.0f / (sacc * (float)G);   // the group mean (reading C2) is folded into the normaliser
      }
    }
    const bool accum = P.st.score_mode[h] == HARDKV_SCORE_ACCUM;
    if (!accum) {
      // S_hat = softmax(z / T) per query head (Solution 1, L120), group mean (reading C2)
      // a thread owns quads of 4 consecutive tokens: one 16-byte load per query head and quad, UQ quads in
      // flight (32 registers of logits), 16-byte stores of the probabilities and of the slice
      constexpr int UQ = 8 / GMAX;
      const int nq = per >> 2;
      for (int q0 = tid; q0 < nq; q0 += UQ * NT) {
        float4 x[UQ][GMAX];
#pragma unroll
        for (int u = 0; u < UQ; ++u) {
          const int qd = q0 + u * NT, pos = s0 + 4 * qd;
          const bool live = qd < nq && pos < hi && pos + 3 >= lo;
          const bool vec = pos + 3 < P.max_ctx;     // the quad lies inside the logits row
#pragma unroll
          for (int g = 0; g < GMAX; ++g) {
            x[u][g] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (live && g < G) {
              const float *src = lg + (size_t)g * P.max_ctx + pos;
              if (vec) {
                x[u][g] = sel_ld4<COHERENT>(reinterpret_cast<const float4 *>(src));
              } else {
                if (pos < P.max_ctx) x[u][g].x = sel_ld<COHERENT>(src);
                if (pos + 1 < P.max_ctx) x[u][g].y = sel_ld<COHERENT>(src + 1);
                if (pos + 2 < P.max_ctx) x[u][g].z = sel_ld<COHERENT>(src + 2);
              }
            }
          }
        }
#pragma unroll
        for (int u = 0; u < UQ; ++u) {
          const int qd = q0 + u * NT, pos = s0 + 4 * qd;
          if (qd >= nq) break;
          float pr[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int g = 0; g < GMAX; ++g) {
            if (g < G) {
              pr[0] = fmaf(fast_exp2(fmaf(x[u][g].x, c2, -mg[g])), rs[g], pr[0]);
              pr[1] = fmaf(fast_exp2(fmaf(x[u][g].y, c2, -mg[g])), rs[g], pr[1]);
              pr[2] = fmaf(fast_exp2(fmaf(x[u][g].z, c2, -mg[g])), rs[g], pr[2]);
              pr[3] = fmaf(fast_exp2(fmaf(x[u][g].w, c2, -mg[g])), rs[g], pr[3]);
            }
          }
          uint32_t bits[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const bool okk = pos + e >= lo && pos + e < hi;
            bits[e] = okk ? __float_as_uint(pr[e]) : SEL_INVALID;
            if (okk) { bits[e] = min(bits[e], SEL_ONE); hist_add(sh, bits[e] >> 20, bits[e]); }
          }
          if (pos >= lo && pos + 3 < hi) {
            *reinterpret_cast<float4 *>(probs + pos) = make_float4(pr[0], pr[1], pr[2], pr[3]);
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
              if (bits[e] != SEL_INVALID) probs[pos + e] = pr[e];
          }
          *reinterpret_cast<uint4 *>(pbits + 4 * qd) = make_uint4(bits[0], bits[1], bits[2], bits[3]);
        }
      }
    } else {
      // ACCUM (reading C4): sliding sum of the last accum_window per-step rows, renormalised.
      const int slot = P.st.ring_slot[unit];
      float *acc = P.st.acc + (size_t)unit * P.max_ctx;
      float *ring = P.st.ring + ((size_t)unit * P.accum_window + slot) * P.max_ctx;
      double tot = 0.0;
      // a thread owns quads of 4 consecutive tokens (s0 and max_ctx are multiples of 4: every row is 16-byte aligned at
      // a quad): one 16-byte load per query head, of acc and of the ring row, 16-byte stores; quads that straddle the
      // pool's ends or the row's end take the scalar path.  Per-token arithmetic is unchanged.
      const int nq = per >> 2;
      for (int qd = tid; qd < nq; qd += NT) {
        const int pos = s0 + 4 * qd;
        uint32_t bits[4] = {SEL_INVALID, SEL_INVALID, SEL_INVALID, SEL_INVALID};
        if (pos >= lo && pos + 3 < hi && pos + 3 < P.max_ctx) {
          const float4 a4 = *reinterpret_cast<const float4 *>(acc + pos), r4 = *reinterpret_cast<const float4 *>(ring + pos);
          float pr[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int g0 = 0; g0 < GMAX; g0 += 4) {     // four heads' loads in flight at a time (registers), heads in order
            float4 x[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
              if (g0 + u < G) x[u] = sel_ld4<COHERENT>(reinterpret_cast<const float4 *>(lg + (size_t)(g0 + u) * P.max_ctx + pos));
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              if (g0 + u < G) {
                pr[0] = fmaf(fast_exp2(fmaf(x[u].x, c2, -mg[g0 + u])), rs[g0 + u], pr[0]);
                pr[1] = fmaf(fast_exp2(fmaf(x[u].y, c2, -mg[g0 + u])), rs[g0 + u], pr[1]);
                pr[2] = fmaf(fast_exp2(fmaf(x[u].z, c2, -mg[g0 + u])), rs[g0 + u], pr[2]);
                pr[3] = fmaf(fast_exp2(fmaf(x[u].w, c2, -mg[g0 + u])), rs[g0 + u], pr[3]);
              }
            }
          }
          const float ao[4] = {a4.x, a4.y, a4.z, a4.w}, ro[4] = {r4.x, r4.y, r4.z, r4.w};
          float an[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            an[e] = fmaxf((ao[e] - ro[e]) + pr[e], 0.f);
            tot += (double)an[e];
            bits[e] = __float_as_uint(an[e]);     // acc for now; normalised below
          }
          *reinterpret_cast<float4 *>(acc + pos) = make_float4(an[0], an[1], an[2], an[3]);
          *reinterpret_cast<float4 *>(ring + pos) = make_float4(pr[0], pr[1], pr[2], pr[3]);
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int pe = pos + e;
            if (pe >= lo && pe < hi) {
              float pr = 0.f;
#pragma unroll
              for (int g = 0; g < GMAX; ++g)
                if (g < G) pr = fmaf(fast_exp2(fmaf(sel_ld<COHERENT>(lg + (size_t)g * P.max_ctx + pe), c2, -mg[g])), rs[g], pr);
              float a = (acc[pe] - ring[pe]) + pr;
              a = fmaxf(a, 0.f);
              acc[pe] = a;
              ring[pe] = pr;
              tot += (double)a;
              bits[e] = __float_as_uint(a);
            }
          }
        }
        *reinterpret_cast<uint4 *>(pbits + 4 * qd) = make_uint4(bits[0], bits[1], bits[2], bits[3]);
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) sh.red_d[warp] = tot;
      __syncthreads();
      if (tid < C) {
        double t = 0.0;
        for (int w = 0; w < NW; ++w) t += sh.red_d[w];
        cluster.map_shared_rank(&sh, tid)->acc_tot[rank] = t;
      }
      cluster.sync();
      tot = 0.0;
      for (int c = 0; c < C; ++c) tot += sh.acc_tot[c];
      for (int qd = tid; qd < nq; qd += NT) {
        const uint4 ab4 = *reinterpret_cast<const uint4 *>(pbits + 4 * qd);
        const uint32_t ab[4] = {ab4.x, ab4.y, ab4.z, ab4.w};
        uint32_t nb[4];
        float pr[4];
        bool whole = true;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          nb[e] = SEL_INVALID; pr[e] = 0.f;
          if (ab[e] == SEL_INVALID) { whole = false; continue; }
          pr[e] = tot > 0.0 ? (float)((double)__uint_as_float(ab[e]) / tot) : 0.f;
          nb[e] = min(__float_as_uint(pr[e]), SEL_ONE);
          hist_add(sh, nb[e] >> 20, nb[e]);
        }
        const int pos = s0 + 4 * qd;
        if (whole) {
          *reinterpret_cast<float4 *>(probs + pos) = make_float4(pr[0], pr[1], pr[2], pr[3]);
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e)
            if (nb[e] != SEL_INVALID) probs[pos + e] = pr[e];
        }
        *reinterpret_cast<uint4 *>(pbits + 4 * qd) = make_uint4(nb[0], nb[1], nb[2], nb[3]);
      }
      if (rank == 0 && tid == 0) P.st.ring_slot[unit] = (slot + 1) % P.accum_window;
    }
  } else {
    __syncthreads();  // histogram zeroed
    if (C > 1) cluster.barrier_wait();
    float psum = 0.f;
    for (int i = tid; i < per; i += NT) {
      const int pos = s0 + i;
      uint32_t bits = SEL_INVALID;
      if (pos >= lo && pos < hi) {
        bits = min(__float_as_uint(probs[pos]) & 0x7fffffffu, SEL_ONE);
        hist_add(sh, bits >> 20, bits);
        psum += __uint_as_float(bits);
      }
      pbits[i] = bits;
    }
    // probabilities given by the caller: the split mass counters of a bin are exact while the row sums to < 4096.  A row
    // in which any warp's share sums to more than 4 is not a probability row (a normalised row sums to 1): flag it
    // (err_flag 3); below that bound the whole row stays under 4 * 32 warps * 8 CTAs = 1024, far from the overflow.
    psum = warp_sum_f32(psum);
    if (lane == 0 && psum > 4.0f) atomicCAS(P.st.err_flag, 0, 3);
  }

  // ---------------- 2b: Top-p threshold --------------------------------------------------------
  const bool all = (p >= 1.0f) || (N <= P.st.l_lower[b]);  // no sparsity yet (L197, reading C8)
  const int kt = P.k_cap;                                   // reading C6: k = min(k_topp, k_cap), same order
  uint32_t tau = 0;          // bit pattern of the smallest selected P
  int r_ties = 0x7fffffff;   // how many tokens with P == tau are taken (ascending position)
  int k = 0;
  {
    uint32_t prefix = 0;
    unsigned long long theta = ~0ull, cum_mass = 0;
    int cum_cnt = 0, bin_cnt = 0;
    bool everything = false, single = false;
#pragma unroll 1
    for (int level = 0; level < 3; ++level) {
      const int db = 10;                            // digit bits: 3 x 10 = the 30 significant bits
      const int shift = level == 0 ? 20 : (level == 1 ? 10 : 0);
      const int nb = 1 << db;
      if (level > 0) {
        // histogram of the next digit over the tokens whose high bits equal the prefix
        for (int d = tid; d < nb; d += NT) { sh.h_cnt[d] = 0; sh.h_hi[d] = 0; sh.h_lo[d] = 0; }
        __syncthreads();
        const int hs = shift + db;
        for (int i = tid * 4; i < per; i += 4 * NT) {
          const uint4 b4 = *reinterpret_cast<const uint4 *>(pbits + i);
          if ((b4.x >> hs) == prefix) hist_add(sh, (b4.x >> shift) & (nb - 1), b4.x);
          if ((b4.y >> hs) == prefix) hist_add(sh, (b4.y >> shift) & (nb - 1), b4.y);
          if ((b4.z >> hs) == prefix) hist_add(sh, (b4.z >> shift) & (nb - 1), b4.z);
          if ((b4.w >> hs) == prefix) hist_add(sh, (b4.w >> shift) & (nb - 1), b4.w);
        }
      }
      __syncthreads();
      const int S = nb / C;  // bins per owner CTA (>= 128)
      // ---- range pass: thread t takes bpt consecutive bins of this CTA's owner range, from the top (local index
      //      jt = t * bpt + u <-> bin S - 1 - jt); across a cluster it first merges the C local histograms of those
      //      bins over DSMEM.  A warp therefore covers one contiguous sub-range, whose (count, mass) it reduces. ----
      const int bpt = S > NT ? S / NT : 1;   // <= 4
      if (C > 1) cluster.sync();      // A: every local histogram of this level is complete
      {
        unsigned long long tm = 0;
        uint32_t tc = 0;
        if (tid * bpt < S) {
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (u < bpt) {
              const int bl = S - 1 - (tid * bpt + u);
              uint32_t c_;
              unsigned long long ms;
              if (C > 1) {
                const int bin = rank * S + bl;
                unsigned long long hi_ = 0, lo_ = 0;
                c_ = 0;
                for (int c = 0; c < C; ++c) {
                  const SelShared *src = cluster.map_shared_rank(&sh, c);
                  c_ += src->h_cnt[bin];
                  hi_ += src->h_hi[bin];
                  lo_ += src->h_lo[bin];
                }
                ms = (hi_ << SEL_MSPLIT) + lo_;
                sh.m_cnt[bl] = c_;
                sh.m_mass[bl] = ms;
              } else {
                c_ = sh.h_cnt[bl];
                ms = ((unsigned long long)sh.h_hi[bl] << SEL_MSPLIT) + sh.h_lo[bl];
              }
              tc += c_;
              tm += ms;
            }
          }
        }
        tm = warp_sum_u64(tm);
        tc = __reduce_add_sync(0xffffffffu, tc);
        if (lane == 0) { sh.red_u[warp] = tm; sh.red_c[warp] = tc; }
      }
      __syncthreads();
      if (C > 1) {
        if (tid < C) {
          unsigned long long m_ = 0;
          uint32_t c_ = 0;
          for (int w = 0; w < NW; ++w) { m_ += sh.red_u[w]; c_ += sh.red_c[w]; }
          SelShared *dst = cluster.map_shared_rank(&sh, tid);
          dst->tot_mass[rank] = m_;
          dst->tot_cnt[rank] = c_;
        }
        cluster.sync();      // B: merged ranges and range totals are visible
      }
      if (warp == 0) {
        // ---- walk from the top: every CTA finds the owner range q of the crossing from the range totals; the
        //      owner descends warp sub-range -> lane -> bin on its own (local) data and publishes the result ----
        int q = 0;
        if (C > 1) {
          if (level == 0) {
            unsigned long long wtot = 0;
            for (int c = 0; c < C; ++c) wtot += sh.tot_mass[c];
            if (!all) {
              // Theta = ceil(p * Wtot) in double: one correctly rounded multiply, identical on host and device
              theta = (unsigned long long)ceil(__dmul_rn((double)p, (double)wtot));
              if (theta < 1) theta = 1;
              if (theta > wtot) theta = ~0ull;  // unreachable mass (Wtot == 0): the nucleus is the whole pool
            }
            everything = (theta == ~0ull && N <= kt);
          }
          if (!everything) {
            for (q = C - 1; q > 0; --q) {
              const unsigned long long rm = sh.tot_mass[q];
              const int rc = (int)sh.tot_cnt[q];
              if ((theta != ~0ull && cum_mass + rm >= theta) || cum_cnt + rc >= kt) break;
              cum_mass += rm;
              cum_cnt += rc;
            }
          }
        }
        const bool walker = C == 1 || rank == q;
        const int nwr = (S / bpt) / 32;                     // active warp sub-ranges (<= 16)
        unsigned long long lm = lane < nwr ? sh.red_u[lane] : 0ull;
        int lc = lane < nwr ? (int)sh.red_c[lane] : 0;
        if (C == 1 && level == 0) {
          const unsigned long long wtot = warp_sum_u64(lm);
          if (!all) {
            theta = (unsigned long long)ceil(__dmul_rn((double)p, (double)wtot));
            if (theta < 1) theta = 1;
            if (theta > wtot) theta = ~0ull;
          }
          everything = (theta == ~0ull && N <= kt);
        }
        if (!everything && walker) {
          // crossing test of an inclusive prefix: theta <= Wtot guarantees the mass condition at the latest in the
          // lowest non-empty bin, and theta == inf implies N > kt so the count condition fires; the last element is
          // taken unconditionally at every level to keep the walk total.
          // level A: the warp sub-ranges (lane w holds sub-range w, top first)
          unsigned long long im = lm;
          int ic = lc;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long om = shfl_up_u64(im, o);
            const int oc = __shfl_up_sync(0xffffffffu, ic, o);
            if (lane >= o) { im += om; ic += oc; }
          }
          const unsigned cmA = __ballot_sync(0xffffffffu, (theta != ~0ull && cum_mass + im >= theta) || cum_cnt + ic >= kt);
          const int wr = cmA ? min(__ffs(cmA) - 1, nwr - 1) : nwr - 1;
          const unsigned long long baseA_m = cum_mass + shfl_u64(im - lm, wr);
          const int baseA_c = cum_cnt + __shfl_sync(0xffffffffu, ic - lc, wr);
          // level B: the 32 lanes of sub-range wr, bpt bins each
          unsigned long long bm[4] = {0, 0, 0, 0};
          int bc[4] = {0, 0, 0, 0};
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (u < bpt) {
              const int bl = S - 1 - ((wr * 32 + lane) * bpt + u);
              if (C > 1) { bc[u] = (int)sh.m_cnt[bl]; bm[u] = sh.m_mass[bl]; }
              else { bc[u] = (int)sh.h_cnt[bl]; bm[u] = ((unsigned long long)sh.h_hi[bl] << SEL_MSPLIT) + sh.h_lo[bl]; }
            }
          }
          const unsigned long long lm2 = bm[0] + bm[1] + bm[2] + bm[3];
          const int lc2 = bc[0] + bc[1] + bc[2] + bc[3];
          unsigned long long im2 = lm2;
          int ic2 = lc2;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long om = shfl_up_u64(im2, o);
            const int oc = __shfl_up_sync(0xffffffffu, ic2, o);
            if (lane >= o) { im2 += om; ic2 += oc; }
          }
          const unsigned cmB = __ballot_sync(0xffffffffu, (theta != ~0ull && baseA_m + im2 >= theta) || baseA_c + ic2 >= kt);
          const int cl2 = cmB ? __ffs(cmB) - 1 : 31;
          int r_bin = 0, r_bc = 0, r_cc = 0;
          unsigned long long r_cm = 0;
          if (lane == cl2) {
            // level C: the (<= 4) bins of the crossing lane
            unsigned long long m_ = baseA_m + (im2 - lm2);
            int c_ = baseA_c + (ic2 - lc2);
            int u = 0;
#pragma unroll
            for (int v = 0; v < 3; ++v) {
              if (u == v && v + 1 < bpt && !((theta != ~0ull && m_ + bm[v] >= theta) || c_ + bc[v] >= kt)) {
                m_ += bm[v]; c_ += bc[v]; u = v + 1;
              }
            }
            r_bin = q * S + (S - 1 - ((wr * 32 + lane) * bpt + u));
            r_bc = u == 0 ? bc[0] : (u == 1 ? bc[1] : (u == 2 ? bc[2] : bc[3]));
            r_cc = c_; r_cm = m_;
          }
          r_bin = __shfl_sync(0xffffffffu, r_bin, cl2);
          r_bc = __shfl_sync(0xffffffffu, r_bc, cl2);
          r_cc = __shfl_sync(0xffffffffu, r_cc, cl2);
          r_cm = shfl_u64(r_cm, cl2);
          if (lane < C) {
            SelShared *dst = C > 1 ? cluster.map_shared_rank(&sh, lane) : &sh;
            dst->res_bin = r_bin; dst->res_bin_cnt = r_bc; dst->res_cum_cnt = r_cc; dst->res_cum_mass = r_cm;
          }
        } else if (everything && lane == 0) {
          sh.res_bin = -1;
        }
        if (lane == 0) sh.res_theta = theta;
      }
      if (C > 1) cluster.sync();   // C: the owner's result has landed in every CTA
      else __syncthreads();
      theta = sh.res_theta;
      if (sh.res_bin < 0) { everything = true; break; }
      prefix = (prefix << db) | (uint32_t)sh.res_bin;
      bin_cnt = sh.res_bin_cnt;
      cum_cnt = sh.res_cum_cnt;
      cum_mass = sh.res_cum_mass;
      // a crossing bin that holds one token ends the descent: that token is the last of the nucleus, whatever its
      // remaining digits (every CTA reads the same bin_cnt, so the exit is uniform over the cluster)
      if (bin_cnt == 1 && level < 2) { single = true; prefix <<= shift; break; }
      // the next level rewrites sh.h_* (after its own __syncthreads) and sh.res_* (after two more barriers)
    }
    if (everything) {
      k = N;  // tau = 0, all ties taken
    } else if (single) {
      tau = prefix;   // low digits zero: the token is > tau, or == tau and the one tie taken
      r_ties = 1;
      k = cum_cnt + 1;
    } else {
      tau = prefix;
      const unsigned long long wt = mass_of_bits(tau);
      long long r = bin_cnt;
      if (theta != ~0ull && wt > 0) {
        const unsigned long long need = theta - cum_mass;  // > 0: the prefix before this bin is short
        const unsigned long long rm = (need + wt - 1) / wt;
        if ((long long)rm < r) r = (long long)rm;
      }
      if ((long long)(kt - cum_cnt) < r) r = kt - cum_cnt;
      r_ties = (int)r;
      k = cum_cnt + r_ties;
    }
  }

  // ---------------- 2c: stream compaction in ascending position order -----------------------------
  // A lane owns 4 consecutive tokens of every 128-token group of its warp's segment (one 16-byte LDS); lane-major order
  // is position order.  Slice entries outside the pool are SEL_INVALID (> every probability): `valid` masks them.
  const int w0 = warp * wseg;  // this warp's contiguous segment of the slice (a multiple of 32 tokens)
  {
    int gt = 0, tie = 0;
    for (int i = w0 + 4 * lane; i < w0 + wseg; i += 128) {
      const uint4 v = *reinterpret_cast<const uint4 *>(pbits + i);
      gt += (v.x > tau && v.x != SEL_INVALID) + (v.y > tau && v.y != SEL_INVALID) + (v.z > tau && v.z != SEL_INVALID) +
            (v.w > tau && v.w != SEL_INVALID);
      tie += (v.x == tau) + (v.y == tau) + (v.z == tau) + (v.w == tau);
    }
    gt = __reduce_add_sync(0xffffffffu, gt);
    tie = __reduce_add_sync(0xffffffffu, tie);
    if (lane == 0) { sh.w_gt[warp] = gt; sh.w_tie[warp] = tie; }
  }
  __syncthreads();
  int tie_before = 0, sel_before = 0;
  if (C > 1) {
    if (tid < C) {
      int g_ = 0, t_ = 0;
      for (int w = 0; w < NW; ++w) { g_ += sh.w_gt[w]; t_ += sh.w_tie[w]; }
      SelShared *dst = cluster.map_shared_rank(&sh, tid);
      dst->c_gt[rank] = g_;
      dst->c_tie[rank] = t_;
    }
    cluster.sync();
    for (int c = 0; c < rank; ++c) {
      const int tw = sh.c_tie[c];
      int take = r_ties - tie_before;
      take = take < 0 ? 0 : (take > tw ? tw : take);
      sel_before += sh.c_gt[c] + take;
      tie_before += tw;
    }
  }
  {
    // this warp's offsets from the per-warp counts, in parallel: lane l stands for warp l (ties are taken in position
    // order, r_ties in all: a warp takes what is left when the ties of the warps before it are counted)
    const int tw = lane < NW ? sh.w_tie[lane] : 0, gw = lane < NW ? sh.w_gt[lane] : 0;
    int tpre = tw;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t_ = __shfl_up_sync(0xffffffffu, tpre, o);
      if (lane >= o) tpre += t_;
    }
    int take = r_ties - (tie_before + tpre - tw);
    take = take < 0 ? 0 : (take > tw ? tw : take);
    sel_before += __reduce_add_sync(0xffffffffu, lane < warp ? gw + take : 0);
    tie_before += __reduce_add_sync(0xffffffffu, lane < warp ? tw : 0);
  }
  int32_t *votes = P.st.votes + (size_t)unit * P.max_ctx;
  for (int g0 = w0; g0 < w0 + wseg; g0 += 128) {
    const int pos0 = s0 + g0;               // multiple of 32
    if (pos0 >= hi) break;                  // warp-uniform
    const int i = g0 + 4 * lane;
    uint4 v = make_uint4(SEL_INVALID, SEL_INVALID, SEL_INVALID, SEL_INVALID);
    if (i < w0 + wseg) v = *reinterpret_cast<const uint4 *>(pbits + i);
    const uint32_t bq[4] = {v.x, v.y, v.z, v.w};
    unsigned m = 0, tq = 0;                 // 4-bit masks of this lane: selected because > tau / equal to tau
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      m |= (unsigned)(bq[e] > tau && bq[e] != SEL_INVALID) << e;
      tq |= (unsigned)(bq[e] == tau) << e;
    }
    if (!want_mask && !__any_sync(0xffffffffu, (m | tq) != 0)) continue;   // most groups of a sparse head hold nothing
    int ntie = 0;
    if (__any_sync(0xffffffffu, tq != 0)) {
      // ties (rare: usually the one token that is the threshold): the first r_ties of them in position order are taken
      ntie = __popc(tq);
      int tpre = ntie;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t_ = __shfl_up_sync(0xffffffffu, tpre, o);
        if (lane >= o) tpre += t_;
      }
      const int tall = __shfl_sync(0xffffffffu, tpre, 31);
      int seen = tie_before + tpre - ntie;
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        if ((tq >> e) & 1) { m |= (unsigned)(seen < r_ties) << e; ++seen; }
      }
      tie_before += tall;
    }
    const int cnt = __popc(m);
    int pre = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t_ = __shfl_up_sync(0xffffffffu, pre, o);
      if (lane >= o) pre += t_;
    }
    const int call = __shfl_sync(0xffffffffu, pre, 31);
    if (m) {
      int dst = sel_before + pre - cnt;
      const int pos = pos0 + 4 * lane;
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        if ((m >> e) & 1) {
          sel_idx[dst++] = pos + e;
          atomicAdd(votes + pos + e, 1);  // cumulative selection mask = votes (L86); result unused -> RED, no round trip
        }
      }
    }
    if (want_mask) {  // bit i%8 of byte i/8 (L439): byte y holds tokens 8y..8y+7 = the nibbles of lanes 2y, 2y + 1
      const unsigned hi_nib = __shfl_down_sync(0xffffffffu, m, 1);
      const int y = (pos0 >> 3) + (lane >> 1);
      if ((lane & 1) == 0 && i < w0 + wseg && y < mask_bytes) mask[y] = (uint8_t)(m | (hi_nib << 4));
    }
    sel_before += call;
  }
  // pads, the head-wise block table (reading C9; L207-209) and the mask bytes outside the slices
  const int gt_ = rank * NT + tid, gs_ = C * NT;
  for (int j = k + gt_; j < P.k_cap; j += gs_) sel_idx[j] = -1;
  const int used = (k + PAGE - 1) / PAGE;
  const int32_t *sp = P.st.sel_pages + (size_t)unit * P.spu;
  for (int j = gt_; j < P.spu; j += gs_) sel_table[j] = j < used ? sp[j] : -1;
  if (rank == 0 && tid == 0) P.st.sel_count[unit] = k;
  if (want_mask) {
    const int y0 = base >> 3, y1 = min(mask_bytes, ((hi + 31) & ~31) >> 3);
    for (int y = gt_; y < y0; y += gs_) mask[y] = 0;
    for (int y = y1 + gt_; y < mask_bytes; y += gs_) mask[y] = 0;
  }
  if (C > 1) cluster.sync();  // no CTA may exit while a peer can still read its shared memory
  else __syncthreads();
  // publish: every thread's stores of this unit (sel_idx, sel_count, sel_table, votes) happen before the barrier above,
  // the fence is cumulative, then the flag -- the attention kernel may already be waiting for it (wait_unit_selected)
  if (rank == 0 && tid == 0 && P.sel_flag) {
    __threadfence();
    *reinterpret_cast<volatile int32_t *>(P.sel_flag + unit) = *reinterpret_cast<volatile int32_t *>(P.epoch);
  }
}

// One thread-block cluster (or one CTA) per (sequence, KV head).
template <int CALIBRATE, int GMAX, int NT>
__global__ void __launch_bounds__(NT, NT == SEL_NT_BIG ? 1 : 2) select_kernel(Params P, float p) {
  pdl_wait_then_trigger();
  KernelClock kclock(P);
  extern __shared__ __align__(16) unsigned char sel_smem[];
  uint32_t *pbits = reinterpret_cast<uint32_t *>(sel_smem);                       // [P.sel_slice_cap]
  SelShared &sh = *reinterpret_cast<SelShared *>(sel_smem + (size_t)P.sel_slice_cap * 4);
  select_unit<CALIBRATE, GMAX, NT, true, false>(P, p, blockIdx.x / P.sel_cluster, pbits, sh);
}

// The select half of the score || select overlap (hardkv_decode_step, variant 4): launched programmatically behind the
// publishing score_tma_kernel; cluster j takes the unit the score kernel finishes j-th (longest pool first), waits for
// its flag and reads the logits / chunk statistics with L2-coherent loads.  512-thread CTAs whose shared memory and
// registers fit beside a score CTA on the same SM.
template <int GMAX>
__global__ void __launch_bounds__(SEL_NT, 2) select_overlap_kernel(Params P, float p) {
  pdl_trigger();
  KernelClock kclock(P);
  extern __shared__ __align__(16) unsigned char sel_smem[];
  uint32_t *pbits = reinterpret_cast<uint32_t *>(sel_smem);
  SelShared &sh = *reinterpret_cast<SelShared *>(sel_smem + (size_t)P.sel_slice_cap * 4);
  const int units = P.B * P.Hkv;
  const int unit = P.unit_order[units - 1 - (int)blockIdx.x / P.sel_cluster];
  int n, lo, hi;
  pool_bounds(P, unit / P.Hkv, n, lo, hi);
  if (hi > lo) wait_unit_scored(P, unit);     // an empty pool has no chunk: nothing is published for it
  select_unit<2, GMAX, SEL_NT, true, true>(P, p, unit, pbits, sh);
}

}  // namespace hardkv
