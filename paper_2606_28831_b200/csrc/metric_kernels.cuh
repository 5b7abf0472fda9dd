// metric_kernels.cuh -- the second importance metric and the temperature solve of Logits Calibration.
//   * SNAPKV metric: g = max-pool of the raw logits along the sequence (odd window, stride 1,
//     clipped to the pool; reading C15), written to a workspace copy that the select kernel calibrates
//     instead of the raw logits (Solution 1, L120: S_hat = S(g(z / T)); g(z / T) = g(z) / T for T > 0).
//   * Algorithm 2 "Binary Search on T" (L625-648, readings C14 / C16) for Problem 1 (L108-110): per KV head,
//     k = Num_Selected_TopP(S, p) on the raw attention scores, then bisection on T until the Top-k mass of the
//     calibrated metric matches M_k(S).  Run once per request (L607), so it is written for clarity, not speed: one
//     CTA per (sequence, KV head), probabilities round-trip through the unit's `probs` row (L2 resident), the Top-k
//     mass comes from the same 3 x 10-bit radix descent on the fp32 pattern with exact integer mass as the select
//     kernel (reading C5).
#pragma once
#include "common.cuh"
#include "select_kernel.cuh"

namespace hardkv {

constexpr int POOL_TOK = 1024;   // tokens per CTA of the pooling kernel

__global__ void __launch_bounds__(256) maxpool_kernel(Params P) {
  KernelClock kclock(P);
  const int unit = blockIdx.y, b = unit / P.Hkv, h = unit % P.Hkv;
  if (P.st.score_mode[h] != HARDKV_SCORE_SNAPKV) return;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  const int i0 = blockIdx.x * POOL_TOK, i1 = min(i0 + POOL_TOK, hi);
  if (i0 >= hi || i1 <= lo) return;
  const int r = (P.pool_kernel - 1) / 2;
  for (int g = 0; g < P.G; ++g) {
    const size_t ro = ((size_t)(b * P.Hq + h * P.G + g)) * P.max_ctx;
    const float *row = P.st.logits + ro;
    float *dst = P.pooled + ro;
    for (int i = max(i0, lo) + threadIdx.x; i < i1; i += blockDim.x) {
      float m = __ldg(row + i);
      const int j0 = max(lo, i - r), j1 = min(hi - 1, i + r);
      for (int j = j0; j <= j1; ++j) m = fmaxf(m, __ldg(row + j));
      dst[i] = m;
    }
  }
}

constexpr int SOLVE_NT = 1024;
constexpr int SOLVE_NW = SOLVE_NT / 32;

struct SolveShared {
  uint32_t cnt[SEL_NB];
  unsigned long long mass[SEL_NB];
  float red[SOLVE_NW][8];
  float st_m[8], st_r[8];
  int res_bin, res_bin_cnt, res_cum_cnt, res_none;
  unsigned long long res_cum_mass, wtot;
};

// P[i] = (1/G) sum_g 2^(x_g[i] c2 - m_g) / s_g over the pool -> probs row (reading C2, C3); whole CTA.
__device__ void solve_eval_probs(const Params &P, SolveShared &sh, const float *rows, float c2, int lo, int hi,
                                 float *probs) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, G = P.G;
  for (int g = 0; g < G; ++g) {
    float m = -INFINITY;
    for (int i = lo + tid; i < hi; i += SOLVE_NT) m = fmaxf(m, __ldg(rows + (size_t)g * P.max_ctx + i) * c2);
    m = warp_max_f32(m);
    if (lane == 0) sh.red[warp][g] = m;
  }
  __syncthreads();
  if (tid < G) {
    float m = -INFINITY;
    for (int w = 0; w < SOLVE_NW; ++w) m = fmaxf(m, sh.red[w][tid]);
    sh.st_m[tid] = m;
  }
  __syncthreads();
  for (int g = 0; g < G; ++g) {
    const float m = sh.st_m[g];
    float s = 0.f;
    for (int i = lo + tid; i < hi; i += SOLVE_NT) s += fast_exp2(fmaf(__ldg(rows + (size_t)g * P.max_ctx + i), c2, -m));
    s = warp_sum_f32(s);
    if (lane == 0) sh.red[warp][g] = s;
  }
  __syncthreads();
  if (tid < G) {
    float s = 0.f;
    for (int w = 0; w < SOLVE_NW; ++w) s += sh.red[w][tid];
    sh.st_r[tid] = 1.0f / (s * (float)G);
  }
  __syncthreads();
  for (int i = lo + tid; i < hi; i += SOLVE_NT) {
    float pr = 0.f;
    for (int g = 0; g < G; ++g)
      pr = fmaf(fast_exp2(fmaf(__ldg(rows + (size_t)g * P.max_ctx + i), c2, -sh.st_m[g])), sh.st_r[g], pr);
    probs[i] = pr;
  }
  __syncthreads();
}

// Walk of the order (bits desc, position asc) over the probs row.  kcount < 0: mass mode, stop where the integer mass
// reaches Theta = ceil(p * Wtot) (Num_Selected_TopP); kcount >= 0: count mode, stop at kcount tokens.
// Returns k; *mass_k = integer mass of the first k tokens, *wtot = total integer mass.  Whole CTA, uniform result.
__device__ int solve_descend(SolveShared &sh, const float *probs, int lo, int hi, float p, int kcount,
                             unsigned long long *mass_k, unsigned long long *wtot_out) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint32_t prefix = 0;
  unsigned long long theta = ~0ull, cum_mass = 0, wtot = 0;
  int cum_cnt = 0, bin_cnt = 0;
  for (int level = 0; level < 3; ++level) {
    const int shift = 20 - 10 * level;
    for (int d = tid; d < SEL_NB; d += SOLVE_NT) { sh.cnt[d] = 0; sh.mass[d] = 0; }
    __syncthreads();
    for (int i = lo + tid; i < hi; i += SOLVE_NT) {
      const uint32_t bits = min(__float_as_uint(probs[i]) & 0x7fffffffu, SEL_ONE);
      if (level == 0 || (bits >> (shift + 10)) == prefix) {
        const int bin = (bits >> shift) & (SEL_NB - 1);
        atomicAdd(&sh.cnt[bin], 1u);
        atomicAdd(&sh.mass[bin], mass_of_bits(bits));
      }
    }
    __syncthreads();
    if (warp == 0) {
      // lane l owns bins 1023 - 32 l ... 1023 - 32 l - 31 (top first)
      unsigned long long lm = 0;
      int lc = 0;
      for (int u = 0; u < 32; ++u) { lm += sh.mass[SEL_NB - 1 - (32 * lane + u)]; lc += (int)sh.cnt[SEL_NB - 1 - (32 * lane + u)]; }
      if (level == 0) {
        wtot = warp_sum_u64(lm);
        if (kcount < 0) {
          theta = (unsigned long long)ceil(__dmul_rn((double)p, (double)wtot));
          if (theta < 1) theta = 1;
        }
      }
      unsigned long long im = lm;
      int ic = lc;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long om = shfl_up_u64(im, o);
        const int oc = __shfl_up_sync(0xffffffffu, ic, o);
        if (lane >= o) { im += om; ic += oc; }
      }
      const bool cross = kcount < 0 ? (cum_mass + im >= theta) : (cum_cnt + ic >= kcount);
      const unsigned cm = __ballot_sync(0xffffffffu, cross);
      if (cm == 0) {
        if (lane == 0) sh.res_none = 1;     // unreachable mass / count: everything is taken
      } else if (lane == __ffs(cm) - 1) {
        unsigned long long m_ = cum_mass + (im - lm);
        int c_ = cum_cnt + (ic - lc), u = 0;
        for (; u < 31; ++u) {
          const int bin = SEL_NB - 1 - (32 * lane + u);
          const bool hit = kcount < 0 ? (m_ + sh.mass[bin] >= theta) : (c_ + (int)sh.cnt[bin] >= kcount);
          if (hit) break;
          m_ += sh.mass[bin]; c_ += (int)sh.cnt[bin];
        }
        const int bin = SEL_NB - 1 - (32 * lane + u);
        sh.res_none = 0; sh.res_bin = bin; sh.res_bin_cnt = (int)sh.cnt[bin]; sh.res_cum_cnt = c_; sh.res_cum_mass = m_;
      }
      if (lane == 0 && level == 0) sh.wtot = wtot;
    }
    __syncthreads();
    wtot = sh.wtot;
    if (kcount < 0 && level == 0) {
      theta = (unsigned long long)ceil(__dmul_rn((double)p, (double)wtot));
      if (theta < 1) theta = 1;
    }
    const bool none = sh.res_none != 0;
    const int rb = sh.res_bin;
    bin_cnt = sh.res_bin_cnt; cum_cnt = none ? cum_cnt : sh.res_cum_cnt; cum_mass = none ? cum_mass : sh.res_cum_mass;
    __syncthreads();   // the next level rewrites sh
    if (none) { *mass_k = wtot; *wtot_out = wtot; return hi - lo; }
    prefix = (prefix << 10) | (uint32_t)rb;
  }
  const unsigned long long wt = mass_of_bits(prefix);
  long long r = bin_cnt;
  if (kcount < 0) {
    if (wt > 0) {
      const unsigned long long need = theta - cum_mass;
      const unsigned long long rm = (need + wt - 1) / wt;
      if ((long long)rm < r) r = (long long)rm;
    }
  } else {
    r = kcount - cum_cnt;
  }
  *mass_k = cum_mass + (unsigned long long)r * wt;
  *wtot_out = wtot;
  return cum_cnt + (int)r;
}

__global__ void __launch_bounds__(SOLVE_NT, 1) solve_temperature_kernel(Params P, float p, float t_min, float t_max,
                                                                        float eps, int max_iter) {
  __shared__ SolveShared sh;
  const int unit = blockIdx.x, b = unit / P.Hkv, h = unit % P.Hkv;
  const int mode = P.st.score_mode[h];
  if (mode == HARDKV_SCORE_ACCUM || mode == HARDKV_SCORE_ACCUM_QCACHE) return;   // readings C4 / C18: accumulated metrics keep their T
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  if (hi <= lo) return;
  const size_t ro = ((size_t)(b * P.Hq + h * P.G)) * P.max_ctx;
  const float *raw = P.st.logits + ro;
  const float *met = (mode == HARDKV_SCORE_SNAPKV && P.pool_kernel > 1) ? P.pooled + ro : raw;
  float *probs = P.st.probs + (size_t)unit * P.max_ctx;
  constexpr float LOG2E = 1.4426950408889634f;

  // line 1: k <- Num_Selected_TopP(S, p) on the raw attention scores (g = id, T = 1)
  solve_eval_probs(P, sh, raw, LOG2E, lo, hi, probs);
  unsigned long long mk = 0, wt = 0;
  const int k = solve_descend(sh, probs, lo, hi, p, p >= 1.0f ? hi - lo : -1, &mk, &wt);
  const double MkS = wt ? (double)mk / (double)wt : 0.0;
  float tlo = t_min, thi = t_max, Tm = P.st.temperature[unit];
  for (int it = 0; it < max_iter; ++it) {
    Tm = 0.5f * (tlo + thi);
    solve_eval_probs(P, sh, met, LOG2E / Tm, lo, hi, probs);
    solve_descend(sh, probs, lo, hi, p, k, &mk, &wt);
    const double MkH = wt ? (double)mk / (double)wt : 0.0;
    const double r = fabs(MkS - MkH);
    if (!(r > (double)eps)) break;
    if (MkS < MkH) tlo = Tm; else thi = Tm;      // S_hat too sharp: raise T (WHERE updates, L640 / L648)
    if (!(tlo < thi)) break;
  }
  if (threadIdx.x == 0) const_cast<float *>(P.st.temperature)[unit] = Tm;
}

}  // namespace hardkv
