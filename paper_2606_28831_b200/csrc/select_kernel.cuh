// select_kernel.cuh -- Logits Calibration (apply-T) + Top-p nucleus + stream compaction.
// One CTA per (sequence, KV head).  PAPER.md L106-128 (calibration), L108 (Top-p), L86 (votes),
// L207-209 / L439 (head-wise block table, packed mask); readings C2-C6, C9.
//
// The nucleus is found without a sort: a most-significant-digit radix descent on the fp32 bit
// pattern of P (all P >= 0, so unsigned order == float order), 5 bits per level.  Each level
// builds, per digit, (count, integer mass) with w_i = rn(P_i * 2^32) in u64: exact and order
// independent, so it reproduces a sorted-prefix definition bit for bit (reading C5).
// Histograms are PRIVATE per thread (hist[digit][tid], one packed u64 = count << 40 | mass):
// plain LDS/STS, no atomics -- shared-memory atomics retire about one lane per clock and would
// bound the whole step on long rows.
#pragma once
#include "common.cuh"

namespace hardkv {

constexpr int SEL_NT = 512;
constexpr int SEL_BINS = 32;
constexpr int SEL_DIGIT = 5;
constexpr int SEL_NW = SEL_NT / 32;
constexpr size_t SEL_SMEM = (size_t)SEL_BINS * SEL_NT * 8;

__device__ __forceinline__ unsigned long long mass_of_bits(uint32_t bits) {
  // w = rn(P * 2^32): the product is exact in fp32 (power-of-two scale), conversion rounds to nearest even
  return __float2ull_rn(__uint_as_float(bits) * 4294967296.0f);
}

struct SelShared {
  float red_f[SEL_NW][8][2];
  unsigned long long red_u[SEL_NW];
  double red_d[SEL_NW];
  unsigned long long bin[SEL_BINS];
  int w_gt[SEL_NW], w_tie[SEL_NW];
  uint32_t mask_words[1];  // placeholder (mask is staged in the histogram area)
};

// CALIBRATE: 1 = logits -> probs (2a) then select; 0 = select on state->probs as given.
template <int CALIBRATE>
__global__ void __launch_bounds__(SEL_NT) select_kernel(Params P, float p) {
  extern __shared__ unsigned long long s_hist[];  // [SEL_BINS][SEL_NT]
  __shared__ SelShared sh;
  const int unit = blockIdx.x, b = unit / P.Hkv, h = unit % P.Hkv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  const int N = hi - lo;
  const int G = P.G;
  float *probs = P.st.probs + (size_t)unit * P.max_ctx;
  int32_t *sel_idx = P.st.sel_idx + (size_t)unit * P.k_cap;
  int32_t *sel_table = P.st.sel_table + (size_t)unit * P.spu;

  // ---------------- 2a: calibration ------------------------------------------------------------
  if (CALIBRATE && N > 0) {
    const float invT = 1.0f / P.st.temperature[unit];
    const float *lg = P.st.logits + ((size_t)(b * P.Hq + h * G)) * P.max_ctx;
    // per query head: max and sum of exp over the pool (softmax over the pool only, reading C3)
    float mg[8], sg[8];
    for (int g = 0; g < G; ++g) {
      float m = -INFINITY, s = 0.f;
      for (int i = lo + tid; i < hi; i += SEL_NT) {
        const float x = __ldcg(lg + (size_t)g * P.max_ctx + i) * invT;
        if (x > m) { s *= expf(m - x); m = x; }
        s += expf(x - m);
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        const float om = __shfl_xor_sync(0xffffffffu, m, o), os = __shfl_xor_sync(0xffffffffu, s, o);
        const float mn = fmaxf(m, om);
        s = (m == -INFINITY ? 0.f : s * expf(m - mn)) + (om == -INFINITY ? 0.f : os * expf(om - mn));
        m = mn;
      }
      if (lane == 0) { sh.red_f[warp][g][0] = m; sh.red_f[warp][g][1] = s; }
    }
    __syncthreads();
    for (int g = 0; g < G; ++g) {
      float m = -INFINITY;
      for (int w = 0; w < SEL_NW; ++w) m = fmaxf(m, sh.red_f[w][g][0]);
      float s = 0.f;
      for (int w = 0; w < SEL_NW; ++w) {
        const float mw = sh.red_f[w][g][0];
        if (mw != -INFINITY) s += sh.red_f[w][g][1] * expf(mw - m);
      }
      mg[g] = m;
      sg[g] = 1.0f / s;
    }
    const float invG = 1.0f / (float)G;
    const bool accum = P.st.score_mode[h] == HARDKV_SCORE_ACCUM;
    if (!accum) {
      // S_hat = softmax(z / T) per query head (Solution 1, L120), group mean (reading C2)
      for (int i = lo + tid; i < hi; i += SEL_NT) {
        float pr = 0.f;
        for (int g = 0; g < G; ++g)
          pr += expf(__ldcg(lg + (size_t)g * P.max_ctx + i) * invT - mg[g]) * sg[g];
        probs[i] = pr * invG;
      }
    } else {
      // ACCUM (reading C4): sliding sum of the last accum_window per-step rows, renormalised.
      const int slot = P.st.ring_slot[unit];
      float *acc = P.st.acc + (size_t)unit * P.max_ctx;
      float *ring = P.st.ring + ((size_t)unit * P.accum_window + slot) * P.max_ctx;
      double tot = 0.0;
      for (int i = lo + tid; i < hi; i += SEL_NT) {
        float pr = 0.f;
        for (int g = 0; g < G; ++g)
          pr += expf(__ldcg(lg + (size_t)g * P.max_ctx + i) * invT - mg[g]) * sg[g];
        pr *= invG;
        float a = (acc[i] - ring[i]) + pr;
        a = fmaxf(a, 0.f);
        acc[i] = a;
        ring[i] = pr;
        tot += (double)a;
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) sh.red_d[warp] = tot;
      __syncthreads();
      tot = 0.0;
      for (int w = 0; w < SEL_NW; ++w) tot += sh.red_d[w];
      for (int i = lo + tid; i < hi; i += SEL_NT)
        probs[i] = tot > 0.0 ? (float)((double)acc[i] / tot) : 0.f;
      if (tid == 0) P.st.ring_slot[unit] = (slot + 1) % P.accum_window;
    }
    __syncthreads();  // probs written by this CTA are read back below
  }

  // ---------------- 2b: Top-p threshold --------------------------------------------------------
  const uint32_t *row = reinterpret_cast<const uint32_t *>(probs) + lo;  // bit patterns of the pool
  uint32_t tau = 0;          // bit pattern of the smallest selected P
  int r_ties = 0x7fffffff;   // how many tokens with P == tau are taken (ascending position)
  int k = 0;
  if (N > 0) {
    const bool all = (p >= 1.0f) || (N <= P.st.l_lower[b]);  // no sparsity yet (L197, reading C8)
    unsigned long long theta = ~0ull;
    if (!all) {
      unsigned long long wsum = 0;
      for (int i = tid; i < N; i += SEL_NT) wsum += mass_of_bits(row[i]);
      wsum = warp_sum_u64(wsum);
      if (lane == 0) sh.red_u[warp] = wsum;
      __syncthreads();
      unsigned long long wtot = 0;
      for (int w = 0; w < SEL_NW; ++w) wtot += sh.red_u[w];
      // Theta = ceil(p * Wtot) in double: one correctly rounded multiply, identical on host and device
      theta = (unsigned long long)ceil(__dmul_rn((double)p, (double)wtot));
      if (theta < 1) theta = 1;
      if (theta > wtot) theta = ~0ull;  // unreachable mass (Wtot == 0): the nucleus is the whole pool
    }
    const int kt = P.k_cap;  // reading C6: k = min(k_topp, k_cap), same order
    if (theta == ~0ull && N <= kt) {
      k = N;  // everything: tau = 0, all ties taken
    } else {
      uint32_t prefix = 0;
      int shift = 31;  // unresolved low bits (bit 31 is the sign: always 0)
      unsigned long long cum_mass = 0;
      int cum_cnt = 0, bin_cnt = 0;
      while (shift > 0) {
        const int db = shift < SEL_DIGIT ? shift : SEL_DIGIT;
        const int nb = 1 << db;
        const int hs = shift;  // bits above the digit: row >> hs == prefix
        shift -= db;
        for (int d = 0; d < nb; ++d) s_hist[d * SEL_NT + tid] = 0ull;
        for (int i = tid; i < N; i += SEL_NT) {
          const uint32_t bits = row[i];
          if ((bits >> hs) == prefix) {
            const int d = (bits >> shift) & (nb - 1);
            s_hist[d * SEL_NT + tid] += (1ull << 40) + mass_of_bits(bits);
          }
        }
        __syncthreads();
        for (int d = warp; d < nb; d += SEL_NW) {
          unsigned long long t = 0;
          for (int c = lane; c < SEL_NT; c += 32) t += s_hist[d * SEL_NT + c];
          t = warp_sum_u64(t);
          if (lane == 0) sh.bin[d] = t;
        }
        __syncthreads();
        int chosen = -1;
        for (int d = nb - 1; d >= 0; --d) {
          const unsigned long long t = sh.bin[d];
          const int c = (int)(t >> 40);
          const unsigned long long ms = t & ((1ull << 40) - 1);
          if ((theta != ~0ull && cum_mass + ms >= theta) || cum_cnt + c >= kt) { chosen = d; bin_cnt = c; break; }
          cum_mass += ms;
          cum_cnt += c;
        }
        // chosen >= 0 always: theta <= Wtot guarantees the mass condition fires at the latest in
        // the lowest digit, and theta == inf implies N > kt so the count condition fires.
        if (chosen < 0) { chosen = 0; bin_cnt = (int)(sh.bin[0] >> 40); }
        prefix = (prefix << db) | (uint32_t)chosen;
        __syncthreads();  // sh.bin / s_hist are rewritten by the next level
      }
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
  uint32_t *s_mask = reinterpret_cast<uint32_t *>(s_hist);  // packed mask staged in shared memory
  const bool want_mask = P.st.sel_mask != nullptr;
  const int mask_words = (P.max_ctx + 31) / 32;
  if (want_mask) {
    for (int i = tid; i < mask_words; i += SEL_NT) s_mask[i] = 0u;
  }
  const int seg = (((N + SEL_NW - 1) / SEL_NW) + 31) & ~31;
  const int w0 = warp * seg, w1 = min(N, w0 + seg);
  {
    int gt = 0, tie = 0;
    for (int base = w0; base < w1; base += 32) {
      const int i = base + lane;
      if (i < w1) {
        const uint32_t bits = row[i];
        gt += bits > tau;
        tie += bits == tau;
      }
    }
    gt = __reduce_add_sync(0xffffffffu, gt);
    tie = __reduce_add_sync(0xffffffffu, tie);
    if (lane == 0) { sh.w_gt[warp] = gt; sh.w_tie[warp] = tie; }
  }
  __syncthreads();
  int tie_before = 0, sel_before = 0;
  for (int w = 0; w < warp; ++w) {
    const int tw = sh.w_tie[w];
    int take = r_ties - tie_before;
    take = take < 0 ? 0 : (take > tw ? tw : take);
    sel_before += sh.w_gt[w] + take;
    tie_before += tw;
  }
  int32_t *votes = P.st.votes + (size_t)unit * P.max_ctx;
  const unsigned lt = (1u << lane) - 1u;
  for (int base = w0; base < w1; base += 32) {
    const int i = base + lane;
    const bool valid = i < w1;
    const uint32_t bits = valid ? row[i] : 0u;
    const bool g = valid && bits > tau;
    const bool t = valid && bits == tau;
    const unsigned tb = __ballot_sync(0xffffffffu, t);
    const bool s = g || (t && (tie_before + __popc(tb & lt)) < r_ties);
    const unsigned sb = __ballot_sync(0xffffffffu, s);
    if (s) {
      const int pos = lo + i;
      sel_idx[sel_before + __popc(sb & lt)] = pos;
      votes[pos] += 1;  // cumulative selection mask = votes (L86)
      if (want_mask) atomicOr(&s_mask[pos >> 5], 1u << (pos & 31));
    }
    tie_before += __popc(tb);
    sel_before += __popc(sb);
  }
  // pads and the head-wise block table (reading C9; L207-209)
  for (int j = k + tid; j < P.k_cap; j += SEL_NT) sel_idx[j] = -1;
  const int used = (k + PAGE - 1) / PAGE;
  const int32_t *sp = P.st.sel_pages + (size_t)unit * P.spu;
  for (int j = tid; j < P.spu; j += SEL_NT) sel_table[j] = j < used ? sp[j] : -1;
  if (tid == 0) P.st.sel_count[unit] = k;
  if (want_mask) {
    __syncthreads();
    uint8_t *mk = P.st.sel_mask + (size_t)unit * (P.max_ctx / 8);
    const uint8_t *sb = reinterpret_cast<const uint8_t *>(s_mask);  // little endian: byte y holds bits 8y..8y+7
    for (int y = tid; y < P.max_ctx / 8; y += SEL_NT) mk[y] = sb[y];
  }
}

}  // namespace hardkv
