// qcache_kernels.cuh -- accumulated attention recomputed from the sliding-window query cache (score_mode
// HARDKV_SCORE_ACCUM_QCACHE; "we store the query cache in a sliding window", L122-124 "vanilla attention
// averaging in H2O" as an order-preserving g, Solution 1; reading C18):
//   A(i) = sum over the n_c cached steps tau and the G heads g of softmax_i(sm_scale q_{tau,g} . k_i / T) / G,  P_hat = A / n_c.
// Unlike every other stage this IS a contraction: M = n_c G <= 256 query rows against the pool's keys (arithmetic
// intensity M flop / byte of K, ~160 for config 4 against a ridge of ~280 on B200).  The logits are never stored
// (M x N fp32 would be 40 MB per unit): pass 1 streams the pool once for the per-row softmax statistics, a small
// reduction turns them into per-row (max, 1 / (sum G n_c)), pass 2 streams the pool again, recomputes the logits and adds
// the rows' probabilities per token.  Both passes are the score kernel's page loop (a K page = the A operand of mma.sync
// m16n8k16 tiles, 8 query rows per tile) with the query block in shared memory.  mma.sync, not tcgen05: the honest
// statement is in DESIGN.md section 11 -- this row is built for parity first.
#pragma once
#include "common.cuh"
#include "fast_kernels.cuh"
#include "score_tma.cuh"   // lds128

namespace hardkv {

constexpr int QC_ROWS = 256;   // capacity of the query block: accum_window * G <= 256

__global__ void __launch_bounds__(256) qcache_push_kernel(Params P, const void *q_) {
  // one CTA per sequence: q [Hq][d] of this step -> slot qc_slot of every query head's window; then slide
  const int b = blockIdx.x;
  if (!P.st.qcache || P.accum_window <= 0) return;
  const int slot = P.st.qc_slot[b];
  const int rowv = P.d * (P.st_esize) / 16;          // 16-byte vectors per query row
  const char *src = reinterpret_cast<const char *>(q_) + (size_t)b * P.Hq * P.d * P.st_esize;
  char *dst = reinterpret_cast<char *>(P.st.qcache);
  for (int i = threadIdx.x; i < P.Hq * rowv; i += blockDim.x) {
    const int hq = i / rowv, v = i % rowv;
    stg(dst + (((size_t)(b * P.Hq + hq) * P.accum_window + slot) * P.d) * P.st_esize + v * 16,
        ldg_ca(src + ((size_t)hq * P.d) * P.st_esize + v * 16));
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    P.st.qc_slot[b] = (slot + 1) % P.accum_window;
    if (P.st.qc_count[b] < P.accum_window) P.st.qc_count[b] += 1;
  }
}

// PASS 1: per-chunk softmax statistics of every query row; PASS 2: probabilities summed over the rows -> probs.
template <int D, int PASS>
__global__ void __launch_bounds__(256) qcache_pass_kernel(Params P) {
  KernelClock kclock(P);
  constexpr int NCH = D / 32, ROWB = D * 2;
  extern __shared__ __align__(16) unsigned char qc_smem[];
  unsigned char *Qs = qc_smem;                                                  // [QC_ROWS][D] bf16, row tau * G + g
  float2 *s_ms = reinterpret_cast<float2 *>(qc_smem + (size_t)QC_ROWS * ROWB);  // PASS 1: [8 warps][QC_ROWS]; PASS 2: [QC_ROWS]
  const int unit = blockIdx.y, b = unit / P.Hkv, h = unit % P.Hkv;
  if (P.st.score_mode[h] != HARDKV_SCORE_ACCUM_QCACHE) return;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  if (hi <= lo) return;
  const int first_page = lo >> 4, last_page = (hi - 1) >> 4;
  const int pg0 = blockIdx.x * SCORE_PAGES_PER_CTA;
  if (pg0 > last_page || pg0 + SCORE_PAGES_PER_CTA <= first_page) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int gid = lane >> 2, tig = lane & 3;
  const int G = P.G, nc = P.st.qc_count[b];
  const int M = nc * G, NB = (M + 7) >> 3;
  // ---- the query block of the unit -> shared memory (rows beyond M are zero) ----
  {
    const char *qc = reinterpret_cast<const char *>(P.st.qcache);
    constexpr int VPR = ROWB / 16;
    for (int i = tid; i < NB * 8 * VPR; i += 256) {
      const int r = i / VPR, v = i % VPR;
      uint4 val = make_uint4(0, 0, 0, 0);
      if (r < M) {
        const int tau = r / G, g = r % G;
        val = ldg_ca(qc + (((size_t)(b * P.Hq + h * G + g) * P.accum_window + tau) * D) * 2 + v * 16);
      }
      *reinterpret_cast<uint4 *>(Qs + (size_t)r * ROWB + v * 16) = val;
    }
    if (PASS == 1) {
      for (int i = tid; i < 8 * QC_ROWS; i += 256) s_ms[i] = make_float2(-INFINITY, 0.f);
    } else {
      const float2 *fin = P.qc_final + (size_t)unit * QC_ROWS;
      for (int i = tid; i < QC_ROWS; i += 256) s_ms[i] = fin[i];
    }
  }
  __syncthreads();
  const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
  const char *klane = reinterpret_cast<const char *>(P.st.k_pool) + gid * ROWB + tig * 16;
  const float c2 = P.sm_scale * 1.4426950408889634f / P.st.temperature[unit];   // logit -> base-2 exponent of z / T
  float *probs = P.st.probs + (size_t)unit * P.max_ctx;
  float2 *my_ms = s_ms + (size_t)warp * QC_ROWS;
  constexpr int PPW = SCORE_PAGES_PER_CTA / 8;
  const int wp0 = pg0 + warp * PPW;
#pragma unroll 1
  for (int j = 0; j < PPW; ++j) {
    const int pg = wp0 + j;
    if (pg < first_page || pg > last_page) continue;            // warp-uniform
    const char *src = klane + (size_t)__ldg(tab + pg) * (PAGE * ROWB);
    uint4 ka[NCH], kb[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) { ka[c] = ldg_nc(src + c * 64); kb[c] = ldg_nc(src + 8 * ROWB + c * 64); }
    const int pa = pg * PAGE + gid, pb = pa + 8;
    const bool va = pa >= lo && pa < hi, vb = pb >= lo && pb < hi;
    float sum_a = 0.f, sum_b = 0.f;                               // PASS 2: probabilities of tokens pa, pb over this lane's columns
#pragma unroll 1
    for (int nb = 0; nb < NB; ++nb) {
      const unsigned char *qrow = Qs + (size_t)(nb * 8 + gid) * ROWB + tig * 16;   // B fragment: query row nb * 8 + gid
      float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        const uint4 qv = lds128(qrow + c * 64);
        mma_bf16_16816(acc, ka[c].x, kb[c].x, ka[c].y, kb[c].y, qv.x, qv.y);
        mma_bf16_16816(acc, ka[c].z, kb[c].z, ka[c].w, kb[c].w, qv.z, qv.w);
      }
      // acc[0], acc[2]: tokens pa, pb of query row (column) nb * 8 + 2 tig; acc[1], acc[3]: the same tokens of column + 1
      const int col = nb * 8 + 2 * tig;
      if (PASS == 1) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const float xa = va ? acc[e] * c2 : -INFINITY, xb = vb ? acc[2 + e] * c2 : -INFINITY;
          float m = fmaxf(xa, xb);
#pragma unroll
          for (int o = 4; o < 32; o <<= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
          float s = (m == -INFINITY) ? 0.f : fast_exp2(xa - m) + fast_exp2(xb - m);
#pragma unroll
          for (int o = 4; o < 32; o <<= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
          if (gid == 0 && m != -INFINITY) {
            float2 st = my_ms[col + e];
            const float mn = fmaxf(st.x, m);
            st.y = st.y * fast_exp2(st.x - mn) + s * fast_exp2(m - mn);
            st.x = mn;
            my_ms[col + e] = st;
          }
        }
        __syncwarp();
      } else {
        const float2 f0 = s_ms[col], f1 = s_ms[col + 1];          // (row max in base-2 units, 1 / (row sum * G * n_c))
        sum_a += fast_exp2(fmaf(acc[0], c2, -f0.x)) * f0.y + fast_exp2(fmaf(acc[1], c2, -f1.x)) * f1.y;
        sum_b += fast_exp2(fmaf(acc[2], c2, -f0.x)) * f0.y + fast_exp2(fmaf(acc[3], c2, -f1.x)) * f1.y;
      }
    }
    if (PASS == 2) {
      sum_a += __shfl_xor_sync(0xffffffffu, sum_a, 1); sum_a += __shfl_xor_sync(0xffffffffu, sum_a, 2);
      sum_b += __shfl_xor_sync(0xffffffffu, sum_b, 1); sum_b += __shfl_xor_sync(0xffffffffu, sum_b, 2);
      if (tig == 0) {
        if (va) probs[pa] = sum_a;
        if (vb) probs[pb] = sum_b;
      }
    }
  }
  if (PASS == 1) {
    __syncthreads();
    float2 *outp = P.qc_stats + ((size_t)unit * P.score_chunks + blockIdx.x) * QC_ROWS;
    for (int col = tid; col < QC_ROWS; col += 256) {
      float m = -INFINITY, s = 0.f;
      for (int w = 0; w < 8; ++w) m = fmaxf(m, s_ms[w * QC_ROWS + col].x);
      for (int w = 0; w < 8; ++w) {
        const float2 st = s_ms[w * QC_ROWS + col];
        if (st.x != -INFINITY) s += st.y * fast_exp2(st.x - m);
      }
      outp[col] = make_float2(m, s);
    }
  }
}

// per unit and query row: chunk statistics -> (max, 1 / (sum * G * n_c)); rows beyond n_c * G get weight 0
__global__ void __launch_bounds__(QC_ROWS) qcache_reduce_kernel(Params P) {
  KernelClock kclock(P);
  const int unit = blockIdx.x, b = unit / P.Hkv, h = unit % P.Hkv, col = threadIdx.x;
  if (P.st.score_mode[h] != HARDKV_SCORE_ACCUM_QCACHE) return;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  if (hi <= lo) return;
  const int nc = P.st.qc_count[b], M = nc * P.G;
  const int ch0 = (lo >> 4) / SCORE_PAGES_PER_CTA, ch1 = ((hi - 1) >> 4) / SCORE_PAGES_PER_CTA;
  const float2 *sp = P.qc_stats + (size_t)unit * P.score_chunks * QC_ROWS;
  float m = -INFINITY, s = 0.f;
  if (col < M) {
    for (int c = ch0; c <= ch1; ++c) m = fmaxf(m, sp[(size_t)c * QC_ROWS + col].x);
    for (int c = ch0; c <= ch1; ++c) {
      const float2 st = sp[(size_t)c * QC_ROWS + col];
      if (st.x != -INFINITY) s += st.y * fast_exp2(st.x - m);
    }
  }
  P.qc_final[(size_t)unit * QC_ROWS + col] = (col < M && s > 0.f) ? make_float2(m, 1.0f / (s * (float)P.G * (float)nc))
                                                                  : make_float2(0.f, 0.f);
}

}  // namespace hardkv
