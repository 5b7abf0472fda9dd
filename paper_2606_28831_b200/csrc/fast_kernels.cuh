// fast_kernels.cuh -- bf16 paths of the two streaming stages on warp-level tensor-core MMAs
// (mma.sync m16n8k16, fp32 accumulate).  The GQA group is the tiny dimension (G <= 8 query heads
// against thousands of keys): a memory-bound GEMV batch, so tcgen05/TMEM would buy nothing; the MMA
// is used only to take the convert + FMA + shuffle-reduce work off the issue slots so that the
// kernels run at the speed of their 16-byte coalesced loads.  Citations are PAPER.md lines.
#pragma once
#include "common.cuh"

namespace hardkv {

__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// =============================================================================================
// score (bf16): z[g][i] = sm_scale * q_g . k_i over the pool (exponent of Eq. 4), plus
// the per-chunk softmax statistics of z/T that Logits Calibration needs (L120).
//
// One warp = one 16-token page per iteration = one M=16 tile: A = the page (16 x d, row major),
// B = q^T (d x 8 query heads, zero-padded above G).  The contraction index may be permuted
// freely as long as A and B use the same permutation, so every lane loads 16 contiguous bytes of
// a key row (4 lanes cover 64 contiguous bytes; a warp load instruction covers 8 rows x 64 B in
// whole 32-byte sectors) and feeds them to two MMAs without any shuffle:
//   lane (gid = lane / 4, tig = lane % 4), 64-byte chunk c of the row, half s in {0, 1}:
//   k-slots (2 tig, 2 tig + 1, 2 tig + 8, 2 tig + 9) of MMA 2c + s  <-  elements 32c + 8 tig + 4s + (0, 1, 2, 3).
// Accumulator fragment: c0/c1 = token gid, heads 2 tig / 2 tig + 1; c2/c3 = token gid + 8.
// =============================================================================================
// PIF: pages a warp keeps in flight (all of their loads are issued before the first MMA); MINB: CTAs per SM the
// register allocation is held to.
template <int D, int PIF = 2, int MINB = 2>
__global__ void __launch_bounds__(256, MINB) score_mma_kernel(Params P, const void *q_) {
  pdl_wait_then_trigger();
  KernelClock kclock(P);
  constexpr int NCH = D / 32;                 // 64-byte chunks per row
  constexpr int ROWB = D * 2;
  const int unit = blockIdx.y, b = unit / P.Hkv, h = unit % P.Hkv;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  if (hi <= lo) return;
  const int first_page = lo >> 4, last_page = (hi - 1) >> 4;
  const int pg0 = blockIdx.x * SCORE_PAGES_PER_CTA;
  if (pg0 > last_page || pg0 + SCORE_PAGES_PER_CTA <= first_page) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int gid = lane >> 2, tig = lane & 3;
  const int G = P.G;

  // B fragments: q of head gid (zero above G), permuted like the key rows
  uint4 qv[NCH];
#pragma unroll
  for (int c = 0; c < NCH; ++c) {
    qv[c] = make_uint4(0, 0, 0, 0);
    if (gid < G) {
      const char *qp = reinterpret_cast<const char *>(q_) + ((size_t)(b * P.Hq + h * G + gid) * D) * 2;
      qv[c] = ldg_ca(qp + c * 64 + tig * 16);
    }
  }
  const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
  const char *klane = reinterpret_cast<const char *>(P.st.k_pool) + gid * ROWB + tig * 16;   // this lane's bytes of row gid of page 0
  float *lg = P.st.logits + ((size_t)(b * P.Hq + h * G)) * P.max_ctx;
  const int h0 = 2 * tig, h1 = 2 * tig + 1;
  const float c2 = P.sm_scale * 1.4426950408889634f / P.st.temperature[unit];  // logit -> base-2 exponent of z/T
  float m0 = -INFINITY, s0 = 0.f, m1 = -INFINITY, s1 = 0.f;  // running (max, sum 2^(x - max)) of heads h0, h1

  // a warp owns SCORE_PAGES_PER_CTA / 8 consecutive logical pages; their physical ids come in with one load
  constexpr int PPW = SCORE_PAGES_PER_CTA / 8;
  const int wp0 = pg0 + warp * PPW;
  int my_page = -1;
  if (lane < PPW && wp0 + lane >= first_page && wp0 + lane <= last_page) my_page = __ldg(tab + wp0 + lane);
#pragma unroll 1
  for (int j0 = 0; j0 < PPW; j0 += PIF) {
    // PIF pages (4 KiB each) in flight per warp: all their loads are issued before the first MMA
    int phys[PIF];
    uint4 ka[PIF][NCH], kb[PIF][NCH];
#pragma unroll
    for (int u = 0; u < PIF; ++u) {
      phys[u] = __shfl_sync(0xffffffffu, my_page, j0 + u);
      if (phys[u] >= 0) {   // warp-uniform; one base per page, every load at an immediate offset from it
        const char *src = klane + (size_t)phys[u] * (PAGE * ROWB);
        ka[u][0] = ldg_nc_off<0>(src);             kb[u][0] = ldg_nc_off<8 * ROWB>(src);
        ka[u][1] = ldg_nc_off<64>(src);            kb[u][1] = ldg_nc_off<8 * ROWB + 64>(src);
        if (NCH > 2) {
          ka[u][NCH - 2] = ldg_nc_off<128>(src);   kb[u][NCH - 2] = ldg_nc_off<8 * ROWB + 128>(src);
          ka[u][NCH - 1] = ldg_nc_off<192>(src);   kb[u][NCH - 1] = ldg_nc_off<8 * ROWB + 192>(src);
        }
      } else {
#pragma unroll
        for (int c = 0; c < NCH; ++c) ka[u][c] = kb[u][c] = make_uint4(0, 0, 0, 0);
      }
    }
#pragma unroll
    for (int u = 0; u < PIF; ++u) {
      if (phys[u] < 0) continue;   // warp-uniform
      const int pg = wp0 + j0 + u;
      float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        mma_bf16_16816(acc, ka[u][c].x, kb[u][c].x, ka[u][c].y, kb[u][c].y, qv[c].x, qv[c].y);
        mma_bf16_16816(acc, ka[u][c].z, kb[u][c].z, ka[u][c].w, kb[u][c].w, qv[c].z, qv[c].w);
      }
      const int pa = pg * PAGE + gid, pb = pa + 8;
      const bool va = pa >= lo && pa < hi, vb = pb >= lo && pb < hi;
      if (h0 < G) {
        if (va) lg[(size_t)h0 * P.max_ctx + pa] = acc[0] * P.sm_scale;
        if (vb) lg[(size_t)h0 * P.max_ctx + pb] = acc[2] * P.sm_scale;
        const float xa = va ? acc[0] * c2 : -INFINITY, xb = vb ? acc[2] * c2 : -INFINITY;
        const float mn = fmaxf(m0, fmaxf(xa, xb));
        if (mn != -INFINITY) { s0 = s0 * fast_exp2(m0 - mn) + fast_exp2(xa - mn) + fast_exp2(xb - mn); m0 = mn; }
      }
      if (h1 < G) {
        if (va) lg[(size_t)h1 * P.max_ctx + pa] = acc[1] * P.sm_scale;
        if (vb) lg[(size_t)h1 * P.max_ctx + pb] = acc[3] * P.sm_scale;
        const float xa = va ? acc[1] * c2 : -INFINITY, xb = vb ? acc[3] * c2 : -INFINITY;
        const float mn = fmaxf(m1, fmaxf(xa, xb));
        if (mn != -INFINITY) { s1 = s1 * fast_exp2(m1 - mn) + fast_exp2(xa - mn) + fast_exp2(xb - mn); m1 = mn; }
      }
    }
  }

  // ---- chunk statistics: reduce over the 8 token lanes of a warp, then over the 8 warps ----------
  __shared__ float s_st[8][8][2];
#pragma unroll
  for (int o = 4; o < 32; o <<= 1) {
    const float om0 = __shfl_xor_sync(0xffffffffu, m0, o), os0 = __shfl_xor_sync(0xffffffffu, s0, o);
    const float om1 = __shfl_xor_sync(0xffffffffu, m1, o), os1 = __shfl_xor_sync(0xffffffffu, s1, o);
    const float n0 = fmaxf(m0, om0), n1 = fmaxf(m1, om1);
    s0 = (n0 == -INFINITY) ? 0.f : s0 * fast_exp2(m0 - n0) + os0 * fast_exp2(om0 - n0);
    s1 = (n1 == -INFINITY) ? 0.f : s1 * fast_exp2(m1 - n1) + os1 * fast_exp2(om1 - n1);
    m0 = n0; m1 = n1;
  }
  if (gid == 0) {
    s_st[warp][h0][0] = m0; s_st[warp][h0][1] = s0;
    s_st[warp][h1][0] = m1; s_st[warp][h1][1] = s1;
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    const int g = threadIdx.x;
    float m = -INFINITY, s = 0.f;
    if (g < G) {
#pragma unroll
      for (int w = 0; w < 8; ++w) m = fmaxf(m, s_st[w][g][0]);
#pragma unroll
      for (int w = 0; w < 8; ++w) {
        const float mw = s_st[w][g][0];
        if (mw != -INFINITY) s += s_st[w][g][1] * fast_exp2(mw - m);
      }
    }
    P.score_stats[((size_t)unit * P.score_chunks + blockIdx.x) * 8 + g] = make_float2(m, s);
  }
}

}  // namespace hardkv
