// attend_mma.cuh -- bf16 split-K decode attention over the three tiers on warp-level tensor-core
// MMAs (mma.sync m16n8k16, fp32 accumulate), optionally fused with the Rewrite Cache write-through.
// PAPER.md L84 (exact attention from the partial outputs of the tiers), Appendix F Eq. 4-6
// (L735-762), L172 (Rewrite Cache).  The GQA group is the tiny dimension (G <= 8): a memory-bound
// batch of GEMVs, so the MMAs only take the convert/FMA/shuffle work off the issue slots.
//
// One warp owns a tile of 16 virtual rows (tokens) at a time.
//   S^T = Q K^T :  A = Q (16 x d, rows >= G zero), B = K^T (d x 8 tokens), two token blocks per tile.
//     The contraction index may be permuted as long as A and B agree, so lane (gid, tig) loads 16
//     contiguous bytes of key row `gid` (4 lanes cover 64 contiguous bytes) and feeds two MMAs with no
//     shuffle.  Accumulator c0/c1 of lane (gid, tig) = head gid, tokens 2 tig / 2 tig + 1 of the block:
//     exactly the B fragment of the next MMA (the register-reuse of flash attention, transposed).
//   O^T = V^T P^T : A = V^T (16 d x 16 tokens), B = P^T (16 tokens x 8 heads).  Lane (gid, tig) loads 16
//     bytes (8 consecutive d) of the value rows of tokens 2 tig, 2 tig + 1, 2 tig + 8, 2 tig + 9; a pair
//     {V[t][d], V[t+1][d]} is one PRMT of two loaded registers; the d rows of an MMA are permuted
//     (row gid <-> d = 64 c + 8 gid + 2 j, row gid + 8 <-> d + 1) which only relabels the outputs.
//   P is fed as bf16 hi + lo (two MMAs) so the weights keep ~16 mantissa bits.
#pragma once
#include <cuda_bf16.h>

#include "common.cuh"
#include "fast_kernels.cuh"

namespace hardkv {

#ifndef HARDKV_ATT_TPW
#define HARDKV_ATT_TPW 4
#endif
constexpr int ATT_TPW = HARDKV_ATT_TPW;       // tiles of 16 rows per warp
constexpr int ATT_MMA_CHUNK = 8 * ATT_TPW * 16;   // virtual rows per CTA: 8 warps x ATT_TPW tiles
constexpr uint32_t ROW_INVALID = 0xffffffffu;

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&v);
}
__device__ __forceinline__ float bf16_round(float x) { return __bfloat162float(__float2bfloat16_rn(x)); }

template <int D, int MODE>
__global__ void __launch_bounds__(256, 2) attend_mma_kernel(Params P, const void *q_, float *out, float *lse) {
  // wait_select: launched programmatically behind the select kernel; units come in the order their selections finish and
  // every CTA waits for its own unit only (the stream predecessors of the select kernel are complete: it was launched
  // with a full dependency on them)
  if (P.wait_select) pdl_trigger(); else pdl_wait_then_trigger();
  KernelClock kclock(P);
  constexpr int NKC = D / 32;   // 64-byte chunks of a key row
  constexpr int NVC = D / 64;   // 128-byte chunks of a value row
  constexpr int ROWB = D * 2;
  const int unit = P.wait_select == 1 ? P.unit_order[blockIdx.y]
                   : (P.wait_select == 2 ? P.unit_order[gridDim.y - 1 - blockIdx.y] : (int)blockIdx.y), b = unit / P.Hkv, h = unit % P.Hkv;
  // forked append (common.cuh): nobody reads the in-place scalars during this launch -- one CTA writes them back
  if (P.use_shadow && blockIdx.x == 0 && blockIdx.y == 0) {
    for (int t = threadIdx.x; t < P.B; t += 256) {
      P.st.ctx_len[t] = P.sh_scal[t];
      P.st.c_lo[t] = P.sh_scal[P.B + t];
      P.st.dense_lo[t] = P.sh_scal[2 * P.B + t];
    }
  }
  if (P.wait_select) wait_unit_selected(P, unit);
  // Virtual row space of a unit: [selected | dense | condensed].  With the selected rows first, row v of the space is
  // selected row v whatever the counts are: the two loads that start its resolution (sel_idx[v], sel_pages[v / 16]) are
  // issued here, together with the loads of the counts, instead of behind them -- one dependent round trip less at the
  // head of every CTA -- and a tile of 16 selected rows is exactly one page of the selected tier (write-through).
  constexpr int RPL = ATT_TPW / 2;
  const int32_t *stab = P.st.sel_pages + (size_t)unit * P.spu;
  const int32_t *idx = P.st.sel_idx + (size_t)unit * P.k_cap;
  int spec_pos[RPL], spec_page[RPL];
#pragma unroll
  for (int r = 0; r < RPL; ++r) {
    const int v = (int)blockIdx.x * ATT_MMA_CHUNK + (int)(threadIdx.x >> 5) * (ATT_TPW * 16) + r * 32 + (int)(threadIdx.x & 31);
    spec_pos[r] = (MODE != ATT_TIER && v < P.k_cap) ? __ldg(idx + v) : -1;
    spec_page[r] = (MODE != ATT_SPARSE && v < P.k_cap) ? __ldg(stab + (v >> 4)) : -1;
  }
  const int n = P.use_shadow ? P.sh_scal[b] : P.st.ctx_len[b];
  int s_end, r_lo;
  if (!dense_bounds(P, b, n, s_end, r_lo)) {   // more reuse steps than cfg.reuse_max: flag, leave the unit untouched
    if (threadIdx.x == 0 && blockIdx.x == 0) atomicExch(P.st.err_flag, 2);
    return;
  }
  const int n_dense = s_end + (n - r_lo);
  const int k = P.st.sel_count[unit];
  const int cc = P.st.cond_count[unit];
  const int total = n_dense + k + cc;
  const int nchunks = (total + ATT_MMA_CHUNK - 1) / ATT_MMA_CHUNK;
  const int c = blockIdx.x;
  if (c >= nchunks) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int gid = lane >> 2, tig = lane & 3;
  const int G = P.G;

  const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
  const char *kp0 = reinterpret_cast<const char *>(P.st.k_pool), *vp0 = reinterpret_cast<const char *>(P.st.v_pool);
  char *kp1 = reinterpret_cast<char *>(P.st.sel_k_pool), *vp1 = reinterpret_cast<char *>(P.st.sel_v_pool);
  const char *kp2 = reinterpret_cast<const char *>(P.st.cond_k), *vp2 = reinterpret_cast<const char *>(P.st.cond_v);

  // A fragments of S^T = Q K^T: q of head gid (zero above G), permuted like the key rows
  uint4 qv[NKC];
#pragma unroll
  for (int ch = 0; ch < NKC; ++ch) {
    qv[ch] = make_uint4(0, 0, 0, 0);
    if (gid < G) {
      const char *qp = reinterpret_cast<const char *>(q_) + ((size_t)(b * P.Hq + h * G + gid) * D) * 2;
      qv[ch] = ldg_ca(qp + ch * 64 + tig * 16);
    }
  }
  const float c2 = P.sm_scale * 1.4426950408889634f;   // logit -> base-2 exponent
  float m_run = -INFINITY, l_run = 0.f;                // head gid (identical in the 4 lanes of a gid)
  float acc[NVC * 4][4];                               // O^T tiles: [64 c + 8 gid + 2 j (+1)][heads 2 tig, 2 tig + 1]
#pragma unroll
  for (int i = 0; i < NVC * 4; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;

  const int v0 = c * ATT_MMA_CHUNK, v1 = min(total, v0 + ATT_MMA_CHUNK);
  // ---- the rows of all tiles of the warp are resolved up front: lane l holds rows l and l + 32 of the warp's
  //      ATT_TPW * 16 rows as source (tier << 30 | row) and rewrite destination ----
  uint32_t srcs[RPL], dsts[RPL];
#pragma unroll
  for (int r = 0; r < RPL; ++r) {
    srcs[r] = ROW_INVALID; dsts[r] = ROW_INVALID;
    const int v = v0 + warp * (ATT_TPW * 16) + r * 32 + lane;
    if (v < k) {                            // Tier 2: selected rows (v = index into sel_idx)
      const uint32_t srow = (uint32_t)(spec_page[r] * PAGE + (v & 15));
      if (MODE != ATT_TIER) {
        const int pos = spec_pos[r];
        srcs[r] = (uint32_t)(__ldg(tab + (pos >> 4)) * PAGE + (pos & 15));
        if (MODE == ATT_REWRITE) dsts[r] = srow;
      } else {
        srcs[r] = (1u << 30) | srow;
      }
    } else if (v < k + n_dense) {           // Tier 1: sinks + recent window, read in place
      const int dv = v - k;
      const int pos = dv < s_end ? dv : r_lo + (dv - s_end);
      srcs[r] = (uint32_t)(__ldg(tab + (pos >> 4)) * PAGE + (pos & 15));
    } else if (v < total) {                 // Tier 3: condensed residents
      srcs[r] = (2u << 30) | (uint32_t)(unit * P.cond_cap + (v - k - n_dense));
    }
  }
#pragma unroll
  for (int it = 0; it < ATT_TPW; ++it) {
    const int vbase = v0 + warp * (ATT_TPW * 16) + it * 16;
    if (vbase >= v1) break;
    const int lb = (it & 1) * 16;
    const uint32_t src = srcs[it >> 1], dst = dsts[it >> 1];
    uint32_t ks[2], vs[4], kd[2], vd[4];
    ks[0] = __shfl_sync(0xffffffffu, src, lb + gid);
    ks[1] = __shfl_sync(0xffffffffu, src, lb + gid + 8);
    vs[0] = __shfl_sync(0xffffffffu, src, lb + 2 * tig);
    vs[1] = __shfl_sync(0xffffffffu, src, lb + 2 * tig + 1);
    vs[2] = __shfl_sync(0xffffffffu, src, lb + 2 * tig + 8);
    vs[3] = __shfl_sync(0xffffffffu, src, lb + 2 * tig + 9);
    if (MODE == ATT_REWRITE) {
      kd[0] = __shfl_sync(0xffffffffu, dst, lb + gid);
      kd[1] = __shfl_sync(0xffffffffu, dst, lb + gid + 8);
      vd[0] = __shfl_sync(0xffffffffu, dst, lb + 2 * tig);
      vd[1] = __shfl_sync(0xffffffffu, dst, lb + 2 * tig + 1);
      vd[2] = __shfl_sync(0xffffffffu, dst, lb + 2 * tig + 8);
      vd[3] = __shfl_sync(0xffffffffu, dst, lb + 2 * tig + 9);
    }
    // ---- loads: 16 x 16 B per lane = the 16 key rows and 16 value rows of the tile ----
    uint4 kr[2][NKC], vr[4][NVC];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const uint32_t w = ks[r];
      const uint32_t tier = w >> 30;
      const char *basep = tier == 0 ? kp0 : (tier == 1 ? kp1 : kp2);
      const char *rp = basep + (size_t)(w & 0x3fffffffu) * ROWB + tig * 16;
#pragma unroll
      for (int ch = 0; ch < NKC; ++ch) kr[r][ch] = w != ROW_INVALID ? ldg_nc(rp + ch * 64) : make_uint4(0, 0, 0, 0);
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const uint32_t w = vs[r];
      const uint32_t tier = w >> 30;
      const char *basep = tier == 0 ? vp0 : (tier == 1 ? vp1 : vp2);
      const char *rp = basep + (size_t)(w & 0x3fffffffu) * ROWB + gid * 16;
#pragma unroll
      for (int ch = 0; ch < NVC; ++ch) vr[r][ch] = w != ROW_INVALID ? ldg_nc(rp + ch * 128) : make_uint4(0, 0, 0, 0);
    }
    // ---- Rewrite Cache write-through (L172): the rows go to the selected tier as they arrive ----
    if (MODE == ATT_REWRITE) {
#pragma unroll
      for (int r = 0; r < 2; ++r)
        if (kd[r] != ROW_INVALID) {
          char *wp = kp1 + (size_t)kd[r] * ROWB + tig * 16;
#pragma unroll
          for (int ch = 0; ch < NKC; ++ch) stg_cs(wp + ch * 64, kr[r][ch]);
        }
#pragma unroll
      for (int r = 0; r < 4; ++r)
        if (vd[r] != ROW_INVALID) {
          char *wp = vp1 + (size_t)vd[r] * ROWB + gid * 16;
#pragma unroll
          for (int ch = 0; ch < NVC; ++ch) stg_cs(wp + ch * 128, vr[r][ch]);
        }
    }
    // ---- S^T = Q K^T for the two 8-token blocks ----
    float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int ch = 0; ch < NKC; ++ch) {
      mma_bf16_16816(s0, qv[ch].x, 0u, qv[ch].y, 0u, kr[0][ch].x, kr[0][ch].y);
      mma_bf16_16816(s0, qv[ch].z, 0u, qv[ch].w, 0u, kr[0][ch].z, kr[0][ch].w);
      mma_bf16_16816(s1, qv[ch].x, 0u, qv[ch].y, 0u, kr[1][ch].x, kr[1][ch].y);
      mma_bf16_16816(s1, qv[ch].z, 0u, qv[ch].w, 0u, kr[1][ch].z, kr[1][ch].w);
    }
    // ---- online softmax of head gid over tokens 2 tig, 2 tig + 1, 2 tig + 8, 2 tig + 9 (Eq. 4, max-shifted) ----
    const int t0 = vbase + 2 * tig;
    float x[4];
    x[0] = t0 < v1 ? s0[0] * c2 : -INFINITY;
    x[1] = t0 + 1 < v1 ? s0[1] * c2 : -INFINITY;
    x[2] = t0 + 8 < v1 ? s1[0] * c2 : -INFINITY;
    x[3] = t0 + 9 < v1 ? s1[1] * c2 : -INFINITY;
    float tmax = fmaxf(fmaxf(x[0], x[1]), fmaxf(x[2], x[3]));
    tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
    tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
    const float m_new = fmaxf(m_run, tmax);             // finite: a tile holds at least one valid row
    if (__any_sync(0xffffffffu, m_new > m_run)) {
      const float alpha = fast_exp2(m_run - m_new);     // 2^-inf = 0 on the first tile
      const float a0 = __shfl_sync(0xffffffffu, alpha, (2 * tig) * 4);
      const float a1 = __shfl_sync(0xffffffffu, alpha, (2 * tig + 1) * 4);
#pragma unroll
      for (int i = 0; i < NVC * 4; ++i) { acc[i][0] *= a0; acc[i][1] *= a1; acc[i][2] *= a0; acc[i][3] *= a1; }
      l_run *= alpha;
      m_run = m_new;
    }
    float ph[4], pl[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float pr = fast_exp2(x[i] - m_run);
      ph[i] = bf16_round(pr);
      pl[i] = pr - ph[i];
      l_run += pr;
    }
    const uint32_t bh0 = pack_bf16(ph[0], ph[1]), bh1 = pack_bf16(ph[2], ph[3]);
    const uint32_t bl0 = pack_bf16(pl[0], pl[1]), bl1 = pack_bf16(pl[2], pl[3]);
    // ---- O^T += V^T P^T ----
#pragma unroll
    for (int ch = 0; ch < NVC; ++ch) {
      const uint32_t r0[4] = {vr[0][ch].x, vr[0][ch].y, vr[0][ch].z, vr[0][ch].w};
      const uint32_t r1[4] = {vr[1][ch].x, vr[1][ch].y, vr[1][ch].z, vr[1][ch].w};
      const uint32_t r2[4] = {vr[2][ch].x, vr[2][ch].y, vr[2][ch].z, vr[2][ch].w};
      const uint32_t r3[4] = {vr[3][ch].x, vr[3][ch].y, vr[3][ch].z, vr[3][ch].w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t a0 = __byte_perm(r0[j], r1[j], 0x5410);   // {V[t0][d], V[t1][d]}      d = 64 ch + 8 gid + 2 j
        const uint32_t a1 = __byte_perm(r0[j], r1[j], 0x7632);   // {V[t0][d+1], V[t1][d+1]}
        const uint32_t a2 = __byte_perm(r2[j], r3[j], 0x5410);
        const uint32_t a3 = __byte_perm(r2[j], r3[j], 0x7632);
        mma_bf16_16816(acc[ch * 4 + j], a0, a1, a2, a3, bh0, bh1);
        mma_bf16_16816(acc[ch * 4 + j], a0, a1, a2, a3, bl0, bl1);
      }
    }
  }

  if (MODE == ATT_REWRITE && k > 0 && (k - 1) >= v0 && (k - 1) < v1) {
    // zero tail of the last valid page of the selected tier (DESIGN reading C9)
    constexpr int LPR = ROWB / 16;
    const int kend = (k + PAGE - 1) & ~(PAGE - 1);
    for (int vec = tid; vec < (kend - k) * LPR; vec += 256) {
      const int j = k + vec / LPR, cch = vec % LPR;
      const size_t so = ((size_t)__ldg(stab + (j >> 4)) * PAGE + (j & 15)) * ROWB + cch * 16;
      stg(kp1 + so, make_uint4(0, 0, 0, 0));
      stg(vp1 + so, make_uint4(0, 0, 0, 0));
    }
  }

  // ---- per-warp state -> shared memory (m in base-2 units) ----
  l_run += __shfl_xor_sync(0xffffffffu, l_run, 1);
  l_run += __shfl_xor_sync(0xffffffffu, l_run, 2);
  __shared__ float s_st[8][8][D + 2];
  __shared__ int s_last;
  if (tig == 0) { s_st[warp][gid][0] = m_run; s_st[warp][gid][1] = l_run; }
#pragma unroll
  for (int i = 0; i < NVC * 4; ++i) {
    const int dd = 64 * (i >> 2) + 8 * gid + 2 * (i & 3);
    s_st[warp][2 * tig][2 + dd] = acc[i][0];
    s_st[warp][2 * tig + 1][2 + dd] = acc[i][1];
    s_st[warp][2 * tig][2 + dd + 1] = acc[i][2];
    s_st[warp][2 * tig + 1][2 + dd + 1] = acc[i][3];
  }
  __syncthreads();
  // ---- combine the 8 warps (Eq. 6 in max-shifted form) into this chunk's partial ----
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
      const float cw = (mw == -INFINITY) ? 0.f : fast_exp2(mw - M);
      L += s_st[w][g][1] * cw;
      A += s_st[w][g][2 + e] * cw;
    }
    part[g * (D + 2) + 2 + e] = A;
    if (e == 0) { part[g * (D + 2)] = M; part[g * (D + 2) + 1] = L; }
  }
  // ---- the last CTA of the unit to arrive merges all chunk partials (Eq. 6): its 8 warps take
  //      chunks w, w + 8, ... in parallel (lanes over d), then combine through shared memory ----
  // every thread's partial stores are ordered before thread 0 by the barrier and thread 0's fence is cumulative: one
  // fence per CTA instead of 256, each of which would wait for its thread's own streaming stores to drain
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const int ticket = atomicAdd(P.att_arrive + unit, 1);
    s_last = (ticket == nchunks - 1);
    if (s_last) __threadfence();
  }
  __syncthreads();
  if (!s_last) return;
  {
    float mm[8], ll[8], aa[8][D / 32];
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      mm[g] = -INFINITY; ll[g] = 0.f;
#pragma unroll
      for (int i = 0; i < D / 32; ++i) aa[g][i] = 0.f;
    }
    const float *pu = P.part + (size_t)unit * P.att_chunks * G * (D + 2);
    for (int ch = warp; ch < nchunks; ch += 8) {
      const float *pc = pu + (size_t)ch * G * (D + 2);
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        if (g < G) {
          const float *pp = pc + g * (D + 2);
          const float mw = __ldcg(pp), lw = __ldcg(pp + 1);
          float v[D / 32];
#pragma unroll
          for (int i = 0; i < D / 32; ++i) v[i] = __ldcg(pp + 2 + lane + 32 * i);
          const float mn = fmaxf(mm[g], mw);
          const float ca = (mm[g] == -INFINITY) ? 0.f : fast_exp2(mm[g] - mn);
          const float cb = (mw == -INFINITY) ? 0.f : fast_exp2(mw - mn);
          ll[g] = ll[g] * ca + lw * cb;
#pragma unroll
          for (int i = 0; i < D / 32; ++i) aa[g][i] = aa[g][i] * ca + v[i] * cb;
          mm[g] = mn;
        }
      }
    }
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      if (g < G) {
        if (lane == 0) { s_st[warp][g][0] = mm[g]; s_st[warp][g][1] = ll[g]; }
#pragma unroll
        for (int i = 0; i < D / 32; ++i) s_st[warp][g][2 + lane + 32 * i] = aa[g][i];
      }
    }
  }
  __syncthreads();
  for (int it = tid; it < G * D; it += 256) {
    const int g = it / D, e = it % D;
    float M = -INFINITY;
#pragma unroll
    for (int w = 0; w < 8; ++w) M = fmaxf(M, s_st[w][g][0]);
    float L = 0.f, A = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
      const float mw = s_st[w][g][0];
      const float cw = (mw == -INFINITY) ? 0.f : fast_exp2(mw - M);
      L += s_st[w][g][1] * cw;
      A += s_st[w][g][2 + e] * cw;
    }
    out[((size_t)(b * P.Hq + h * G + g)) * D + e] = A / L;
    if (e == 0 && lse) lse[b * P.Hq + h * G + g] = (M + log2f(L)) * 0.6931471805599453f;
  }
  if (tid == 0) P.att_arrive[unit] = 0;  // restore for the next launch / graph replay
}

}  // namespace hardkv
