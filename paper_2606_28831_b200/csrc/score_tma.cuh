// score_tma.cuh -- bf16 GQA score as a persistent, TMA-staged streaming kernel (sm_100a).
// z[g][i] = sm_scale * q_g . k_i over the pool (exponent of Eq. 4) plus the per-chunk
// softmax statistics of z / T that Logits Calibration needs (L120).
//
// One CTA per SM.  A K page is 16 rows = one contiguous 4 KiB (d = 128) block of the paged pool, so a page
// is one 1-D bulk async copy (cp.async.bulk, the TMA engine; SASS UBLKCP) into a ring of shared-memory
// stages tracked by mbarriers: producer warps keep SCORE_STAGES pages in flight per SM with no register
// or L1-miss-tracking cost, 8 consumer warps take pages round-robin, read their MMA fragments from shared
// memory (16-byte LDS in the same permuted layout as score_mma_kernel) and release the stage.
// Work items are (unit, chunk of SCORE_PAGES_PER_CTA pages); CTA i takes the active items i, i + grid, ...
// (equal-sized items, so a static round-robin is balanced); the item list is rebuilt by every CTA from
// ctx_len / c_lo with a prefix sum over the units.
#pragma once
#include "common.cuh"
#include "fast_kernels.cuh"

namespace hardkv {

#ifndef HARDKV_SCORE_STAGES
#define HARDKV_SCORE_STAGES 32
#endif
constexpr int SCORE_STAGES = HARDKV_SCORE_STAGES;   // pages in flight per SM (multiple of 8): 128 KiB at d = 128 (measured
                                                    // flat from 24 stages up); leaves room for a co-resident select CTA
constexpr int SCORE_CONSUMERS = 8;          // consumer warps
constexpr int SCORE_PRODUCERS = 4;          // producer warps (one issuing lane each): a copy costs ~150 issue cycles
constexpr int SCORE_TMA_THREADS = (SCORE_CONSUMERS + SCORE_PRODUCERS) * 32;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ uint4 lds128(const void *p) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(smem_u32(p)));
  return v;
}
__device__ __forceinline__ void consumer_bar_sync() { asm volatile("bar.sync 1, %0;" ::"n"(SCORE_CONSUMERS * 32)); }

// Dynamic shared memory: [stages][page bytes] | full[stages] | empty[stages] | unit_first[units + 1] | lo[B] | hi[B]
__host__ __device__ inline size_t score_tma_smem(int d, int units, int B) {
  return (size_t)SCORE_STAGES * PAGE * d * 2 + 2 * SCORE_STAGES * 8 + (size_t)(units + 1 + 2 * B) * 4 + 1024;
}

// PUBLISH (the score || select overlap of hardkv_decode_step, variant 4): the units are streamed longest pool first
// (the reverse of unit_order), the kernel lets its dependent launch start at once, and the CTA that retires a unit's
// last chunk publishes score_flag[unit] = *epoch -- the select kernel, co-resident on the same SMs (the register and
// shared-memory budget of this kernel is held to half an SM for that), takes the unit while the stream goes on.
template <int D, bool PUBLISH>
__global__ void __launch_bounds__(SCORE_TMA_THREADS, 2) score_tma_kernel(Params P, const void *q_) {
  if (PUBLISH) pdl_trigger();
  KernelClock kclock(P);
  constexpr int NCH = D / 32;                 // 64-byte chunks per row
  constexpr int ROWB = D * 2, PAGEB = PAGE * ROWB;
  constexpr int SPC = SCORE_PAGES_PER_CTA;
  extern __shared__ __align__(128) unsigned char score_smem[];
  const int units = P.B * P.Hkv;
  unsigned char *ring = score_smem;
  uint64_t *full = reinterpret_cast<uint64_t *>(score_smem + (size_t)SCORE_STAGES * PAGEB);
  uint64_t *empty = full + SCORE_STAGES;
  int *unit_first = reinterpret_cast<int *>(empty + SCORE_STAGES);   // [units + 1] first active item of a unit
  int *s_lo = unit_first + units + 1, *s_hi = s_lo + P.B;            // pool bounds per sequence
  __shared__ float s_st[2][SCORE_CONSUMERS][8][2];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  for (int b = tid; b < P.B; b += SCORE_TMA_THREADS) {
    int n, lo, hi;
    pool_bounds(P, b, n, lo, hi);
    s_lo[b] = lo; s_hi[b] = hi;
  }
  if (tid == 0) {
    for (int s = 0; s < SCORE_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (warp == 0) {   // exclusive prefix sum of the chunk counts of the units
    int run = 0;
    for (int u0 = 0; u0 < units; u0 += 32) {
      const int u = u0 + lane;     // rank in the streaming order
      int cnt = 0;
      if (u < units) {
        const int uu = PUBLISH ? P.unit_order[units - 1 - u] : u;
        const int lo = s_lo[uu / P.Hkv], hi = s_hi[uu / P.Hkv];
        if (hi > lo) cnt = ((hi - 1) >> 4) / SPC - (lo >> 4) / SPC + 1;
      }
      int inc = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      if (u < units) unit_first[u] = run + inc - cnt;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) unit_first[units] = run;
  }
  __syncthreads();
  const int nitems = unit_first[units];
  const char *kpool = reinterpret_cast<const char *>(P.st.k_pool);
  int nbase = 0;   // pages this CTA has streamed before the current item (same count in every warp)

  for (int it = blockIdx.x; it < nitems; it += gridDim.x) {
    // item -> (unit, chunk): largest unit with unit_first[unit] <= it
    int ul = 0, uh = units - 1;
    while (ul < uh) {
      const int mid = (ul + uh + 1) >> 1;
      if (unit_first[mid] <= it) ul = mid; else uh = mid - 1;
    }
    const int unit = PUBLISH ? P.unit_order[units - 1 - ul] : ul, b = unit / P.Hkv, h = unit % P.Hkv;
    const int lo = s_lo[b], hi = s_hi[b];
    const int first_page = lo >> 4, last_page = (hi - 1) >> 4;
    const int chunk = first_page / SPC + (it - unit_first[ul]);
    const int pa = max(first_page, chunk * SPC), pb = min(last_page, chunk * SPC + SPC - 1);
    const int np = pb - pa + 1;
    const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;

    if (warp >= SCORE_CONSUMERS) {
      // ---- producers: warp pw issues, from one lane, the copies of the pages n = pw (mod 4) of this CTA's page
      //      sequence; the physical page ids of its (<= 16) pages of the item come in with one coalesced load ----
      const int pw = warp - SCORE_CONSUMERS;
      const int j0 = (pw - nbase) & (SCORE_PRODUCERS - 1);
      const int mine = j0 < np ? (np - j0 + SCORE_PRODUCERS - 1) / SCORE_PRODUCERS : 0;
      const int pid = lane < mine ? __ldg(tab + pa + j0 + lane * SCORE_PRODUCERS) : 0;
      for (int i = 0; i < mine; ++i) {
        const int page = __shfl_sync(0xffffffffu, pid, i);
        if (lane == 0) {
          const int n = nbase + j0 + i * SCORE_PRODUCERS, s = n % SCORE_STAGES, k = n / SCORE_STAGES;
          mbar_wait(&empty[s], (k & 1) ^ 1);        // the consumer of the stage's previous page has read it
          mbar_expect_tx(&full[s], PAGEB);
          bulk_g2s(ring + (size_t)s * PAGEB, kpool + (size_t)page * PAGEB, PAGEB, &full[s]);
        }
      }
    } else {
      // ---- consumers: warp w takes the pages n = w (mod 8) ----
      const int gid = lane >> 2, tig = lane & 3;
      const int G = P.G;
      uint4 qv[NCH];                                // B fragments: q of head gid (zero above G), permuted like the key rows
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        qv[c] = make_uint4(0, 0, 0, 0);
        if (gid < G) {
          const char *qp = reinterpret_cast<const char *>(q_) + ((size_t)(b * P.Hq + h * G + gid) * D) * 2;
          qv[c] = ldg_ca(qp + c * 64 + tig * 16);
        }
      }
      float *lg = P.st.logits + ((size_t)(b * P.Hq + h * G)) * P.max_ctx;
      const int h0 = 2 * tig, h1 = 2 * tig + 1;
      const float c2 = P.sm_scale * 1.4426950408889634f / P.st.temperature[unit];  // logit -> base-2 exponent of z/T
      float m0 = -INFINITY, s0 = 0.f, m1 = -INFINITY, s1 = 0.f;
      for (int j = (warp - nbase) & 7; j < np; j += SCORE_CONSUMERS) {
        const int n = nbase + j, s = n % SCORE_STAGES, k = n / SCORE_STAGES;
        const unsigned char *src = ring + (size_t)s * PAGEB;
        mbar_wait(&full[s], k & 1);                 // the page has landed
        uint4 ka[NCH], kb[NCH];
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          ka[c] = lds128(src + gid * ROWB + c * 64 + tig * 16);
          kb[c] = lds128(src + (gid + 8) * ROWB + c * 64 + tig * 16);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);      // fragments are in registers: hand the stage back
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          mma_bf16_16816(acc, ka[c].x, kb[c].x, ka[c].y, kb[c].y, qv[c].x, qv[c].y);
          mma_bf16_16816(acc, ka[c].z, kb[c].z, ka[c].w, kb[c].w, qv[c].z, qv[c].w);
        }
        const int ta = (pa + j) * PAGE + gid, tb = ta + 8;
        const bool va = ta >= lo && ta < hi, vb = tb >= lo && tb < hi;
        if (h0 < G) {
          if (va) lg[(size_t)h0 * P.max_ctx + ta] = acc[0] * P.sm_scale;
          if (vb) lg[(size_t)h0 * P.max_ctx + tb] = acc[2] * P.sm_scale;
          const float xa = va ? acc[0] * c2 : -INFINITY, xb = vb ? acc[2] * c2 : -INFINITY;
          const float mn = fmaxf(m0, fmaxf(xa, xb));
          if (mn != -INFINITY) { s0 = s0 * fast_exp2(m0 - mn) + fast_exp2(xa - mn) + fast_exp2(xb - mn); m0 = mn; }
        }
        if (h1 < G) {
          if (va) lg[(size_t)h1 * P.max_ctx + ta] = acc[1] * P.sm_scale;
          if (vb) lg[(size_t)h1 * P.max_ctx + tb] = acc[3] * P.sm_scale;
          const float xa = va ? acc[1] * c2 : -INFINITY, xb = vb ? acc[3] * c2 : -INFINITY;
          const float mn = fmaxf(m1, fmaxf(xa, xb));
          if (mn != -INFINITY) { s1 = s1 * fast_exp2(m1 - mn) + fast_exp2(xa - mn) + fast_exp2(xb - mn); m1 = mn; }
        }
      }
      // ---- chunk statistics: over the 8 token lanes of a warp, then over the consumer warps ----
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) {
        const float om0 = __shfl_xor_sync(0xffffffffu, m0, o), os0 = __shfl_xor_sync(0xffffffffu, s0, o);
        const float om1 = __shfl_xor_sync(0xffffffffu, m1, o), os1 = __shfl_xor_sync(0xffffffffu, s1, o);
        const float n0 = fmaxf(m0, om0), n1 = fmaxf(m1, om1);
        s0 = (n0 == -INFINITY) ? 0.f : s0 * fast_exp2(m0 - n0) + os0 * fast_exp2(om0 - n0);
        s1 = (n1 == -INFINITY) ? 0.f : s1 * fast_exp2(m1 - n1) + os1 * fast_exp2(om1 - n1);
        m0 = n0; m1 = n1;
      }
      const int par = ((it - blockIdx.x) / gridDim.x) & 1;   // double-buffered: one barrier per item
      if (gid == 0) {
        s_st[par][warp][h0][0] = m0; s_st[par][warp][h0][1] = s0;
        s_st[par][warp][h1][0] = m1; s_st[par][warp][h1][1] = s1;
      }
      consumer_bar_sync();
      if (tid < 8) {
        const int g = tid;
        float m = -INFINITY, sacc = 0.f;
        if (g < G) {
#pragma unroll
          for (int w = 0; w < SCORE_CONSUMERS; ++w) m = fmaxf(m, s_st[par][w][g][0]);
#pragma unroll
          for (int w = 0; w < SCORE_CONSUMERS; ++w) {
            const float mw = s_st[par][w][g][0];
            if (mw != -INFINITY) sacc += s_st[par][w][g][1] * fast_exp2(mw - m);
          }
        }
        P.score_stats[((size_t)unit * P.score_chunks + chunk) * 8 + g] = make_float2(m, sacc);
      }
      if (PUBLISH) {
        // every logit of the item was stored before the consumer barrier above; the statistics by the 8 threads of
        // warp 0, which lane 0 orders behind itself with the warp barrier; the fence is cumulative; then the ticket
        if (warp == 0) {
          __syncwarp();
          if (lane == 0) {
            __threadfence();
            const int nch = last_page / SPC - first_page / SPC + 1;
            if (atomicAdd(P.ss_arrive + unit, 1) == nch - 1) {
              P.ss_arrive[unit] = 0;                 // re-arm for the next launch / graph replay
              __threadfence();
              *reinterpret_cast<volatile int32_t *>(P.score_flag + unit) = *reinterpret_cast<volatile int32_t *>(P.epoch);
            }
          }
        }
      }
    }
    nbase += np;
  }
}

}  // namespace hardkv
