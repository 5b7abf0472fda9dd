// qcache_umma.cuh -- the query-cache metric (reading C18; see qcache_kernels.cuh for the arithmetic) on the 5th-generation
// tensor cores: tcgen05.mma with both operands in shared memory and the accumulator in tensor memory (TMEM).
//
// This is the one stage of the path that is a contraction: per unit, the block of the last n_c G <= 256 cached query rows
// against every key of the pool.  A tile is 128 pool tokens (8 pages of the paged bf16 K pool) against the whole query
// block, contraction over d:
//   pass 1 (row statistics)  D[query row][token] = Q K^T : A = query block (M = 128 rows per instruction), B = K tile (N = 128)
//   pass 2 (probabilities)   D[token][query row] = K Q^T : A = K tile (M = 128), B = query block (N = 128 or 256)
// so that in the epilogue a thread (= one TMEM lane) owns a query row in pass 1 (online-softmax statistics in registers,
// no cross-lane work) and a token in pass 2 (the sum over the rows is a loop in one thread, the store is coalesced).
//
// Shared-memory operand layout: K-major, 128-byte swizzle (the canonical layout of the UMMA descriptor: rows of 64
// elements = 128 B, 8-row groups 1024 B apart, the 16-byte chunk index XORed with the row index modulo 8).  A K page in
// HBM is 16 rows of d elements, row-major: neither a bulk copy nor a tiled TMA box of a RANDOM page list produces that
// layout without a tensor map per pool, so four producer warps gather the pages with 16-byte cp.async copies straight to
// their swizzled places (each warp instruction covers two whole rows: coalesced), three tiles in flight; completion
// reaches the MMA warp through an mbarrier after a proxy fence (the copies are generic-proxy writes, the tensor core
// reads through the async proxy).
//
// Warp roles (13 warps): 0-3 and 4-7 = two epilogue warpgroups, one per accumulator stage in TMEM (even / odd tiles);
// 8 = TMEM allocation and the single MMA-issuing thread; 9-12 = producers.  Pipelines: full / empty mbarriers over
// the K-tile stages (producers <-> MMA, released by tcgen05.commit), tfull / tempty over the two accumulator stages
// (MMA <-> epilogue).
#pragma once
#include "common.cuh"
#include "qcache_kernels.cuh"
#include "score_tma.cuh"   // mbarrier helpers, smem_u32

namespace hardkv {

constexpr int QU_TILE = 128;            // pool tokens per tile (8 pages)
constexpr int QU_STAGES = 4;            // K tiles in shared memory
constexpr int QU_LAG = 2;               // a producer signals tile t - QU_LAG after issuing tile t: 3 tiles in flight
constexpr int QU_CPC = 2;               // score chunks (of 64 pages) per CTA
constexpr int QU_EPI_THREADS = 256, QU_MMA_WARP = 8, QU_PROD_THREADS = 128;
constexpr int QU_THREADS = QU_EPI_THREADS + 32 + QU_PROD_THREADS;

__host__ __device__ inline size_t qcache_umma_smem(int d) {
  return (size_t)QU_STAGES * QU_TILE * d * 2 + (size_t)QC_ROWS * d * 2 + 2 * QC_ROWS * sizeof(float2) + 256 + 1024;
}

// UMMA shared-memory descriptor: K-major, SWIZZLE_128B, 8-row groups 1024 B apart (version 1 = sm_100)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor of kind::f16: bf16 x bf16 -> fp32, both operands K-major, M = 128
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n"
               ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {   // arrives on bar when every MMA issued so far has completed
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void proxy_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 32 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,"
               "%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
                 "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
                 "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
               : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// byte offset of 16-byte chunk g of row r inside an operand block of `rows` rows (K halves of 64 elements back to back)
__device__ __forceinline__ uint32_t umma_sw128_off(int r, int g, int rows) {
  return (uint32_t)((g >> 3) * (rows * 128) + (r >> 3) * 1024 + (r & 7) * 128 + (((g & 7) ^ (r & 7)) << 4));
}

// PASS 1: per-(CTA, query row) softmax statistics -> qc_stats; PASS 2: probabilities summed over the query rows -> probs.
template <int D, int PASS>
__global__ void __launch_bounds__(QU_THREADS, 1) qcache_umma_kernel(Params P) {
  KernelClock kclock(P);
  constexpr int ROWB = D * 2, CPR = D / 8, KSTEPS = D / 16;
  constexpr int TILEB = QU_TILE * ROWB;
  extern __shared__ __align__(1024) unsigned char qu_raw[];
  const int unit = blockIdx.y, b = unit / P.Hkv, h = unit % P.Hkv;
  if (P.st.score_mode[h] != HARDKV_SCORE_ACCUM_QCACHE) return;
  int n, lo, hi;
  pool_bounds(P, b, n, lo, hi);
  if (hi <= lo) return;
  const int first_page = lo >> 4, last_page = (hi - 1) >> 4;
  const int cpg0 = blockIdx.x * (QU_CPC * SCORE_PAGES_PER_CTA);                 // first page of this CTA's range
  const int pgA = max(first_page, cpg0), pgB = min(last_page, cpg0 + QU_CPC * SCORE_PAGES_PER_CTA - 1);
  if (pgA > pgB) return;
  const int tile_pg0 = cpg0 + ((pgA - cpg0) & ~7);                              // tiles are 8-page aligned
  const int T = (pgB - tile_pg0) / 8 + 1;

  unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(qu_raw) + 1023) & ~(uintptr_t)1023);
  unsigned char *ktile = smem;                                                  // [QU_STAGES][TILEB]
  unsigned char *qblk = smem + (size_t)QU_STAGES * TILEB;                       // [RB rows], swizzled
  float2 *s_aux = reinterpret_cast<float2 *>(qblk + (size_t)QC_ROWS * ROWB);    // PASS 1: [2][QC_ROWS] statistics of the two
                                                                                // warpgroups; PASS 2: [QC_ROWS] (max, weight)
  uint64_t *full = reinterpret_cast<uint64_t *>(s_aux + 2 * QC_ROWS);
  uint64_t *empty = full + QU_STAGES, *tfull = empty + QU_STAGES, *tempty = tfull + 2;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + 2);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = P.G, nc = P.st.qc_count[b];
  const int M = nc * G, RB = M <= 128 ? 128 : 256;                              // query rows, padded to the MMA shape
  const uint32_t tmem_cols = 2 * RB;                                            // two accumulator stages

  if (tid == 0) {
    for (int s = 0; s < QU_STAGES; ++s) { mbar_init(&full[s], QU_PROD_THREADS); mbar_init(&empty[s], 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(&tfull[a], 1); mbar_init(&tempty[a], 128); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == QU_MMA_WARP) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const float c2 = P.sm_scale * 1.4426950408889634f / P.st.temperature[unit];   // logit -> base-2 exponent of z / T

  if (warp > QU_MMA_WARP) {
    // ================= producers: gather the pages of tile t into stage t % QU_STAGES =================
    const int p = tid - (QU_EPI_THREADS + 32);
    const int g = p % CPR, rsub = p / CPR;
    constexpr int RPI = QU_PROD_THREADS / CPR;                                  // rows per iteration (8 at d = 128)
    const int32_t *tab = P.st.base_table + (size_t)unit * P.ppu;
    const char *kpool = reinterpret_cast<const char *>(P.st.k_pool);
    for (int t = 0; t < T; ++t) {
      const int s = t % QU_STAGES;
      mbar_wait(&empty[s], ((t / QU_STAGES) & 1) ^ 1);                          // the MMAs that read the stage have completed
      const int pg = tile_pg0 + 8 * t + (lane & 7);
      const int pid = (pg >= pgA && pg <= pgB) ? __ldg(tab + pg) : -1;           // pages outside the pool are not fetched: their
      const uint32_t dst0 = smem_u32(ktile + (size_t)s * TILEB);                //  rows hold stale data, masked in the epilogue
#pragma unroll
      for (int i = 0; i < QU_TILE / RPI; ++i) {
        const int row = i * RPI + rsub;
        const int page = __shfl_sync(0xffffffffu, pid, row >> 4);
        if (page >= 0)
          cp_async16(dst0 + umma_sw128_off(row, g, QU_TILE), kpool + ((size_t)page * PAGE + (row & 15)) * ROWB + g * 16);
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      if (t >= QU_LAG) {
        cp_async_wait<QU_LAG>();
        proxy_fence_async();
        mbar_arrive(&full[(t - QU_LAG) % QU_STAGES]);
      }
    }
    // drain: the last min(T, QU_LAG) tiles
    if (T >= 2) { cp_async_wait<1>(); proxy_fence_async(); mbar_arrive(&full[(T - 2) % QU_STAGES]); }
    cp_async_wait<0>(); proxy_fence_async(); mbar_arrive(&full[(T - 1) % QU_STAGES]);
  } else {
    // ================= the query block -> shared memory (epilogue warps), rows beyond M are zero =================
    if (warp < QU_MMA_WARP) {
      const char *qc = reinterpret_cast<const char *>(P.st.qcache);
      for (int i = tid; i < RB * CPR; i += QU_EPI_THREADS) {
        const int r = i / CPR, gq = i % CPR;
        uint4 val = make_uint4(0, 0, 0, 0);
        if (r < M) {
          const int tau = r / G, gh = r % G;
          val = ldg_ca(qc + (((size_t)(b * P.Hq + h * G + gh) * P.accum_window + tau) * D) * 2 + gq * 16);
        }
        *reinterpret_cast<uint4 *>(qblk + umma_sw128_off(r, gq, RB)) = val;
      }
      if (PASS == 2) {
        const float2 *fin = P.qc_final + (size_t)unit * QC_ROWS;
        for (int i = tid; i < QC_ROWS; i += QU_EPI_THREADS) s_aux[i] = fin[i];
      }
      proxy_fence_async();
    }
    asm volatile("bar.sync 1, %0;" ::"n"(QU_EPI_THREADS + 32) : "memory");      // epilogue warps + the MMA warp
    if (warp == QU_MMA_WARP) {
      // ================= MMA issue: one thread =================
      const uint32_t qaddr = smem_u32(qblk);
      for (int t = 0; t < T; ++t) {
        const int s = t % QU_STAGES, a = t & 1;
        mbar_wait(&full[s], (t / QU_STAGES) & 1);                               // the tile has landed
        mbar_wait(&tempty[a], ((t >> 1) & 1) ^ 1);                              // the epilogue has drained the accumulator stage
        tc_fence_after();
        proxy_fence_async();
        if (lane == 0) {
          const uint32_t kaddr = smem_u32(ktile + (size_t)s * TILEB);
          if (PASS == 1) {
            for (int rh = 0; rh < RB / 128; ++rh) {
#pragma unroll
              for (int kk = 0; kk < KSTEPS; ++kk) {
                const uint32_t o = (uint32_t)((kk & 3) * 32);
                umma_bf16(tmem + a * RB + rh * 128, umma_desc(qaddr + (kk >> 2) * (RB * 128) + rh * 16384 + o),
                          umma_desc(kaddr + (kk >> 2) * (QU_TILE * 128) + o), umma_idesc_bf16(QU_TILE), kk > 0);
              }
            }
          } else {
#pragma unroll
            for (int kk = 0; kk < KSTEPS; ++kk) {
              const uint32_t o = (uint32_t)((kk & 3) * 32);
              umma_bf16(tmem + a * RB, umma_desc(kaddr + (kk >> 2) * (QU_TILE * 128) + o),
                        umma_desc(qaddr + (kk >> 2) * (RB * 128) + o), umma_idesc_bf16(RB), kk > 0);
            }
          }
          umma_commit(&empty[s]);     // the stage goes back to the producers when these MMAs have read it
          umma_commit(&tfull[a]);     // ... and the accumulator stage to its epilogue warpgroup
        }
        __syncwarp();
      }
    } else {
      // ================= epilogue: warpgroup a drains accumulator stage a (tiles a, a + 2, ...) =================
      const int a = warp >> 2, quad = warp & 3;
      const uint32_t tlane = (uint32_t)(quad * 32) << 16;
      if (PASS == 1) {
        float m0 = -INFINITY, s0 = 0.f, m1 = -INFINITY, s1 = 0.f;              // rows quad * 32 + lane and + 128
        for (int t = a; t < T; t += 2) {
          mbar_wait(&tfull[a], (t >> 1) & 1);
          tc_fence_after();
          const int tok0 = (tile_pg0 + 8 * t) * PAGE;
          for (int rh = 0; rh < RB / 128; ++rh) {
            float m = rh ? m1 : m0, sacc = rh ? s1 : s0;
#pragma unroll 1
            for (int c0 = 0; c0 < QU_TILE; c0 += 32) {
              float v[32];
              tmem_ld32(tmem + tlane + a * RB + rh * 128 + c0, v);
              const int tk = tok0 + c0;
              const bool inside = tk >= lo && tk + 32 <= hi;
              float mx = m;
#pragma unroll
              for (int j = 0; j < 32; ++j) {
                v[j] = (inside || (tk + j >= lo && tk + j < hi)) ? v[j] * c2 : -INFINITY;
                mx = fmaxf(mx, v[j]);
              }
              if (mx != -INFINITY) {
                float acc = 0.f;
#pragma unroll
                for (int j = 0; j < 32; ++j) acc += fast_exp2(v[j] - mx);
                sacc = sacc * fast_exp2(m - mx) + acc;
                m = mx;
              }
            }
            if (rh) { m1 = m; s1 = sacc; } else { m0 = m; s0 = sacc; }
          }
          tc_fence_before();
          mbar_arrive(&tempty[a]);
        }
        // the two warpgroups' statistics -> one (max, sum) per row -> this CTA's first chunk slot; its other slots stay neutral
        const int r0 = quad * 32 + lane;
        s_aux[a * QC_ROWS + r0] = make_float2(m0, s0);
        s_aux[a * QC_ROWS + r0 + 128] = make_float2(m1, s1);
        asm volatile("bar.sync 2, %0;" ::"n"(QU_EPI_THREADS) : "memory");
        const int ch0 = max(first_page / SCORE_PAGES_PER_CTA, (int)blockIdx.x * QU_CPC);
        const int ch1 = min(last_page / SCORE_PAGES_PER_CTA, (int)blockIdx.x * QU_CPC + QU_CPC - 1);
        float2 *outp = P.qc_stats + ((size_t)unit * P.score_chunks + ch0) * QC_ROWS;
        for (int col = tid; col < QC_ROWS; col += QU_EPI_THREADS) {
          const float2 x = s_aux[col], y = s_aux[QC_ROWS + col];
          const float mm = fmaxf(x.x, y.x);
          float ss = 0.f;
          if (x.x != -INFINITY) ss += x.y * fast_exp2(x.x - mm);
          if (y.x != -INFINITY) ss += y.y * fast_exp2(y.x - mm);
          const bool live = col < RB;
          outp[col] = live ? make_float2(mm, ss) : make_float2(-INFINITY, 0.f);
          for (int c = ch0 + 1; c <= ch1; ++c) outp[(size_t)(c - ch0) * QC_ROWS + col] = make_float2(-INFINITY, 0.f);
        }
      } else {
        float *probs = P.st.probs + (size_t)unit * P.max_ctx;
        const int ncol = (M + 31) & ~31;                                        // rows beyond M carry weight 0: skip whole groups
        for (int t = a; t < T; t += 2) {
          mbar_wait(&tfull[a], (t >> 1) & 1);
          tc_fence_after();
          const int tok = (tile_pg0 + 8 * t) * PAGE + quad * 32 + lane;
          float sum = 0.f;
#pragma unroll 1
          for (int c0 = 0; c0 < ncol; c0 += 32) {
            float v[32];
            tmem_ld32(tmem + tlane + a * RB + c0, v);
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const float2 f = s_aux[c0 + j];                                   // (row max in base-2 units, 1 / (row sum * G * n_c))
              sum = fmaf(fast_exp2(fmaf(v[j], c2, -f.x)), f.y, sum);
            }
          }
          tc_fence_before();
          mbar_arrive(&tempty[a]);
          if (tok >= lo && tok < hi) probs[tok] = sum;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == QU_MMA_WARP) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(tmem_cols));
  }
}

}  // namespace hardkv
