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
// Warp roles (13 warps): 0-3 and 4-7 = two epilogue warpgroups (even / odd tiles); 8 = TMEM allocation and the single
// MMA-issuing thread; 9-12 = producers.  Pipelines: full / empty mbarriers over the K-tile stages (producers <-> MMA,
// released by tcgen05.commit), tfull / tempty over the accumulator stages in TMEM (MMA <-> epilogue; 512 columns = four
// stages of 128 or two of 256).
#pragma once
#include "common.cuh"
#include "qcache_kernels.cuh"
#include "score_tma.cuh"   // mbarrier helpers, smem_u32

namespace hardkv {

constexpr int QU_TILE = 128;            // pool tokens per tile (8 pages)
#ifndef HARDKV_QU_STAGES
#define HARDKV_QU_STAGES 4
#endif
#ifndef HARDKV_QU_LAG
#define HARDKV_QU_LAG 2
#endif
constexpr int QU_STAGES = HARDKV_QU_STAGES;   // K tiles in shared memory
constexpr int QU_LAG = HARDKV_QU_LAG;         // a producer signals tile t - QU_LAG after issuing tile t: QU_LAG + 1 tiles in flight
#ifndef HARDKV_QU_PROD
#define HARDKV_QU_PROD 128
#endif
constexpr int QU_EPI_THREADS = 256, QU_MMA_WARP = 8, QU_PROD_THREADS = HARDKV_QU_PROD;
constexpr int QU_THREADS = QU_EPI_THREADS + 32 + QU_PROD_THREADS;

// rows = the query block's capacity for this config: 128 or 256 (accum_window * G rounded up to the MMA shape)
__host__ __device__ inline int qcache_umma_rows(int accum_window, int G) { return accum_window * G <= 128 ? 128 : 256; }
__host__ __device__ inline size_t qcache_umma_smem(int d, int rows) {
  return (size_t)QU_STAGES * QU_TILE * d * 2 + (size_t)rows * d * 2 + 1024;   // + 4.2 KB static (statistics, barriers)
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
// 32 consecutive fp32 columns of this thread's TMEM lane: the load is asynchronous, the registers are valid after
// tmem_ld_wait() -- issue the next group's load before working on the current one
__device__ __forceinline__ void tmem_ld32_issue(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,"
               "%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
                 "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
                 "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
               : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// byte offset of 16-byte chunk g of row r inside an operand block of `rows` rows (K halves of 64 elements back to back)
__device__ __forceinline__ uint32_t umma_sw128_off(int r, int g, int rows) {
  return (uint32_t)((g >> 3) * (rows * 128) + (r >> 3) * 1024 + (r & 7) * 128 + (((g & 7) ^ (r & 7)) << 4));
}


constexpr int QU_MAX_UNITS = 1024;      // capacity of the per-CTA item index (units beyond it: the mma.sync kernels run instead)

// One work item = one score chunk (64 pages = up to 8 tiles) of one query-cache unit.
struct QuItem {
  int unit, b, h, chunk, lo, hi, pgA, pgB, tile_pg0, T, M, RB;
};

// PASS 1: per-(chunk, query row) softmax statistics -> qc_stats; PASS 2: probabilities summed over the query rows -> probs.
// Persistent: one CTA per SM takes a contiguous block of the item list; the K-tile ring and the TMEM accumulator stages
// run on across items (a global tile counter gives stage and parity), the query block is reloaded only when the unit
// changes, by the epilogue warps, while the producers already fetch the next tiles.
template <int D, int PASS>
__global__ void __launch_bounds__(QU_THREADS, 1) qcache_umma_kernel(Params P) {
  KernelClock kclock(P);
  constexpr int ROWB = D * 2, CPR = D / 8, KSTEPS = D / 16;
  constexpr int TILEB = QU_TILE * ROWB;
  constexpr int SPC = SCORE_PAGES_PER_CTA;
  extern __shared__ __align__(1024) unsigned char qu_raw[];
  unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(qu_raw) + 1023) & ~(uintptr_t)1023);
  unsigned char *ktile = smem;                                                  // [QU_STAGES][TILEB]
  unsigned char *qblk = smem + (size_t)QU_STAGES * TILEB;                       // [RBmax rows], swizzled
  __shared__ __align__(16) float2 s_aux[2 * QC_ROWS];   // PASS 1: [2][QC_ROWS] statistics of the two warpgroups; PASS 2: (max, weight)
  __shared__ uint64_t full[QU_STAGES], empty[QU_STAGES], tfull[4], tempty[4];
  __shared__ uint32_t tmem_slot[1];
  __shared__ int s_first[QU_MAX_UNITS + 1];             // first item of every unit (exclusive prefix sum of the chunk counts)

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int units = P.B * P.Hkv, G = P.G;
  const int RBmax = qcache_umma_rows(P.accum_window, G);
  const int NACC = 512 / RBmax;                                                 // accumulator stages in TMEM: 4 or 2
  const uint32_t tmem_cols = 512;

  if (tid == 0) {
    for (int s = 0; s < QU_STAGES; ++s) { mbar_init(&full[s], QU_PROD_THREADS); mbar_init(&empty[s], 1); }
    for (int a = 0; a < 4; ++a) { mbar_init(&tfull[a], 1); mbar_init(&tempty[a], 128); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {   // chunk counts of the units -> exclusive prefix sum
    int run = 0;
    for (int u0 = 0; u0 < units; u0 += 32) {
      const int u = u0 + lane;
      int cnt = 0;
      if (u < units && P.st.score_mode[u % P.Hkv] == HARDKV_SCORE_ACCUM_QCACHE) {
        int n, lo, hi;
        pool_bounds(P, u / P.Hkv, n, lo, hi);
        if (hi > lo) cnt = ((hi - 1) >> 4) / SPC - (lo >> 4) / SPC + 1;
      }
      int inc = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t_ = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t_;
      }
      if (u < units) s_first[u] = run + inc - cnt;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) s_first[units] = run;
  }
  if (warp == QU_MMA_WARP) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const int nitems = s_first[units];
  // a CTA takes a contiguous block of items: consecutive chunks of (mostly) one unit, so the query block is reloaded once
  // or twice per CTA, not per item; items are equal-sized up to the units' partial first / last chunks
  const int it_begin = (int)(((long long)blockIdx.x * nitems) / gridDim.x);
  const int it_end = (int)(((long long)(blockIdx.x + 1) * nitems) / gridDim.x);

  auto decode = [&](int it, QuItem &I) {
    int ul = 0, uh = units - 1;
    while (ul < uh) {
      const int mid = (ul + uh + 1) >> 1;
      if (s_first[mid] <= it) ul = mid; else uh = mid - 1;
    }
    I.unit = ul; I.b = ul / P.Hkv; I.h = ul % P.Hkv;
    int n;
    pool_bounds(P, I.b, n, I.lo, I.hi);
    const int first_page = I.lo >> 4, last_page = (I.hi - 1) >> 4;
    I.chunk = first_page / SPC + (it - s_first[ul]);
    const int cpg0 = I.chunk * SPC;
    I.pgA = max(first_page, cpg0); I.pgB = min(last_page, cpg0 + SPC - 1);
    I.tile_pg0 = cpg0 + ((I.pgA - cpg0) & ~7);                                  // tiles are 8-page aligned
    I.T = (I.pgB - I.tile_pg0) / 8 + 1;
    I.M = P.st.qc_count[I.b] * G;
    I.RB = I.M <= 128 ? 128 : 256;                                              // query rows, padded to the MMA shape
  };

  if (warp > QU_MMA_WARP) {
    // ================= producers: gather the pages of every tile into the ring, LAG + 1 tiles in flight =================
    const int p = tid - (QU_EPI_THREADS + 32);
    const int g = p % CPR, rsub = p / CPR;
    constexpr int RPI = QU_PROD_THREADS / CPR;                                  // rows per iteration (8 at d = 128)
    const char *kpool = reinterpret_cast<const char *>(P.st.k_pool);
    // the physical ids of an item's (<= 64) pages with one coalesced load per 32 pages, fetched one item ahead; pages
    // outside the pool are not fetched (their rows hold stale data, masked in the epilogue)
    auto page_ids = [&](const QuItem &I, int &p0, int &p1) {
      const int32_t *tab = P.st.base_table + (size_t)I.unit * P.ppu;
      const int pg = I.tile_pg0 + lane;
      p0 = (pg >= I.pgA && pg <= I.pgB) ? __ldg(tab + pg) : -1;
      p1 = (pg + 32 >= I.pgA && pg + 32 <= I.pgB) ? __ldg(tab + pg + 32) : -1;
    };
    QuItem I, In;
    int pid0 = -1, pid1 = -1, np0 = -1, np1 = -1;
    int it = it_begin, gi = 0;
    if (it < it_end) { decode(it, I); page_ids(I, pid0, pid1); }
    while (it < it_end) {
      const int itn = it + 1;
      if (itn < it_end) { decode(itn, In); page_ids(In, np0, np1); }
      for (int t = 0; t < I.T; ++t, ++gi) {
        const int s = gi % QU_STAGES;
        mbar_wait(&empty[s], ((gi / QU_STAGES) & 1) ^ 1);                       // the MMAs that read the stage have completed
        const int pidw = (t >> 2) ? pid1 : pid0;
        const uint32_t dst0 = smem_u32(ktile + (size_t)s * TILEB);
#pragma unroll
        for (int i = 0; i < QU_TILE / RPI; ++i) {
          const int row = i * RPI + rsub;
          const int page = __shfl_sync(0xffffffffu, pidw, (t & 3) * 8 + (row >> 4));
          if (page >= 0)
            cp_async16(dst0 + umma_sw128_off(row, g, QU_TILE), kpool + ((size_t)page * PAGE + (row & 15)) * ROWB + g * 16);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        if (gi >= QU_LAG) {
          cp_async_wait<QU_LAG>();
          proxy_fence_async();
          mbar_arrive(&full[(gi - QU_LAG) % QU_STAGES]);
        }
      }
      I = In; pid0 = np0; pid1 = np1; it = itn;
    }
    // drain: the last min(gi, QU_LAG) tiles
    if (QU_LAG >= 3 && gi >= 3) { cp_async_wait<2>(); proxy_fence_async(); mbar_arrive(&full[(gi - 3) % QU_STAGES]); }
    if (QU_LAG >= 2 && gi >= 2) { cp_async_wait<1>(); proxy_fence_async(); mbar_arrive(&full[(gi - 2) % QU_STAGES]); }
    if (gi >= 1) { cp_async_wait<0>(); proxy_fence_async(); mbar_arrive(&full[(gi - 1) % QU_STAGES]); }
  } else if (warp == QU_MMA_WARP) {
    // ================= MMA issue: one thread =================
    const uint32_t qaddr = smem_u32(qblk);
    QuItem I;
    int gi = 0, prev_unit = -1;
    for (int it = it_begin; it < it_end; ++it) {
      decode(it, I);
      if (I.unit != prev_unit)
        asm volatile("bar.sync 1, %0;" ::"n"(QU_EPI_THREADS + 32) : "memory");  // the unit's query block is in shared memory
      prev_unit = I.unit;
      const int RB = I.RB;
      for (int t = 0; t < I.T; ++t, ++gi) {
        const int s = gi % QU_STAGES, a = gi % NACC;
        mbar_wait(&full[s], (gi / QU_STAGES) & 1);                              // the tile has landed
        mbar_wait(&tempty[a], ((gi / NACC) & 1) ^ 1);                           // the epilogue has drained the accumulator stage
        tc_fence_after();
        proxy_fence_async();
        if (lane == 0) {
          const uint32_t kaddr = smem_u32(ktile + (size_t)s * TILEB);
          const uint32_t dcol = tmem + a * RBmax;
          if (PASS == 1) {
            for (int rh = 0; rh < RB / 128; ++rh) {
#pragma unroll
              for (int kk = 0; kk < KSTEPS; ++kk) {
                const uint32_t o = (uint32_t)((kk & 3) * 32);
                umma_bf16(dcol + rh * 128, umma_desc(qaddr + (kk >> 2) * (RB * 128) + rh * 16384 + o),
                          umma_desc(kaddr + (kk >> 2) * (QU_TILE * 128) + o), umma_idesc_bf16(QU_TILE), kk > 0);
              }
            }
          } else {
#pragma unroll
            for (int kk = 0; kk < KSTEPS; ++kk) {
              const uint32_t o = (uint32_t)((kk & 3) * 32);
              umma_bf16(dcol, umma_desc(kaddr + (kk >> 2) * (QU_TILE * 128) + o),
                        umma_desc(qaddr + (kk >> 2) * (RB * 128) + o), umma_idesc_bf16(RB), kk > 0);
            }
          }
          umma_commit(&empty[s]);     // the stage goes back to the producers when these MMAs have read it
          umma_commit(&tfull[a]);     // ... and the accumulator stage to its epilogue warpgroup
        }
        __syncwarp();
      }
    }
  } else {
    // ================= epilogue: warpgroup wg drains the tiles of its parity =================
    const int wg = warp >> 2, quad = warp & 3;
    const uint32_t tlane = (uint32_t)(quad * 32) << 16;
    const char *qc = reinterpret_cast<const char *>(P.st.qcache);
    QuItem I;
    int gi = 0, prev_unit = -1;
    // PASS 1: the statistics of a thread's rows run on over all of this CTA's chunks of a unit (the reduction over the
    // chunk slots only needs SOME partition of the pool): one flush per unit into the slot of the first chunk, the CTA's
    // other slots of the unit are written neutral
    float m0 = -INFINITY, s0 = 0.f, m1 = -INFINITY, s1 = 0.f;                  // rows quad * 32 + lane and + 128 (logit units)
    int run_chunk0 = 0, run_chunk1 = -1, run_rb = 128;
    float run_c2 = 1.f;
    auto flush = [&]() {   // after a bar.sync 2 has NOT yet been passed: every thread publishes, then combines
      const int r0 = quad * 32 + lane;
      s_aux[wg * QC_ROWS + r0] = make_float2(m0 * run_c2, s0);                  // logit units -> base-2 exponent units
      s_aux[wg * QC_ROWS + r0 + 128] = make_float2(m1 * run_c2, s1);
      asm volatile("bar.sync 2, %0;" ::"n"(QU_EPI_THREADS) : "memory");
      float2 *outp = P.qc_stats + ((size_t)prev_unit * P.score_chunks + run_chunk0) * QC_ROWS;
      const int col = tid;                                                      // QU_EPI_THREADS == QC_ROWS
      const float2 x = s_aux[col], y = s_aux[QC_ROWS + col];
      const float mm = fmaxf(x.x, y.x);
      float ss = 0.f;
      if (x.x != -INFINITY) ss += x.y * fast_exp2(x.x - mm);
      if (y.x != -INFINITY) ss += y.y * fast_exp2(y.x - mm);
      outp[col] = col < run_rb ? make_float2(mm, ss) : make_float2(-INFINITY, 0.f);
      for (int c = run_chunk0 + 1; c <= run_chunk1; ++c) outp[(size_t)(c - run_chunk0) * QC_ROWS + col] = make_float2(-INFINITY, 0.f);
      m0 = m1 = -INFINITY; s0 = s1 = 0.f;
    };
    for (int it = it_begin; it < it_end; ++it) {
      decode(it, I);
      const int M = I.M, RB = I.RB, lo = I.lo, hi = I.hi;
      if (I.unit != prev_unit) {
        if (PASS == 1 && prev_unit >= 0) flush();
        // both warpgroups are through with the previous unit: all of its MMAs have completed, the query block and s_aux are free
        asm volatile("bar.sync 2, %0;" ::"n"(QU_EPI_THREADS) : "memory");
        run_chunk0 = I.chunk;
        for (int i = tid; i < RB * CPR; i += QU_EPI_THREADS) {                  // the unit's query block; rows beyond M are zero
          const int r = i / CPR, gq = i % CPR;
          uint4 val = make_uint4(0, 0, 0, 0);
          if (r < M) {
            const int tau = r / G, gh = r % G;
            val = ldg_ca(qc + (((size_t)(I.b * P.Hq + I.h * G + gh) * P.accum_window + tau) * D) * 2 + gq * 16);
          }
          *reinterpret_cast<uint4 *>(qblk + umma_sw128_off(r, gq, RB)) = val;
        }
        if (PASS == 2) {
          const float2 *fin = P.qc_final + (size_t)I.unit * QC_ROWS;
          for (int i = tid; i < QC_ROWS; i += QU_EPI_THREADS) s_aux[i] = fin[i];
        }
        proxy_fence_async();
        asm volatile("bar.sync 1, %0;" ::"n"(QU_EPI_THREADS + 32) : "memory");  // with the MMA warp
      }
      prev_unit = I.unit;
      const float c2 = P.sm_scale * 1.4426950408889634f / P.st.temperature[I.unit];   // logit -> base-2 exponent of z / T
      if (PASS == 1) {
        run_chunk1 = I.chunk; run_rb = RB; run_c2 = c2;
        for (int t = 0; t < I.T; ++t) {
          const int gt = gi + t;
          if ((gt & 1) != wg) continue;
          const int a = gt % NACC;
          mbar_wait(&tfull[a], (gt / NACC) & 1);
          tc_fence_after();
          const int tok0 = (I.tile_pg0 + 8 * t) * PAGE;
          for (int rh = 0; rh < RB / 128; ++rh) {
            float m = rh ? m1 : m0, sacc = rh ? s1 : s0;
            const uint32_t tbase = tmem + tlane + a * RBmax + rh * 128;
            uint32_t rb[2][32];                                                 // two groups of 32 columns: one in flight
            tmem_ld32_issue(tbase, rb[0]);
            tmem_ld_wait();
#pragma unroll
            for (int cg = 0; cg < QU_TILE / 32; ++cg) {
              if (cg + 1 < QU_TILE / 32) tmem_ld32_issue(tbase + (cg + 1) * 32, rb[(cg + 1) & 1]);
              float v[32];
#pragma unroll
              for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(rb[cg & 1][j]);
              const int tk = tok0 + cg * 32;
              if (!(tk >= lo && tk + 32 <= hi)) {                               // warp-uniform: only the pool's first / last tile
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = (tk + j >= lo && tk + j < hi) ? v[j] : -INFINITY;
              }
              // m is kept in logit units (c2 > 0: the maximum commutes with the scale); four independent chains
              float x0 = fmaxf(v[0], v[1]), x1 = fmaxf(v[2], v[3]), x2 = fmaxf(v[4], v[5]), x3 = fmaxf(v[6], v[7]);
#pragma unroll
              for (int j = 8; j < 32; j += 4) {
                x0 = fmaxf(x0, v[j]); x1 = fmaxf(x1, v[j + 1]); x2 = fmaxf(x2, v[j + 2]); x3 = fmaxf(x3, v[j + 3]);
              }
              const float mx = fmaxf(fmaxf(fmaxf(x0, x1), fmaxf(x2, x3)), m);
              if (mx != -INFINITY) {
                const float nb = -mx * c2;
                float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll
                for (int j = 0; j < 32; j += 4) {
                  a0 += fast_exp2(fmaf(v[j], c2, nb)); a1 += fast_exp2(fmaf(v[j + 1], c2, nb));
                  a2 += fast_exp2(fmaf(v[j + 2], c2, nb)); a3 += fast_exp2(fmaf(v[j + 3], c2, nb));
                }
                sacc = sacc * fast_exp2(fmaf(m, c2, nb)) + ((a0 + a1) + (a2 + a3));
                m = mx;
              }
              tmem_ld_wait();                                                   // the next group has landed
            }
            if (rh) { m1 = m; s1 = sacc; } else { m0 = m; s0 = sacc; }
          }
          tc_fence_before();
          mbar_arrive(&tempty[a]);
        }
      } else {
        float *probs = P.st.probs + (size_t)I.unit * P.max_ctx;
        const int ncol = (M + 31) & ~31;                                        // rows beyond M carry weight 0: skip whole groups
        for (int t = 0; t < I.T; ++t) {
          const int gt = gi + t;
          if ((gt & 1) != wg) continue;
          const int a = gt % NACC;
          mbar_wait(&tfull[a], (gt / NACC) & 1);
          tc_fence_after();
          const int tok = (I.tile_pg0 + 8 * t) * PAGE + quad * 32 + lane;
          float sum = 0.f, sum1 = 0.f, sum2 = 0.f, sum3 = 0.f;
#ifdef QU_PROBE_NOEPI
          for (int c0 = 0; c0 < 0; c0 += 32) {
#else
#pragma unroll 1
          for (int c0 = 0; c0 < ncol; c0 += 32) {
#endif
            float v[32];
            {
              uint32_t r[32];
              tmem_ld32_issue(tmem + tlane + a * RBmax + c0, r);
              tmem_ld_wait();
#pragma unroll
              for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
            }
#pragma unroll
            for (int j = 0; j < 32; j += 4) {
              const float4 f01 = *reinterpret_cast<const float4 *>(&s_aux[c0 + j]);      // (row max in base-2 units,
              const float4 f23 = *reinterpret_cast<const float4 *>(&s_aux[c0 + j + 2]);  //  1 / (row sum * G * n_c)) x 2
              sum = fmaf(fast_exp2(fmaf(v[j], c2, -f01.x)), f01.y, sum);
              sum1 = fmaf(fast_exp2(fmaf(v[j + 1], c2, -f01.z)), f01.w, sum1);
              sum2 = fmaf(fast_exp2(fmaf(v[j + 2], c2, -f23.x)), f23.y, sum2);
              sum3 = fmaf(fast_exp2(fmaf(v[j + 3], c2, -f23.z)), f23.w, sum3);
            }
          }
          sum = (sum + sum1) + (sum2 + sum3);
          tc_fence_before();
          mbar_arrive(&tempty[a]);
          if (tok >= lo && tok < hi) probs[tok] = sum;
        }
      }
      gi += I.T;
    }
    if (PASS == 1 && prev_unit >= 0) flush();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == QU_MMA_WARP) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(tmem_cols));
  }
}

}  // namespace hardkv
