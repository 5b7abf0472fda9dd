// common.cuh -- shared device helpers of libhardkv (sm_100a). Product code: never includes oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/hardkv.h"

namespace hardkv {

constexpr int PAGE = 16;

// Everything a kernel needs, passed by value (no device-side config object to keep in sync).
struct Params {
  int B, Hq, Hkv, G, d, max_ctx, sink, recent, k_cap, cond_cap, accum_window;
  int reuse_max;  // most steps between two compressions: the dense tier may hold recent + reuse_max rows
  int ppu;        // base pages per unit  = max_ctx / PAGE
  int spu;        // selected pages per unit = k_cap / PAGE
  int att_chunks; // static number of attention chunks per unit
  float sm_scale;
  hardkv_state st;
  // workspace
  float *part;          // [units][att_chunks][G][d + 2] split-K partial states (m, l, acc[d])
  int32_t *att_arrive;  // [units] arrival counters of the split-K merge (zero between launches)
  float2 *score_stats;   // [units][score_chunks][8] per (chunk, query head): (max, sum of 2^(x - max)) of x = z*log2(e)/T
  int score_chunks;
  int sel_cluster;       // CTAs per (b, h) cluster of the select kernel
  int sel_slice_cap;     // capacity (tokens) of one CTA's probability slice in shared memory
  int sel_nt;            // threads per CTA of the select kernel (512 or 1024)
  float *pooled;         // [B][Hq][max_ctx] max-pooled logits of SNAPKV heads (NULL when pool_kernel <= 1)
  int pool_kernel;       // SNAPKV max-pool window (odd), <= 1: no SNAPKV head in this config
  int cond_merge;        // 1: evictees of a full condensed tier are merged into a resident (Appendix G)
  // fused score -> select kernel (score_select.cuh)
  int ss_slice_cap;      // capacity (tokens) of the probability slice of one unit held by one 1024-thread CTA
  int32_t *ss_next;      // [1] next work item (zero between launches)
  int32_t *ss_arrive;    // [units] chunks of a unit scanned so far (zero between launches)
  // select -> attention overlap (hardkv_decode_step with programmatic dependent launch)
  int32_t *epoch;        // [1] decode steps appended so far: the append kernel bumps it, select publishes it per unit
  int32_t *sel_flag;     // [units] == *epoch once the unit's selection of this step is complete and visible
  int32_t *unit_order;   // [units] units by increasing pool length (the order their selections finish in)
  // Forked append (hardkv_decode_step): the append / retire kernel runs beside the score kernel and does NOT write the
  // per-sequence scalars ctx_len / c_lo / dense_lo in place (the score kernel is reading them) but into sh_scal; the
  // kernels after the join read them there (use_shadow), and the attention kernel writes them back in place.
  int pre_append;        // score launch: pool bounds as the step's append kernel will leave them (pool_bounds)
  int defer_commit;      // append launch: scalars -> sh_scal
  int use_shadow;        // launches after the join: scalars <- sh_scal
  int32_t *sh_scal;      // [3][B]: ctx_len, c_lo, dense_lo after this step's append / retirement
  int wait_select;       // attention launch: 1 = launched programmatically behind the select kernel: wait per unit, units by
                         // increasing pool length; 2 = the same behind the score || select pair: longest pool first
  int32_t *score_flag;   // [units] == *epoch once every logit / chunk statistic of the unit is stored (score || select overlap)
  // query-cache form of the accumulated-attention metric (qcache_kernels.cuh)
  float2 *qc_stats;      // [units][score_chunks][256] per chunk and query row: (max, sum 2^(x - max)) of x = z log2(e) / T
  float2 *qc_final;      // [units][256] per query row: (max, 1 / (sum * G * n_c))
  int st_esize;          // bytes of one q / K / V element
  // in-graph kernel timing (hardkv_set_timing): NULL in normal runs
  unsigned long long *timing;   // [2 * slots]: (start of the first CTA, end of the last CTA) in globaltimer ns per launch
  int timing_slot;
};

// Records when the first CTA of a launch starts and when its last CTA ends (thread 0 of every CTA: one atomicMin, one
// atomicMax), so that bench.py can report each kernel's duration INSIDE the captured graph it times.  Costs nothing
// when P.timing is NULL.  The destructor covers every return path.
struct KernelClock {
  unsigned long long *slot;
  static __device__ __forceinline__ unsigned long long now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
  }
  __device__ __forceinline__ explicit KernelClock(const Params &P) : slot(P.timing ? P.timing + 2 * P.timing_slot : nullptr) {
    if (slot && threadIdx.x == 0) atomicMin(slot, now());
  }
  __device__ __forceinline__ ~KernelClock() {
    if (slot && threadIdx.x == 0) atomicMax(slot + 1, now());
  }
};

// ---- programmatic dependent launch (PDL): every hot kernel waits here for the preceding kernel of the stream to complete
// and flush before it touches memory, then lets its own successor be scheduled onto SMs as they drain -- the launch
// latency between the dependent kernels of a step overlaps the tail of the previous kernel.  Both are no-ops when the
// kernel was launched without the attribute.
__device__ __forceinline__ void pdl_wait_then_trigger() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Consumer side of the select -> attention overlap: the attention kernel is launched programmatically behind the select
// kernel (its CTAs take the SMs that select CTAs leave) and each CTA waits here until its unit's selection of this step is
// published.  Deadlock-free: every select CTA is resident before the first attention CTA exists.  A watchdog turns a
// protocol error into err_flag = 120 instead of a hang.
__device__ __forceinline__ void wait_unit_selected(const Params &P, int unit) {
  if (threadIdx.x == 0) {
    const int want = *reinterpret_cast<volatile int32_t *>(P.epoch);
    volatile int32_t *f = P.sel_flag + unit;
    unsigned polls = 0;
    while (*f != want) {
      __nanosleep(100);
      if (++polls > (1u << 24)) { atomicCAS(P.st.err_flag, 0, 120); break; }
    }
    __threadfence();    // acquire: the unit's sel_idx / sel_count / probs are visible to this CTA after the barrier
  }
  __syncthreads();
}

// Consumer side of the score || select overlap: the select kernel is launched programmatically behind the persistent
// score kernel (every score CTA is resident before the first select CTA exists, and no score CTA ever waits for
// anything, so the wait is deadlock-free) and takes a unit as soon as the score kernel has published it.
__device__ __forceinline__ void wait_unit_scored(const Params &P, int unit) {
  if (threadIdx.x == 0) {
    const int want = *reinterpret_cast<volatile int32_t *>(P.epoch);
    volatile int32_t *f = P.score_flag + unit;
    unsigned polls = 0;
    while (*f != want) {
      __nanosleep(200);
      if (++polls > (1u << 24)) { atomicCAS(P.st.err_flag, 0, 121); break; }
    }
    __threadfence();
  }
  __syncthreads();
}

// ---- 16-byte vector access -------------------------------------------------------------------
__device__ __forceinline__ uint4 ldg_nc(const void *p) {   // streaming read-only data (K, V rows)
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
// the same at base + OFF with the offset as an immediate of the instruction (no per-load address arithmetic)
template <int OFF>
__device__ __forceinline__ uint4 ldg_nc_off(const void *base) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4+%5];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(base), "n"(OFF));
  return v;
}
__device__ __forceinline__ uint4 ldg_ca(const void *p) { return *reinterpret_cast<const uint4 *>(p); }
__device__ __forceinline__ void stg(void *p, uint4 v) { *reinterpret_cast<uint4 *>(p) = v; }
// streaming store (evict-first in L2): the rewritten tier is not read again before the next step's K scan has pushed
// it out of L2 anyway, so its write-back should drain during the attention kernel (DRAM at ~40 %) rather than sit
// dirty in L2 and compete with the bandwidth-bound score kernel of the next step
__device__ __forceinline__ void stg_cs(void *p, uint4 v) {
  asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// Elements per 16-byte vector and their widening to fp32 (bf16 -> fp32 is exact: a 16-bit shift).
template <typename T> struct Elem;
template <> struct Elem<float> {
  static constexpr int EPL = 4;
  __device__ static __forceinline__ void unpack(const uint4 &r, float (&f)[4]) {
    f[0] = __uint_as_float(r.x); f[1] = __uint_as_float(r.y);
    f[2] = __uint_as_float(r.z); f[3] = __uint_as_float(r.w);
  }
  __device__ static __forceinline__ uint4 pack(const float (&f)[4]) {
    return make_uint4(__float_as_uint(f[0]), __float_as_uint(f[1]), __float_as_uint(f[2]), __float_as_uint(f[3]));
  }
};
struct bf16_t { uint16_t bits; };
template <> struct Elem<bf16_t> {
  static constexpr int EPL = 8;
  __device__ static __forceinline__ void unpack(const uint4 &r, float (&f)[8]) {
    f[0] = __uint_as_float(r.x << 16); f[1] = __uint_as_float(r.x & 0xffff0000u);
    f[2] = __uint_as_float(r.y << 16); f[3] = __uint_as_float(r.y & 0xffff0000u);
    f[4] = __uint_as_float(r.z << 16); f[5] = __uint_as_float(r.z & 0xffff0000u);
    f[6] = __uint_as_float(r.w << 16); f[7] = __uint_as_float(r.w & 0xffff0000u);
  }
  __device__ static __forceinline__ uint4 pack(const float (&f)[8]) {   // round to nearest even
    auto two = [](float lo, float hi) {
      return (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(lo)) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(hi)) << 16);
    };
    return make_uint4(two(f[0], f[1]), two(f[2], f[3]), two(f[4], f[5]), two(f[6], f[7]));
  }
};

// Address of row `pos` of a unit in a paged pool (table holds the physical page of logical page pos/16).
template <typename T, int D>
__device__ __forceinline__ const char *paged_row(const void *pool, const int32_t *table_unit, int pos) {
  int page = __ldg(table_unit + (pos >> 4));
  return reinterpret_cast<const char *>(pool) + ((size_t)page * PAGE + (pos & 15)) * (D * sizeof(T));
}

// Pool bounds of sequence b (Tier-2 address range): [lo, hi).
// pre_append: the arithmetic of append_retire_kernel on the scalars it has not written: n + 1 unless the context is
// full, and c_lo pushed up until the pool fits l_upper (a compression step).
__device__ __forceinline__ void pool_bounds(const Params &P, int b, int &n, int &lo, int &hi) {
  if (P.use_shadow) {
    n = P.sh_scal[b];
    lo = P.sh_scal[P.B + b];
  } else {
    n = P.st.ctx_len[b];
    lo = P.st.c_lo[b];
    if (P.pre_append && n < P.max_ctx) {
      n += 1;
      const int over = n - P.recent - lo - P.st.l_upper[b];
      if (over > 0) lo += over;
    }
  }
  hi = n - P.recent;
  if (hi < lo) hi = lo;
}

__device__ __forceinline__ float fast_exp2(float x) {   // MUFU.EX2; 2^-inf = +0
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float warp_max_f32(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum_f32(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// Dense tier of sequence b with context n (PAPER.md L71, L78 steps 1-2): sinks [0, s_end) and [r_lo, n), r_lo = dense_lo
// = n - recent at the last compression step.  Returns false (the caller flags the unit) when the tier outgrew the
// recent + reuse_max rows the attention grid was sized for.
__device__ __forceinline__ bool dense_bounds(const Params &P, int b, int n, int &s_end, int &r_lo) {
  s_end = min(P.sink, n);
  r_lo = min(max(P.use_shadow ? P.sh_scal[2 * P.B + b] : P.st.dense_lo[b], s_end), n);
  return n - r_lo <= P.recent + P.reuse_max;
}

constexpr int SCORE_PAGES_PER_CTA = 64;  // score kernel: 8 warps x 8 pages = 1024 tokens = 256 KiB of K per CTA

__device__ __forceinline__ unsigned long long shfl_xor_u64(unsigned long long v, int off) {
  unsigned lo = __shfl_xor_sync(0xffffffffu, (unsigned)v, off);
  unsigned hi = __shfl_xor_sync(0xffffffffu, (unsigned)(v >> 32), off);
  return ((unsigned long long)hi << 32) | lo;
}
__device__ __forceinline__ unsigned long long shfl_up_u64(unsigned long long v, int off) {
  unsigned lo = __shfl_up_sync(0xffffffffu, (unsigned)v, off);
  unsigned hi = __shfl_up_sync(0xffffffffu, (unsigned)(v >> 32), off);
  return ((unsigned long long)hi << 32) | lo;
}
__device__ __forceinline__ unsigned long long shfl_u64(unsigned long long v, int src) {
  unsigned lo = __shfl_sync(0xffffffffu, (unsigned)v, src);
  unsigned hi = __shfl_sync(0xffffffffu, (unsigned)(v >> 32), src);
  return ((unsigned long long)hi << 32) | lo;
}
__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += shfl_xor_u64(v, o);
  return v;
}

}  // namespace hardkv
