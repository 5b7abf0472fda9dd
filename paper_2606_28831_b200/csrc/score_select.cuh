// score_select.cuh -- stages 1 + 2a-2c as ONE persistent kernel (sm_100a): the K scan of every unit and, hidden under
// it, the calibrated Top-p selection of the units whose scan has finished.
//   score:  z[g][i] = sm_scale * q_g . k_i over the pool (exponent of Eq. 4)
//   select: Logits Calibration (L106-128), Top-p (L108), compaction + votes + block table (L86) -- select_unit()
//
// Why one kernel.  The scan is bound by HBM (the chip-wide stream saturates with ~125 of the 148 SMs busy: measured,
// DESIGN.md section 7), the selection by issue slots and latency with almost no DRAM traffic; run back to back the
// selection left the memory system idle for 40 us of a 227 us step.  Here one CTA per SM streams K pages; the CTA that
// retires the LAST chunk of a unit (an arrival counter per unit: no CTA ever waits for another one) switches role and
// runs that unit's selection on its own SM while the other SMs keep streaming.  Work items are (unit, 64-page chunk),
// handed out by a global counter in order of decreasing pool length, so the long selections start first and the tail
// of the kernel holds only the short ones.
//
// A CTA = 16 consumer warps + 1 producer warp (+ 15 warps that only work in selections).  A K page (16 rows, 4 KiB at d = 128) is one 1-D bulk async copy
// (cp.async.bulk, the TMA engine; SASS UBLKCP) into a 32-stage shared-memory ring tracked by mbarriers; the 32 lanes of
// the producer warp issue 32 copies with one pass over the instruction stream.  Consumers read MMA fragments by 16-byte
// LDS (layout of score_mma_kernel), one mma.sync m16n8k16 tile per page, write fp32 logits and the chunk's softmax
// statistics.  The ring's shared memory doubles as the probability slice of a selection: the role switch happens at a
// phase boundary, when every page this CTA has claimed is consumed.
#pragma once
#include "common.cuh"
#include "fast_kernels.cuh"
#include "score_tma.cuh"
#include "select_kernel.cuh"

namespace hardkv {

constexpr int SS_THREADS = 1024;
constexpr int SS_NCW = 16;                 // consumer warps 0..15; warp 16 produces; the rest only take part in selections
constexpr int SS_STAGES = 32;              // pages in flight per SM.  MUST be a multiple of SS_NCW: page n goes to warp
                                           // n % SS_NCW and stage n % SS_STAGES, so the successive users of a stage are the
                                           // same warp -- a parity wait cannot tell "two phases ahead" from "done"
static_assert(SS_STAGES % SS_NCW == 0, "successive users of a ring stage must be the same consumer warp");
constexpr int SS_Q = 4;                    // item descriptors the producer may run ahead
constexpr int SS_PENDING = 8;              // units waiting for their selection on this CTA (<= SS_Q + 2 by construction)
constexpr int SS_MAX_UNITS = 2048;

struct SsItem { int unit, chunk, pa, np; };   // np < 0: end of phase (np == -2: no work left)

struct SsControl {
  uint64_t full[SS_STAGES], empty[SS_STAGES], dfull[SS_Q], dempty[SS_Q];
  SsItem item[SS_Q];
  int pending[SS_PENDING];
  volatile int n_pending;
  int nitems;
  int last_phase;                          // written by the producer with an end-of-phase descriptor: no work is left
  float st[2][SS_NCW][8][2];
};

// mbarrier wait with a watchdog: a protocol error must end in a finished launch with *err_flag set (>= 100: which
// wait gave up), never in a kernel that spins forever on a shared GPU.  Once the flag is up every wait of every CTA
// returns at once, so all loops run out.  ~2^26 failed polls is seconds; a healthy wait takes microseconds.
__device__ __forceinline__ void ss_wait(uint64_t *bar, uint32_t parity, int code, int32_t *err_flag) {
  uint32_t done = 0;
  for (uint32_t polls = 1;; ++polls) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (done) return;
    if ((polls & 1023u) == 0) {
      if (*reinterpret_cast<volatile int32_t *>(err_flag) >= 100) return;
      if (polls > (1u << 26)) { atomicCAS(err_flag, 0, code); return; }
    }
  }
}

__device__ __forceinline__ void consumers_bar_sync() { asm volatile("bar.sync 1, %0;" ::"n"(SS_NCW * 32) : "memory"); }

// Dynamic shared memory: [ring / probability slice (aliased)] | SelShared | SsControl | order[units] | first[units + 1]
// | nchunks[units] | lo[B] | hi[B]
__host__ __device__ inline size_t score_select_buf_bytes(int d, int slice_cap) {
  const size_t ring = (size_t)SS_STAGES * PAGE * d * 2, slice = (size_t)slice_cap * 4;
  return ((ring > slice ? ring : slice) + 127) & ~(size_t)127;
}
__host__ __device__ inline size_t score_select_smem(int d, int slice_cap, int units, int B) {
  return score_select_buf_bytes(d, slice_cap) + ((sizeof(SelShared) + 127) & ~(size_t)127) +
         ((sizeof(SsControl) + 127) & ~(size_t)127) + (size_t)(3 * units + 1 + 2 * B) * 4 + 128;
}

template <int D, int GMAX>
__global__ void __launch_bounds__(SS_THREADS, 1) score_select_kernel(Params P, const void *q_, float p) {
  pdl_wait_then_trigger();
  KernelClock kclock(P);
  constexpr int NCH = D / 32;                 // 64-byte chunks per row
  constexpr int ROWB = D * 2, PAGEB = PAGE * ROWB;
  constexpr int SPC = SCORE_PAGES_PER_CTA;
  extern __shared__ __align__(128) unsigned char ss_smem[];
  const int units = P.B * P.Hkv;
  unsigned char *ring = ss_smem;
  size_t off = score_select_buf_bytes(D, P.ss_slice_cap);
  SelShared &sh = *reinterpret_cast<SelShared *>(ss_smem + off);
  off += (sizeof(SelShared) + 127) & ~(size_t)127;
  SsControl &ct = *reinterpret_cast<SsControl *>(ss_smem + off);
  off += (sizeof(SsControl) + 127) & ~(size_t)127;
  int *s_order = reinterpret_cast<int *>(ss_smem + off);   // units by decreasing pool length
  int *s_first = s_order + units;                          // [units + 1] first item of the i-th unit of that order
  int *s_nch = s_first + units + 1;                        // [units] chunks of a unit (by unit id)
  int *s_lo = s_nch + units, *s_hi = s_lo + P.B;           // pool bounds per sequence
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  // ---- the item list: every CTA rebuilds it from ctx_len / c_lo (a few hundred integer operations) ---------------
  for (int b = tid; b < P.B; b += SS_THREADS) {
    int n, lo, hi;
    pool_bounds(P, b, n, lo, hi);
    s_lo[b] = lo; s_hi[b] = hi;
  }
  if (tid == 0) {
    for (int s = 0; s < SS_STAGES; ++s) { mbar_init(&ct.full[s], 1); mbar_init(&ct.empty[s], 1); }
    for (int s = 0; s < SS_Q; ++s) { mbar_init(&ct.dfull[s], 1); mbar_init(&ct.dempty[s], 1); }
    ct.n_pending = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  for (int u = tid; u < units; u += SS_THREADS) {
    const int lo = s_lo[u / P.Hkv], hi = s_hi[u / P.Hkv];
    s_nch[u] = hi > lo ? ((hi - 1) >> 4) / SPC - (lo >> 4) / SPC + 1 : 0;
  }
  __syncthreads();
  for (int u = tid; u < units; u += SS_THREADS) {   // rank by (length desc, unit asc): O(units) compares per thread
    const int len = s_hi[u / P.Hkv] - s_lo[u / P.Hkv];
    int r = 0;
    for (int v = 0; v < units; ++v) {
      const int lv = s_hi[v / P.Hkv] - s_lo[v / P.Hkv];
      r += (lv > len) || (lv == len && v < u);
    }
    s_order[r] = u;
  }
  __syncthreads();
  if (warp == 0) {   // exclusive prefix sum of the chunk counts in that order
    int run = 0;
    for (int i0 = 0; i0 < units; i0 += 32) {
      const int i = i0 + lane;
      const int cnt = i < units ? s_nch[s_order[i]] : 0;
      int inc = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      if (i < units) s_first[i] = run + inc - cnt;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) { s_first[units] = run; ct.nitems = run; }
  }
  __syncthreads();
  const int nitems = ct.nitems;
  // units with an empty pool have no chunk and therefore no last-chunk owner: their (trivial) selection -- count 0, pads,
  // an empty table and mask -- is dealt out round-robin before the scan starts
  for (int u = blockIdx.x; u < units; u += gridDim.x) {
    if (s_nch[u] == 0) {
      select_unit<2, GMAX, SS_THREADS, false, true>(P, p, u, reinterpret_cast<uint32_t *>(ring), sh);
      __syncthreads();
    }
  }
  const char *kpool = reinterpret_cast<const char *>(P.st.k_pool);
  int nbase = 0;      // pages this CTA has streamed so far (the same count in every thread)
  int kseq = 0;       // descriptors this CTA has passed so far (the same count in every thread)

  for (;;) {
    // =========================== phase S: stream K pages ===========================================================
    if (warp == SS_NCW) {
      // ---- producer: claims items, publishes their descriptors, keeps the ring full ----
      for (;;) {
        int it = 0x7fffffff;
        // a finished unit is waiting for this CTA: end the phase (one lane reads, so the branch is warp-uniform)
        const bool stop = __shfl_sync(0xffffffffu, ct.n_pending, 0) > 0;
        if (!stop) {
          if (lane == 0) it = atomicAdd(P.ss_next, 1);
          it = __shfl_sync(0xffffffffu, it, 0);
        }
        SsItem d;
        if (stop || it >= nitems) {
          d.unit = -1; d.chunk = 0; d.pa = 0; d.np = (stop ? -1 : -2);
          if (!stop && it == nitems + (int)gridDim.x - 1 && lane == 0) *P.ss_next = 0;   // the very last claim re-arms
        } else {
          int il = 0, ih = units - 1;                // largest i with first[i] <= it
          while (il < ih) {
            const int mid = (il + ih + 1) >> 1;
            if (s_first[mid] <= it) il = mid; else ih = mid - 1;
          }
          d.unit = s_order[il];
          const int b = d.unit / P.Hkv, lo = s_lo[b], hi = s_hi[b];
          const int first_page = lo >> 4, last_page = (hi - 1) >> 4;
          d.chunk = first_page / SPC + (it - s_first[il]);
          d.pa = max(first_page, d.chunk * SPC);
          d.np = min(last_page, d.chunk * SPC + SPC - 1) - d.pa + 1;
        }
        const int slot = kseq % SS_Q;
        if (lane == 0) {
          ss_wait(&ct.dempty[slot], ((kseq / SS_Q) & 1) ^ 1, 101, P.st.err_flag);
          ct.item[slot] = d;
          mbar_arrive(&ct.dfull[slot]);
        }
        __syncwarp();
        ++kseq;
        if (d.np < 0) {
          if (lane == 0) ct.last_phase = d.np == -2;
          break;
        }
        const int32_t *tab = P.st.base_table + (size_t)d.unit * P.ppu;
        for (int j0 = 0; j0 < d.np; j0 += 32) {      // lane j issues the copy of page j0 + j: 32 copies per pass
          const int j = j0 + lane;
          if (j < d.np) {
            const int page = __ldg(tab + d.pa + j);
            const int n = nbase + j, s = n % SS_STAGES, k = n / SS_STAGES;
            ss_wait(&ct.empty[s], (k & 1) ^ 1, 102, P.st.err_flag);    // the consumer of the stage's previous page has read it
            mbar_expect_tx(&ct.full[s], PAGEB);
            bulk_g2s(ring + (size_t)s * PAGEB, kpool + (size_t)page * PAGEB, PAGEB, &ct.full[s]);
          }
          __syncwarp();
        }
        nbase += d.np;
      }
    } else if (warp < SS_NCW) {
      // ---- consumers: warp w takes the pages n = w (mod SS_NCW) of this CTA's page sequence ----
      const int gid = lane >> 2, tig = lane & 3;
      const int G = P.G;
      const int h0 = 2 * tig, h1 = 2 * tig + 1;
      for (;;) {
        const int slot = kseq % SS_Q;
        ss_wait(&ct.dfull[slot], (kseq / SS_Q) & 1, 103, P.st.err_flag);
        const SsItem d = ct.item[slot];
        if (d.np < 0) {
          consumers_bar_sync();                       // every consumer has read the descriptor
          if (tid == 0) mbar_arrive(&ct.dempty[slot]);
          ++kseq;
          break;
        }
        const int unit = d.unit, b = unit / P.Hkv, h = unit % P.Hkv;
        const int lo = s_lo[b], hi = s_hi[b];
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
        const float c2 = P.sm_scale * 1.4426950408889634f / P.st.temperature[unit];  // logit -> base-2 exponent of z/T
        float m0 = -INFINITY, s0 = 0.f, m1 = -INFINITY, s1 = 0.f;
        int j = (warp - nbase % SS_NCW + SS_NCW) % SS_NCW;
        for (; j < d.np; j += SS_NCW) {
          const int n = nbase + j, s = n % SS_STAGES, k = n / SS_STAGES;
          const unsigned char *src = ring + (size_t)s * PAGEB + gid * ROWB + tig * 16;
          ss_wait(&ct.full[s], k & 1, 104, P.st.err_flag);              // the page has landed
          float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int c = 0; c < NCH; ++c) {
            const uint4 ka = lds128(src + c * 64), kb = lds128(src + 8 * ROWB + c * 64);
            mma_bf16_16816(acc, ka.x, kb.x, ka.y, kb.y, qv[c].x, qv[c].y);
            mma_bf16_16816(acc, ka.z, kb.z, ka.w, kb.w, qv[c].z, qv[c].w);
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(&ct.empty[s]);   // fragments are consumed: hand the stage back
          const int ta = (d.pa + j) * PAGE + gid, tb = ta + 8;
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
        const int par = kseq & 1;                     // double-buffered: one barrier per item
        if (gid == 0) {
          ct.st[par][warp][h0][0] = m0; ct.st[par][warp][h0][1] = s0;
          ct.st[par][warp][h1][0] = m1; ct.st[par][warp][h1][1] = s1;
        }
        consumers_bar_sync();                         // orders every consumer's logit stores before warp 0's fence below
        if (warp == 0) {
          if (lane < 8) {
            const int g = lane;
            float m = -INFINITY, sacc = 0.f;
            if (g < G) {
              for (int w = 0; w < SS_NCW; ++w) m = fmaxf(m, ct.st[par][w][g][0]);
              for (int w = 0; w < SS_NCW; ++w) {
                const float mw = ct.st[par][w][g][0];
                if (mw != -INFINITY) sacc += ct.st[par][w][g][1] * fast_exp2(mw - m);
              }
            }
            P.score_stats[((size_t)unit * P.score_chunks + d.chunk) * 8 + g] = make_float2(m, sacc);
          }
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(&ct.dempty[slot]);            // the descriptor slot is free (every consumer passed the barrier)
            // release: the barrier above made every consumer's stores of this chunk (and the syncwarp the statistics)
            // happen before this fence, which is cumulative -- the pattern of a cooperative grid barrier
            __threadfence();
            int ticket = atomicAdd(P.ss_arrive + unit, 1);
            if (ticket == s_nch[unit] - 1) {          // this CTA retired the unit's last chunk: it selects for it
              const int np_ = ct.n_pending;
              if (np_ < SS_PENDING) {
                ct.pending[np_] = unit;
                __threadfence_block();
                ct.n_pending = np_ + 1;
              } else {
                atomicExch(P.st.err_flag, 3);         // cannot happen (<= SS_Q + 2 by construction): flag, never overrun
              }
            }
          }
        }
        nbase += d.np;
        ++kseq;
      }
    }
    __syncthreads();   // phase boundary: every page this CTA claimed is consumed, the ring is idle
    const bool final_phase = ct.last_phase != 0;
    // =========================== phase T: selections this CTA owes =================================================
    const int npend = ct.n_pending;
    if (npend > 0) {
      __threadfence();                                // acquire side of the tickets: other CTAs' logits / statistics
      for (int i = 0; i < npend; ++i) {
        const int unit = ct.pending[i];
        select_unit<2, GMAX, SS_THREADS, false, true>(P, p, unit, reinterpret_cast<uint32_t *>(ring), sh);
        if (tid == 0) P.ss_arrive[unit] = 0;          // re-arm for the next launch / graph replay
        __syncthreads();
      }
      if (tid == 0) ct.n_pending = 0;
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes of the slice before the next bulk copies
      __syncthreads();
    }
    if (final_phase) break;
  }
}

}  // namespace hardkv
