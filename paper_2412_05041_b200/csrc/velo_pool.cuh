// velo_pool.cuh — persistent-CTA infrastructure shared by the three pipeline kernels of libvelo
// (velo_sort.cu, velo_track.cu, velo_fit.cu; sm_100a).
//
// One persistent CTA per SM owns the SM's shared memory as a pool of 64 units. The CTA is cut into
// teams of G threads (a warp, or a few warps behind a named barrier); a team's leader takes the
// next event from a global ticket and allocates from the pool exactly what that event needs in
// this stage (events span 0 ... ~6 k hits at mu = 5: a fixed slot per event would waste more than
// half of the SM). Also here: the team barrier and scans, and the 1-D TMA bulk copy (cp.async.bulk +
// mbarrier) that feeds shared memory.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace velo {

constexpr uint32_t kUnitBytes = 3456;   // pool allocation unit: at most 64 of them (one bitmap word)
constexpr uint32_t kPoolUnitsMax = 64;  //   = 216 KB of pool; + the control block <= 227 KB per CTA

struct PoolCtl {
  unsigned long long bitmap;            // 1 = unit in use
  uint32_t alloc_next, alloc_serving;   // FIFO ticket lock around the allocator: no starvation
  uint32_t units;                       // units in this CTA's pool (set at kernel start)
  uint32_t pad;
};

// ---- stage windows for `bench.py --timeline` (a -DVELO_TIMELINE build only) -----------------------
// phase_clk[2k] = ~(earliest start) and phase_clk[2k + 1] = latest end of stage k's CTAs, in ns of
// the GPU's global timer; zeroed by launch_reconstruct. Compiled out of the product library.
#ifdef VELO_TIMELINE
__device__ __forceinline__ unsigned long long velo_globaltimer() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
#define VELO_STAGE_BEGIN(clk, k) do { if (threadIdx.x == 0) atomicMax(&(clk)[2 * (k)], ~velo_globaltimer()); } while (0)
#define VELO_STAGE_END(clk, k) do { __syncthreads(); if (threadIdx.x == 0) atomicMax(&(clk)[2 * (k) + 1], velo_globaltimer()); } while (0)
#else
#define VELO_STAGE_BEGIN(clk, k) do { } while (0)
#define VELO_STAGE_END(clk, k) do { } while (0)
#endif

// ---- team barrier: G threads; G == 32 is a warp -------------------------------------------------
template <int G>
__device__ __forceinline__ void team_sync(uint32_t team) {
  if constexpr (G == 32) __syncwarp();
  else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(G) : "memory");
}

// ---- exclusive scan of a predicate over the team (ballot inside a warp, warp totals in shared) --
// wsum: 2 * (G / 32) words of team-private shared memory; parity toggles per call, so that one
// barrier per call suffices. Every thread of the team must call it.
template <int G>
__device__ __forceinline__ uint32_t team_scan_pred(bool p, uint32_t* wsum, uint32_t team, uint32_t& parity,
                                                   uint32_t* total) {
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t b = __ballot_sync(0xffffffffu, p);
  const uint32_t pre = (uint32_t)__popc(b & ((1u << lane) - 1u));
  if constexpr (G == 32) {
    *total = (uint32_t)__popc(b);
    return pre;
  } else {
    constexpr uint32_t W = G / 32;
    const uint32_t wid = (threadIdx.x % G) >> 5;
    uint32_t* ws = wsum + (parity & 1u) * W;
    parity ^= 1u;
    if (lane == 0) ws[wid] = (uint32_t)__popc(b);
    team_sync<G>(team);
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (uint32_t k = 0; k < W; ++k) { const uint32_t s = ws[k]; if (k < wid) base += s; tot += s; }
    *total = tot;
    return base + pre;
  }
}

// Exclusive scan of two u32 values per thread over the team (wsum: 4 * (G / 32) words).
template <int G>
__device__ __forceinline__ uint32_t team_scan2(uint32_t v, uint32_t v2, uint32_t* wsum, uint32_t team, uint32_t& parity,
                                               uint32_t* total, uint32_t* prefix2, uint32_t* total2) {
  constexpr uint32_t W = G / 32;
  const uint32_t lane = threadIdx.x & 31u, wid = (threadIdx.x % G) >> 5;
  uint32_t inc = v, inc2 = v2;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d), o2 = __shfl_up_sync(0xffffffffu, inc2, d);
    if (lane >= (uint32_t)d) { inc += o; inc2 += o2; }
  }
  if constexpr (G == 32) {
    *total = __shfl_sync(0xffffffffu, inc, 31); *total2 = __shfl_sync(0xffffffffu, inc2, 31);
    *prefix2 = inc2 - v2;
    return inc - v;
  } else {
    uint32_t* ws = wsum + (parity & 1u) * 2u * W;
    parity ^= 1u;
    if (lane == 31) { ws[wid] = inc; ws[W + wid] = inc2; }
    team_sync<G>(team);
    uint32_t base = 0, base2 = 0, tot = 0, tot2 = 0;
#pragma unroll
    for (uint32_t k = 0; k < W; ++k) {
      const uint32_t s = ws[k], s2 = ws[W + k];
      if (k < wid) { base += s; base2 += s2; }
      tot += s; tot2 += s2;
    }
    *total = tot; *total2 = tot2; *prefix2 = base2 + inc2 - v2;
    return base + inc - v;
  }
}

// ---- pool allocator (called by a team's leader thread only) ------------------------------------
__device__ __forceinline__ uint32_t pool_alloc(PoolCtl& ctl, uint32_t units) {
  const uint32_t my = atomicAdd(&ctl.alloc_next, 1u);
  volatile uint32_t* serving = &ctl.alloc_serving;
  while (*serving != my) __nanosleep(400);
  volatile unsigned long long* bm = &ctl.bitmap;
  const uint32_t pu = ctl.units;
  const unsigned long long all = pu >= 64u ? ~0ull : (1ull << pu) - 1ull;
  uint32_t first;
  unsigned long long seen = ~0ull;
  for (;;) {
    const unsigned long long used = *bm;
    if (used == seen) { __nanosleep(400); continue; }   // nothing was freed since the last failed try
    unsigned long long r = ~used & all;          // bit p: unit p free
    for (uint32_t i = 1; i < units && r; ++i) r &= (r >> 1);   // bit p: units p .. p+i free
    if (r) {
      first = (uint32_t)__ffsll((long long)r) - 1u;
      const unsigned long long claim = ((units >= 64u ? ~0ull : ((1ull << units) - 1ull)) << first);
      if (atomicCAS(&ctl.bitmap, used, used | claim) == used) break;
    } else {
      seen = used;
    }
  }
  __threadfence_block();
  *serving = my + 1u;
  return first;
}
__device__ __forceinline__ void pool_free(PoolCtl& ctl, uint32_t first, uint32_t units) {
  const unsigned long long claim = ((units >= 64u ? ~0ull : ((1ull << units) - 1ull)) << first);
  atomicAnd(&ctl.bitmap, ~claim);
}

// ---- mbarrier + 1-D TMA bulk copy (global -> shared::cta), PTX ISA 8.x --------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// dst, src and bytes are multiples of 16; completes `bytes` of transaction count on `bar`.
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

}  // namespace velo
