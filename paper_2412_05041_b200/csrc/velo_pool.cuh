// velo_pool.cuh — persistent-CTA infrastructure shared by the three pipeline kernels of libvelo
// (velo_sort.cu, velo_track.cu, velo_fit.cu; sm_100a).
//
// One persistent CTA per SM owns the SM's shared memory as a pool of 128 units. The CTA is cut into
// teams of G threads (a warp, or a few warps behind a named barrier); a team's leader takes the
// next event from a global ticket and allocates from the pool exactly what that event needs in
// this stage (events span 0 ... ~6 k hits at mu = 5: a fixed slot per event would waste more than
// half of the SM). Also here: the team barrier and scans, and the 1-D TMA bulk copy (cp.async.bulk +
// mbarrier) that feeds shared memory.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace velo {

constexpr uint32_t kUnitBytes = 1728;    // pool allocation unit: at most 128 of them (two bitmap words)
constexpr uint32_t kPoolUnitsMax = 128;  //   = 216 KB of pool; + the control block <= 227 KB per CTA

struct PoolCtl {
  unsigned long long bitmap[2];         // 1 = unit in use; unit u is bit u & 63 of word u >> 6
  uint32_t alloc_next, alloc_serving;   // FIFO ticket lock around the allocator: no starvation
  uint32_t units;                       // units in this CTA's pool (set at kernel start)
  uint32_t pad;
};
__device__ __forceinline__ void pool_init(PoolCtl& ctl, uint32_t units) {
  ctl.bitmap[0] = 0ull; ctl.bitmap[1] = 0ull; ctl.alloc_next = 0; ctl.alloc_serving = 0; ctl.units = units;
}

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
// Phase clocks: the team leader adds the SM clocks since its previous mark to phase_clk[i] (sort 8..15,
// track 16..27, fit 32..43; slot i + 0 of each range counts events).
#define VELO_PH_START(ts) do { if (tid == 0) (ts).ph_last = clock64(); } while (0)
#define VELO_PH(clk, ts, i) do { if (tid == 0) { const unsigned long long now_ = clock64(); atomicAdd(&(clk)[i], now_ - (ts).ph_last); (ts).ph_last = now_; } } while (0)
#define VELO_PH_COUNT(clk, i, v) do { if (tid == 0) atomicAdd(&(clk)[i], (unsigned long long)(v)); } while (0)
#else
#define VELO_PH_START(ts) do { } while (0)
#define VELO_PH(clk, ts, i) do { } while (0)
#define VELO_PH_COUNT(clk, i, v) do { } while (0)
#define VELO_STAGE_BEGIN(clk, k) do { } while (0)
#define VELO_STAGE_END(clk, k) do { } while (0)
#endif

// Asks L2 for the line at p (no register, no wait): what a thread will read a few microseconds later.
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

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
// First fit over a 128-bit occupancy map. Allocations are serialised by the FIFO ticket, so only
// the ticket holder ever sets bits; frees (any leader, any time) only clear bits. The holder may
// therefore read a stale map, which errs on the safe side, and no compare-and-swap is needed.
struct Bits128 { unsigned long long lo, hi; };
__device__ __forceinline__ Bits128 shr128(Bits128 v, uint32_t s) {     // 0 < s < 128
  Bits128 r;
  if (s >= 64u) { r.lo = v.hi >> (s - 64u); r.hi = 0ull; }
  else { r.lo = (v.lo >> s) | (v.hi << (64u - s)); r.hi = v.hi >> s; }
  return r;
}
__device__ __forceinline__ Bits128 ones128(uint32_t first, uint32_t count) {   // bits first .. first+count-1, count >= 1
  const uint32_t end = first + count;                                          // <= 128
  Bits128 r;
  const unsigned long long below_end_lo = end >= 64u ? ~0ull : ((1ull << end) - 1ull);
  const unsigned long long below_first_lo = first >= 64u ? ~0ull : ((1ull << first) - 1ull);
  r.lo = below_end_lo & ~below_first_lo;
  const unsigned long long below_end_hi = end >= 128u ? ~0ull : (end > 64u ? ((1ull << (end - 64u)) - 1ull) : 0ull);
  const unsigned long long below_first_hi = first > 64u ? ((1ull << (first - 64u)) - 1ull) : 0ull;
  r.hi = below_end_hi & ~below_first_hi;
  return r;
}
__device__ __forceinline__ uint32_t pool_alloc(PoolCtl& ctl, uint32_t units) {
  const uint32_t my = atomicAdd(&ctl.alloc_next, 1u);
  volatile uint32_t* serving = &ctl.alloc_serving;
  while (*serving != my) __nanosleep(1000);
  volatile unsigned long long* bm = ctl.bitmap;
  const Bits128 all = ones128(0u, ctl.units);
  uint32_t first;
  Bits128 seen{~0ull, ~0ull};
  for (;;) {
    const Bits128 used{bm[0], bm[1]};
    if (used.lo == seen.lo && used.hi == seen.hi) { __nanosleep(500); continue; }   // nothing was freed since the last failed try
    Bits128 r{~used.lo & all.lo, ~used.hi & all.hi};   // bit p: unit p free
    // after the loop, bit p: units p .. p+units-1 free (run length doubles per trip)
    for (uint32_t len = 1; len < units && (r.lo | r.hi); ) {
      const uint32_t sh = min(len, units - len);
      const Bits128 t = shr128(r, sh);
      r.lo &= t.lo; r.hi &= t.hi;
      len += sh;
    }
    if (r.lo | r.hi) {
      first = r.lo ? (uint32_t)__ffsll((long long)r.lo) - 1u : 63u + (uint32_t)__ffsll((long long)r.hi);
      const Bits128 claim = ones128(first, units);
      if (claim.lo) atomicOr(&ctl.bitmap[0], claim.lo);
      if (claim.hi) atomicOr(&ctl.bitmap[1], claim.hi);
      break;
    }
    seen = used;
  }
  __threadfence_block();
  *serving = my + 1u;
  return first;
}
__device__ __forceinline__ void pool_free(PoolCtl& ctl, uint32_t first, uint32_t units) {
  const Bits128 claim = ones128(first, units);
  if (claim.lo) atomicAnd(&ctl.bitmap[0], ~claim.lo);
  if (claim.hi) atomicAnd(&ctl.bitmap[1], ~claim.hi);
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
