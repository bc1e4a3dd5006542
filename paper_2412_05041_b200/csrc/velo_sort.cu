// velo_sort.cu — stage 1 of the pipeline: S0 decode + S1 per-module phi sort (sm_100a).
//
// A streaming kernel: every event is read once from the caller's SoA planes (128-bit loads on the
// aligned interior), gets its phi16 (O-1) and its (module, phi16, original index) order (O-2) in
// shared memory, and leaves as one contiguous, 16-byte aligned block of sorted 16-byte hit records
// in global scratch, which stage 2 pulls into shared memory module by module with 1-D TMA copies:
//
//   rec16[h] = { x, y, (phi16 + 32768) << 16 | start(m+1), start(m-1) << 16 | start(m-2) }
//
// start(m') = position inside module m' of its first hit with phi >= phi(h) - W (W = the wider of
// the two O-3 windows), i.e. where a window scan of module m' around h begins: stage 2 then never
// searches, it scans from `start` until the window test fails (a window across +-pi has a second
// run that starts at position 0). Also written: sorted (x, y) and original indices for stage 3,
// the module offsets, and the event's state (ready / deferred to the general kernel / bad input).
//
// Shared memory is held only for the sort (17 bytes per hit + the bucket table). Step semantics:
// SURVEY.md §8(c) O-1, O-2, O-3.
#include "velo_device.cuh"
#include "velo_internal.h"
#include "velo_pool.cuh"

namespace velo {

namespace {

constexpr uint32_t kMaxBinSlot = 2047;      // slot inside a phi bucket is stashed in 11 bits

template <int G>
struct SortTeam {
  uint32_t wsum[4 * (G / 32)];
  uint32_t event, n, o0, ol;         // event index, hits, first hit (absolute), first hit relative to the batch
  uint32_t units, first_unit, pool_off;
  uint32_t skip;                     // nothing to sort (empty / bad / deferred before the sort)
  uint32_t unpack;                   // packed input: decode the deferred event for the general kernel
  uint32_t trouble;                  // bit 0: defer to the general kernel, bit 31: bad input
  unsigned long long ph_last;        // phase clocks (-DVELO_TIMELINE builds)
};

template <int G, int kTeams>
struct SortCtl {
  PoolCtl pool;
  float module_z[VELO_MAX_MODULES];
  SortTeam<G> team[kTeams];
};

__device__ __forceinline__ uint32_t align16u(uint32_t v) { return (v + 15u) & ~15u; }

struct SortLayout { uint32_t xy, w, bins, stash, mod8, side, bytes; };
__device__ __forceinline__ SortLayout sort_layout(uint32_t n, uint32_t M, uint32_t bins_per_module = kBinsPerModule) {
  SortLayout L;
  uint32_t o = 0;
  L.xy = o; o += align16u(8u * n);
  L.w = o; o += align16u(4u * n);
  L.bins = o; o += align16u(2u * (M * bins_per_module + 2u));
  L.stash = o; o += align16u(4u * n);
  L.mod8 = o; o += align16u(n);
  L.side = o; o += align16u(4u * ((n + 31u) >> 5));   // two-plane geometries: one bit per ORIGINAL index
  L.bytes = o;
  return L;
}

__device__ __forceinline__ void set_status(uint32_t* counters, int code) {
  atomicCAS(&counters[kCtrStatus], 0u, (uint32_t)code);   // first error wins
}

template <int G>
__device__ void sort_fetch(const KernelArgs& a, PoolCtl& pool, SortTeam<G>& ts) {
  const uint32_t e = atomicAdd(&a.ws.counters[kCtrSortTicket], 1u);
  ts.event = e; ts.units = 0; ts.skip = 1; ts.n = 0; ts.trouble = 0; ts.unpack = 0;
  if (e >= a.n_events) return;
  const uint32_t base = a.event_offsets[0];
  const uint32_t o0 = a.event_offsets[e], o1 = a.event_offsets[e + 1];
  atomicAdd(&a.ws.size_hist[size_class(o0, o1)], 1u);    // events per size class, for velo_order_kernel
  EvInfo info{0u, kEvEmpty, 0u, 0u};
  // every event must stay inside the batch, [base, base + n_hits]: nothing is read out of bounds
  if (o1 < o0 || o0 < base || o1 - base > a.n_hits || o1 - o0 > VELO_MAX_EVENT_HITS) {
    set_status(a.ws.counters, VELO_ERR_INPUT);
    info.state = kEvBad; a.ws.ev_info[e] = info;
    return;
  }
  const uint32_t n = o1 - o0;
  info.n = n;
  if (n == 0) { a.ws.ev_info[e] = info; return; }
  const SortLayout L = sort_layout(n, a.n_modules);
  const uint32_t units = (L.bytes + kUnitBytes - 1u) / kUnitBytes;
  if (n > a.team_max_hits && a.big_path) {       // too large for an SM's pool: the one-event-per-CTA pipeline
    info.state = kEvBig; a.ws.ev_info[e] = info;
    a.ws.big_list[atomicAdd(&a.ws.counters[kCtrBigN], 1u)] = e;
    return;
  }
  if (n > a.team_max_hits || units > pool.units || fit_smem_bound(n) > pool.units * kUnitBytes) {
    info.state = kEvDeferred; a.ws.ev_info[e] = info;
    a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
    ts.unpack = a.pixel != nullptr;
    return;
  }
  const uint32_t first = pool_alloc(pool, units);
  ts.n = n; ts.o0 = o0; ts.ol = o0 - base; ts.units = units; ts.first_unit = first; ts.pool_off = first * kUnitBytes;
  ts.skip = 0;
}

// kShift: phi units per bucket = 1 << kShift (the one-event-per-CTA form uses finer buckets: its events
// have tens of hits per 1024-unit bucket, and the rank inside a bucket is a loop over the bucket).
template <int G, int kShift = kBinShift>
__device__ void sort_event(const KernelArgs& a, const float* mz, SortTeam<G>& ts, unsigned char* blk, uint32_t team,
                           uint32_t tid, uint32_t& parity, uint32_t done_state = kEvReady) {
  constexpr uint32_t kBinsPerModule = 65536u >> kShift;
  constexpr uint32_t kBinShift = kShift;
  const uint32_t M = a.n_modules, nbins = M * kBinsPerModule;
  const uint32_t e = ts.event, n = ts.n;
  const SortLayout L = sort_layout(n, M, kBinsPerModule);
  float2* xyo = (float2*)(blk + L.xy);          // (x, y) by ORIGINAL index
  uint32_t* w = (uint32_t*)(blk + L.w);
  uint32_t* binsw = (uint32_t*)(blk + L.bins);
  uint16_t* bo = (uint16_t*)binsw;
  uint32_t* stash = (uint32_t*)(blk + L.stash);
  uint8_t* mod8 = blk + L.mod8;                 // module by SORTED position (bit 7: the hit's plane, two-plane geometries)
  uint32_t* sideb = (uint32_t*)(blk + L.side);
  const float* mzb = a.module_z_b;              // (constant bank: read once per hit, two-plane geometries only)
  const bool two_plane = a.two_plane != 0u;
  const size_t g0 = (size_t)(ts.o0 - a.hit_base);
  const float* gx = a.x + g0; const float* gy = a.y + g0; const float* gz = a.z + g0;
  const uint8_t* gm = a.module + g0;
  const uint32_t* gp = a.pixel + g0;

  // Tickets go out in event order and events lie one behind the other in the input planes: what this team
  // asks L2 for now, its own length of input kPrefetchAhead hits further on, is what the teams of the events
  // a few hundred tickets later will read (every line of the batch is asked for once, by some team).
  {
    constexpr uint32_t kPrefetchAhead = 1u << 20;      // hits: about the events in flight on the GPU at mu = 5
    const uint32_t end = a.event_offsets[0] + a.n_hits - a.hit_base;   // first hit index (relative to the planes) behind the batch
    const uint32_t p0 = ((uint32_t)g0 + kPrefetchAhead) & ~31u;
    const uint32_t p1 = min((uint32_t)g0 + n + kPrefetchAhead, end);
    if (a.pixel) { for (uint32_t i = p0 + 32u * tid; i < p1; i += 32u * G) prefetch_l2(a.pixel + i); }
    else {
      for (uint32_t i = p0 + 32u * tid; i < p1; i += 32u * G) { prefetch_l2(a.x + i); prefetch_l2(a.y + i); prefetch_l2(a.z + i); }
      for (uint32_t i = (p0 & ~127u) + 128u * tid; i < p1; i += 128u * G) prefetch_l2(a.module + i);
    }
  }
  // ---- S0 decode: phi16 (O-1), bucket histogram; the plane check of the pipeline path -------------
  const uint32_t nwords = nbins / 2u;
  for (uint32_t b = tid; b <= nwords; b += G) binsw[b] = 0;
  if (two_plane) for (uint32_t b = tid; b < ((n + 31u) >> 5); b += G) sideb[b] = 0;
  team_sync<G>(team);
  {
    uint32_t trouble = 0;
    auto decode = [&](uint32_t i, float x, float y, float z, uint32_t m) {
      if (m >= M) { trouble |= 0x80000000u; return; }
      if (__float_as_uint(z) != __float_as_uint(mz[m])) {
        // L-1: the station's second sensor plane, else the event is the general kernel's
        if (two_plane && __float_as_uint(z) == __float_as_uint(mzb[m])) atomicOr(&sideb[i >> 5], 1u << (i & 31u));
        else trouble |= 1u;
      }
      const uint32_t pu = (uint32_t)(phi16(x, y) + 32768);
      const uint32_t bin = m * kBinsPerModule + (pu >> kBinShift);
      const uint32_t sh = (bin & 1u) * 16u;
      const uint32_t slot = (atomicAdd(&binsw[bin >> 1], 1u << sh) >> sh) & 0xffffu;
      if (slot > kMaxBinSlot) trouble |= 1u;
      stash[i] = (m << 27) | (pu << 11) | (slot & kMaxBinSlot);
      xyo[i] = make_float2(x, y);
    };
    if (a.pixel) {
      // F-1, F-2: packed pixel addresses, four per 128-bit load on the aligned interior; z is the
      // module's plane by construction
      auto decode_px = [&](uint32_t i, uint32_t wd) {
        uint32_t m; float x, y;
        pixel_decode(wd, a.pitch, a.half_shift_x, m, x, y);
        decode(i, x, y, m < M ? mz[m] : 0.0f, m);
      };
      uint32_t head = (4u - (uint32_t)(((uintptr_t)gp >> 2) & 3u)) & 3u;
      if (head > n) head = n;
      const uint32_t nq = (n - head) / 4u;
      for (uint32_t i = tid; i < head; i += G) decode_px(i, gp[i]);
      const uint4* vp = (const uint4*)(gp + head);
      for (uint32_t q = tid; q < nq; q += G) {
        const uint4 W4 = vp[q];
        const uint32_t i = head + 4u * q;
        decode_px(i, W4.x); decode_px(i + 1, W4.y); decode_px(i + 2, W4.z); decode_px(i + 3, W4.w);
      }
      for (uint32_t i = head + 4u * nq + tid; i < n; i += G) decode_px(i, gp[i]);
    } else {
    // 128-bit loads where the planes allow them. The three float planes and the byte plane are
    // indexed by the same hit index, so with the usual allocations they reach 16-byte (4-byte for
    // the modules) alignment after the same number of leading hits; otherwise everything is scalar.
    const uint32_t px = (uint32_t)(((uintptr_t)gx >> 2) & 3u), py = (uint32_t)(((uintptr_t)gy >> 2) & 3u),
                   pz = (uint32_t)(((uintptr_t)gz >> 2) & 3u), pm = (uint32_t)((uintptr_t)gm & 3u);
    const bool vec = (((uintptr_t)gx | (uintptr_t)gy | (uintptr_t)gz) & 3u) == 0 && px == py && px == pz &&
                     (((4u - px) & 3u) == ((4u - pm) & 3u));
    uint32_t head = vec ? ((4u - px) & 3u) : n;
    if (head > n) head = n;
    const uint32_t nq = (n - head) / 4u;
    for (uint32_t i = tid; i < head; i += G) decode(i, gx[i], gy[i], gz[i], gm[i]);
    {
      const float4* vx = (const float4*)(gx + head); const float4* vy = (const float4*)(gy + head);
      const float4* vz = (const float4*)(gz + head); const uint32_t* vm = (const uint32_t*)(gm + head);
      for (uint32_t q = tid; q < nq; q += G) {
        const float4 X = vx[q], Y = vy[q], Z = vz[q]; const uint32_t Mq = vm[q];
        const uint32_t i = head + 4u * q;
        decode(i, X.x, Y.x, Z.x, Mq & 0xffu);
        decode(i + 1, X.y, Y.y, Z.y, (Mq >> 8) & 0xffu);
        decode(i + 2, X.z, Y.z, Z.z, (Mq >> 16) & 0xffu);
        decode(i + 3, X.w, Y.w, Z.w, Mq >> 24);
      }
    }
    for (uint32_t i = head + 4u * nq + tid; i < n; i += G) decode(i, gx[i], gy[i], gz[i], gm[i]);
    }
    if (trouble) atomicOr(&ts.trouble, trouble);
  }
  team_sync<G>(team);
  VELO_PH(a.ws.phase_clk, ts, 10);
  if (ts.trouble) {
    if (tid == 0) {
      EvInfo info{n, kEvDeferred, 0u, 0u};
      if (ts.trouble & 0x80000000u) { set_status(a.ws.counters, VELO_ERR_INPUT); info.state = kEvBad; }
      else a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
      a.ws.ev_info[e] = info;
    }
    if (a.pixel && !(ts.trouble & 0x80000000u)) unpack_event<G>(a, e, tid);
    return;
  }
  // exclusive scan of the packed histogram -> bucket offsets; bo[nbins] = n
  {
    const uint32_t per = (nwords + G - 1) / G;
    const uint32_t w0 = min(tid * per, nwords), w1 = min(w0 + per, nwords);
    uint32_t s = 0;
    for (uint32_t k = w0; k < w1; ++k) { const uint32_t v = binsw[k]; s += (v & 0xffffu) + (v >> 16); }
    uint32_t tot, p2, t2;
    uint32_t run = team_scan2<G>(s, 0u, ts.wsum, team, parity, &tot, &p2, &t2);
    for (uint32_t k = w0; k < w1; ++k) {
      const uint32_t v = binsw[k], c0 = v & 0xffffu, c1 = v >> 16;
      binsw[k] = run | ((run + c0) << 16);
      run += c0 + c1;
    }
    if (tid == 0) bo[nbins] = (uint16_t)n;
  }
  team_sync<G>(team);
  VELO_PH(a.ws.phase_clk, ts, 11);
  // ---- S1 phi sort (O-2): group by bucket in w[], rank inside the bucket by (phi16, index), place --
  for (uint32_t i = tid; i < n; i += G) {
    const uint32_t st = stash[i], pu = (st >> 11) & 0xffffu;
    const uint32_t bin = (st >> 27) * kBinsPerModule + (pu >> kBinShift);
    w[(uint32_t)bo[bin] + (st & kMaxBinSlot)] = (pu << 16) | i;
  }
  team_sync<G>(team);
  for (uint32_t i = tid; i < n; i += G) {
    const uint32_t st = stash[i], pu = (st >> 11) & 0xffffu;
    const uint32_t bin = (st >> 27) * kBinsPerModule + (pu >> kBinShift);
    const uint32_t item = (pu << 16) | i;
    const uint32_t lo = bo[bin], hi = bo[bin + 1];
    uint32_t r = 0;                      // rank inside the bucket: at most kMaxBinSlot
    for (uint32_t j = lo; j < hi; ++j) r += (w[j] < item) ? 1u : 0u;
    stash[i] = (st & ~kMaxBinSlot) | r;
  }
  team_sync<G>(team);                    // every rank is known: w[] can take its final content
  VELO_PH(a.ws.phase_clk, ts, 12);
  for (uint32_t i = tid; i < n; i += G) {
    const uint32_t st = stash[i], pu = (st >> 11) & 0xffffu, m = st >> 27;
    const uint32_t r = (uint32_t)bo[m * kBinsPerModule + (pu >> kBinShift)] + (st & kMaxBinSlot);
    w[r] = (pu << 16) | i;
    mod8[r] = (uint8_t)(two_plane ? m | (((sideb[i >> 5] >> (i & 31u)) & 1u) << 7) : m);
  }
  team_sync<G>(team);
  VELO_PH(a.ws.phase_clk, ts, 13);
  // ---- window starts and the event's sorted block -------------------------------------------------
  const int Wseed = a.P.phi_window_seed, Wfwd = a.P.phi_window_fwd;
  const int W = Wseed > Wfwd ? Wseed : Wfwd;                 // >= 0 (the host clamps negative windows)
  const bool whole = 2 * (long long)W + 1 >= 65536;
  // position inside module mm of its first hit with unsigned phi >= lo
  auto start_in = [&](uint32_t mm, uint32_t lo) -> uint32_t {
    const uint16_t* bm = bo + mm * kBinsPerModule;
    uint32_t j0 = bm[lo >> kBinShift], j1 = bm[(lo >> kBinShift) + 1];
    while (j0 < j1) {                                        // binary search inside one phi bucket
      const uint32_t mid = (j0 + j1) >> 1;
      if ((w[mid] >> 16) < lo) j0 = mid + 1u; else j1 = mid;
    }
    return j0 - (uint32_t)bm[0];
  };
  const uint32_t sb = sorted_base(ts.ol, e);
  uint4* rec = a.ws.rec16 + sb;
  uint16_t* sorig = a.ws.sorig + sb;
  for (uint32_t h = tid; h < n; h += G) {
    const uint32_t item = w[h], pu = item >> 16, i = item & 0xffffu, m8 = mod8[h], m = m8 & 31u;
    const float2 p = xyo[i];
    uint32_t sp1 = 0, sm1 = 0, sm2 = 0;
    if (!whole) {
      const uint32_t lo = (pu - (uint32_t)W) & 0xffffu;
      if (m + 1u < M) sp1 = start_in(m + 1u, lo);
      if (m >= 1u) sm1 = start_in(m - 1u, lo);
      if (m >= 2u) sm2 = start_in(m - 2u, lo);
    }
    // two-plane geometries: bit 15 of the last word is the hit's plane (a module of a pipeline event has
    // fewer than 32768 hits, so start(m-2) leaves it free)
    rec[h] = make_uint4(__float_as_uint(p.x), __float_as_uint(p.y), (pu << 16) | sp1, (sm1 << 16) | sm2 | ((m8 >> 7) << 15));
    sorig[h] = (uint16_t)i;
  }
  // module offsets and the largest module
  uint16_t* mo = a.ws.mod_off + (size_t)e * kModOffStride;
  if (tid < 32) {
    const uint32_t lo = tid <= M ? (uint32_t)bo[tid * kBinsPerModule] : n;
    const uint32_t hi = tid < M ? (uint32_t)bo[(tid + 1u) * kBinsPerModule] : lo;
    uint32_t sz = hi - lo;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sz = max(sz, __shfl_xor_sync(0xffffffffu, sz, o));
    mo[tid] = (uint16_t)lo;
    if (tid == 0) { mo[32] = (uint16_t)n; mo[kModOffStride - 1] = (uint16_t)sz; }
  }
  if (tid == 0) a.ws.ev_info[e] = EvInfo{n, done_state, 0u, 0u};
  VELO_PH(a.ws.phase_clk, ts, 14);
}

// ---- the kernel: one CTA per SM, kTeams teams of G threads, events by ticket in event order -----
template <int G, int kTeams>
__global__ void __launch_bounds__(G * kTeams, 1) velo_sort_kernel(const KernelArgs a, const uint32_t pool_units) {
  extern __shared__ __align__(16) unsigned char smem[];
  using Ctl = SortCtl<G, kTeams>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  Ctl& ctl = *reinterpret_cast<Ctl*>(smem);
  unsigned char* pool = smem + kCtl;
  const uint32_t team = threadIdx.x / G, tid = threadIdx.x % G;
  if (threadIdx.x == 0) pool_init(ctl.pool, pool_units);
  if (threadIdx.x < VELO_MAX_MODULES) ctl.module_z[threadIdx.x] = a.module_z[threadIdx.x];
  __syncthreads();
  VELO_STAGE_BEGIN(a.ws.phase_clk, 0);
  SortTeam<G>& ts = ctl.team[team];
  uint32_t parity = 0;
  VELO_PH_START(ts);
  for (;;) {
    if (tid == 0) sort_fetch<G>(a, ctl.pool, ts);
    team_sync<G>(team);
    if (ts.event >= a.n_events) break;
    VELO_PH(a.ws.phase_clk, ts, 9);      // ticket, offsets, pool
    if (!ts.skip) sort_event<G>(a, ctl.module_z, ts, pool + ts.pool_off, team, tid, parity);
    else if (ts.unpack) unpack_event<G>(a, ts.event, tid);
    team_sync<G>(team);
    if (tid == 0 && ts.units) pool_free(ctl.pool, ts.first_unit, ts.units);
    VELO_PH(a.ws.phase_clk, ts, 15);
    VELO_PH_COUNT(a.ws.phase_clk, 8, 1);
  }
  VELO_STAGE_END(a.ws.phase_clk, 0);
}

// ---- the same stage for the events of ws.big_list: one CTA of G threads per event, the per-event
// arrays in the CTA's global slab (L2-resident) instead of shared memory --------------------------
template <int G>
__global__ void __launch_bounds__(G, 1) velo_sort_big_kernel(const KernelArgs a) {
  __shared__ SortTeam<G> ts;
  __shared__ float module_z[VELO_MAX_MODULES];
  const uint32_t tid = threadIdx.x;
  if (tid < VELO_MAX_MODULES) module_z[tid] = a.module_z[tid];
  unsigned char* blk = a.ws.slabs + (size_t)blockIdx.x * slab_layout().bytes;
  uint32_t parity = 0;
  const uint32_t base = a.event_offsets[0];
  for (;;) {
    __syncthreads();
    if (tid == 0) {
      const uint32_t k = atomicAdd(&a.ws.counters[kCtrBigSortTicket], 1u);
      ts.skip = k >= a.ws.counters[kCtrBigN];
      if (!ts.skip) {
        const uint32_t e = a.ws.big_list[k], o0 = a.event_offsets[e];
        ts.event = e; ts.n = a.event_offsets[e + 1] - o0; ts.o0 = o0; ts.ol = o0 - base; ts.trouble = 0; ts.unpack = 0;
      }
    }
    __syncthreads();
    if (ts.skip) break;
    sort_event<G, 8>(a, module_z, ts, blk, 0u, tid, parity, kEvBig);
  }
}

int launch_sort_big_impl(const KernelArgs& a, cudaStream_t stream) {
  const uint32_t sms = num_sms();
  const uint32_t grid = a.ws.n_slabs < sms ? a.ws.n_slabs : sms;
  if (grid == 0) return 0;
  velo_sort_big_kernel<1024><<<grid, 1024, 0, stream>>>(a);
  return (int)cudaGetLastError();
}

template <int G, int kTeams>
int launch_sort_t(const KernelArgs& a, cudaStream_t stream, uint32_t pool_units) {
  using Ctl = SortCtl<G, kTeams>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  const uint32_t smem = kCtl + pool_units * kUnitBytes;
  cudaError_t err = cudaFuncSetAttribute(velo_sort_kernel<G, kTeams>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err != cudaSuccess) return (int)err;
  const uint32_t sms = num_sms();
  const uint32_t want = (a.n_events + kTeams - 1) / kTeams;
  const uint32_t grid = want < sms ? (want ? want : 1u) : sms;
  velo_sort_kernel<G, kTeams><<<grid, G * kTeams, smem, stream>>>(a, pool_units);
  return (int)cudaGetLastError();
}

}  // namespace

int launch_sort_big(const KernelArgs& a, cudaStream_t stream) { return launch_sort_big_impl(a, stream); }

int launch_sort(const KernelArgs& a, cudaStream_t stream, const PipeOpts& o) {
  const uint32_t pu = o.pool_units ? (o.pool_units > kPoolUnitsMax ? kPoolUnitsMax : o.pool_units) : kPoolUnitsMax;
  // small events (open VELO: 320 hits) keep more teams busy with 128 threads each; from mu = 5 sizes on
  // 256 threads finish an event in half the time and four of them fill the pool (measured: profiles/r02e)
  const uint32_t mean = a.n_events ? a.n_hits / a.n_events : 0u;
  const uint32_t teams = o.sort_teams ? o.sort_teams : (mean < 768u ? 8u : 0u);
  switch (teams) {
    case 4: return launch_sort_t<128, 4>(a, stream, pu);
    case 6: return launch_sort_t<128, 6>(a, stream, pu);
    case 7: return launch_sort_t<128, 7>(a, stream, pu);
    case 8: return launch_sort_t<128, 8>(a, stream, pu);
    case 253: return launch_sort_t<256, 3>(a, stream, pu);
    case 252: return launch_sort_t<512, 2>(a, stream, pu);
    default: return launch_sort_t<256, 4>(a, stream, pu);   // 22 us per event with 256 threads, 43 us with 128
  }
}

}  // namespace velo
