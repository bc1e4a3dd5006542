// velo_fit.cu — stage 3 of the pipeline: O-10 weak-track filter, O-11 straight-line fit, O-12 chi2
// cut, O-13 clone filter (hit ownership by 64-bit key), then S7 output as count -> scan -> write,
// every final array written once (sm_100a).
//
// velo_fit_kernel: teams of G threads in persistent CTAs take the events largest-first. An event's
// candidates (rows of sorted hit indices and of hit coordinates in discovery order, module masks,
// seed scatters) and final flag bits come from stage 2's global scratch: a thread fits its candidate
// straight from its coordinate row, no gather. Shared memory holds only what threads share: the
// O-13 owner per hit and the candidates' keys. One thread per candidate fits and filters. What leaves: per candidate its fate and nine state words
// (coalesced planes in global scratch), per event the number of surviving tracks and track hits.
// velo_offsets_kernel (velo_kernels.cu) scans those counts into event_track_offsets. Then
// velo_write_kernel, a streaming kernel with one warp per event and no shared memory, places every
// surviving track: state planes, track_hit_offsets, and track_hits as original hit indices. Events
// that the pipeline deferred to the general slab kernel (whose tracks sit in temp blocks) are
// copied into place by the same kernel.
//
// Step semantics: SURVEY.md §8(c) O-10 ... O-14; every float operation is a round-to-nearest
// intrinsic in the oracle's order (no FMA contraction), so states are bit-identical to the oracle's.
#include "velo_device.cuh"
#include "velo_internal.h"
#include "velo_pool.cuh"

namespace velo {

namespace {


template <int G>
struct FitTeam {
  uint32_t wsum[4 * (G / 32)];
  uint32_t event, skip, n, sb, o0;
  uint32_t units, first_unit, pool_off;
  uint32_t cbase, ncand;
  unsigned long long ph_last;        // phase clocks (-DVELO_TIMELINE builds)
};

template <int G, int kTeams>
struct FitCtl {
  PoolCtl pool;
  float module_z[VELO_MAX_MODULES];
  float module_z_b[VELO_MAX_MODULES];  // two-plane geometries (L-1)
  FitTeam<G> team[kTeams];
};

__device__ __forceinline__ uint32_t a16(uint32_t v) { return (v + 15u) & ~15u; }

struct FitLayout { uint32_t rowc, own, fbits, key, mask, state, bytes; };
__device__ __forceinline__ FitLayout fit_layout(uint32_t n, uint32_t nt, bool cache_rows) {
  FitLayout L;
  uint32_t o = 0;
  L.rowc = o; o += cache_rows ? 32u * nt : 0u;   // the first 16 hit indices of every candidate's row (teams in shared memory)
  L.own = o; o += a16(4u * n);           // O-13 owner (candidate id) per hit
  L.fbits = o; o += a16(4u * ((n + 31u) >> 5));
  L.key = o; o += a16(8u * nt);
  L.mask = o; o += a16(4u * nt);
  L.state = o; o += a16(nt);
  L.bytes = o;
  return L;
}

// Calls f(i, h) for the hits h (sorted indices) of candidate row `row` in discovery order.
template <class F>
__device__ __forceinline__ void for_hits(const uint16_t* row, uint32_t n, F&& f) {
  const uint4* r4 = reinterpret_cast<const uint4*>(row);
  for (uint32_t g = 0; g * 8u < n; ++g) {
    const uint4 v = r4[g];
    const uint32_t q[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (uint32_t j = 0; j < 8; ++j) {
      if (g * 8u + j < n) f(g * 8u + j, (q[j >> 1] >> ((j & 1u) * 16u)) & 0xffffu);
    }
  }
}

// The same with the row's first 32 bytes (16 hits) taken from the event's copy `c` in shared memory: a
// candidate's row is read in four passes of fit_event, and each read from global scratch is a round trip
// to L2/HBM that the few warps of a team cannot hide. Longer tracks (rare) read their tail from the row.
template <bool kCache, class F>
__device__ __forceinline__ void for_hits_c(const uint4* c, const uint16_t* row, uint32_t n, F&& f) {
  const uint4* r4 = reinterpret_cast<const uint4*>(row);
  for (uint32_t g = 0; g * 8u < n; ++g) {
    const uint4 v = (kCache && g < 2u) ? c[g] : r4[g];
    const uint32_t q[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (uint32_t j = 0; j < 8; ++j) {
      if (g * 8u + j < n) f(g * 8u + j, (q[j >> 1] >> ((j & 1u) * 16u)) & 0xffffu);
    }
  }
}

// ---- O-11 straight-line fit with z taken from the module planes ---------------------------------
// s9 = x, y, tx, ty, z, cxx, cxtx, vt, chi2 (the 13 state words repeat cxx, cxtx, vt for y and add n).
// Hits are visited in discovery order = decreasing module = the set bits of `mask` from the top.
// The (x, y) of a candidate's hits in discovery order: the first 16 hits are loaded into registers
// up front (eight independent 16-byte loads in flight per thread), the rare rest comes on demand.
struct XyRow {
  float4 v[8];
  const float4* r4;
  __device__ __forceinline__ void load(const float2* rxy, uint32_t n) {
    r4 = reinterpret_cast<const float4*>(rxy);
#pragma unroll
    for (uint32_t g = 0; g < 8; ++g) v[g] = 2u * g < n ? __ldcs(r4 + g) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
};
// Calls f(p) for the hits in discovery order.
template <class F>
__device__ __forceinline__ void for_xy(const XyRow& r, uint32_t n, F&& f) {
#pragma unroll
  for (uint32_t g = 0; g < 8; ++g) {
    if (2u * g >= n) break;
    f(make_float2(r.v[g].x, r.v[g].y));
    if (2u * g + 1u < n) f(make_float2(r.v[g].z, r.v[g].w));
  }
  for (uint32_t g = 8; 2u * g < n; ++g) {
    const float4 v = r.r4[g];
    f(make_float2(v.x, v.y));
    if (2u * g + 1u < n) f(make_float2(v.z, v.w));
  }
}

// kTwoPlane (L-1): bit m of the row's kSideSlot entry says on which of module m's two planes the hit lies.
template <bool kTwoPlane>
__device__ __forceinline__ void fit_track(const float2* rxy_g, const float* mz, const float* mzb, uint32_t n, uint32_t mask,
                                          float sig2, float inv_s2, float* s9) {
  XyRow rxy;
  rxy.load(rxy_g, n);
  const uint32_t sides = kTwoPlane ? __float_as_uint(__ldcs(reinterpret_cast<const float*>(rxy_g + kSideSlot))) : 0u;
  auto zof = [&](uint32_t m) -> float { return (kTwoPlane && ((sides >> m) & 1u)) ? mzb[m] : mz[m]; };
  float sz = 0.0f, sx = 0.0f, sy = 0.0f;
  uint32_t mk = mask;
  for_xy(rxy, n, [&](const float2 p) {
    const uint32_t m = 31u - __clz(mk); mk &= ~(1u << m);
    sz = __fadd_rn(sz, zof(m)); sx = __fadd_rn(sx, p.x); sy = __fadd_rn(sy, p.y);
  });
  const float nf = (float)n;
  const float zb = __fdiv_rn(sz, nf), xb = __fdiv_rn(sx, nf), yb = __fdiv_rn(sy, nf);
  float sdd = 0.0f, sdx = 0.0f, sdy = 0.0f;
  mk = mask;
  for_xy(rxy, n, [&](const float2 p) {
    const uint32_t m = 31u - __clz(mk); mk &= ~(1u << m);
    const float d = __fsub_rn(zof(m), zb);
    sdd = __fadd_rn(sdd, __fmul_rn(d, d));
    sdx = __fadd_rn(sdx, __fmul_rn(d, __fsub_rn(p.x, xb)));
    sdy = __fadd_rn(sdy, __fmul_rn(d, __fsub_rn(p.y, yb)));
  });
  const float tx = __fdiv_rn(sdx, sdd), ty = __fdiv_rn(sdy, sdd);
  float c = 0.0f;
  mk = mask;
  for_xy(rxy, n, [&](const float2 p) {
    const uint32_t m = 31u - __clz(mk); mk &= ~(1u << m);
    const float d = __fsub_rn(zof(m), zb);
    const float rx = __fsub_rn(__fsub_rn(p.x, xb), __fmul_rn(tx, d));
    const float ry = __fsub_rn(__fsub_rn(p.y, yb), __fmul_rn(ty, d));
    c = __fadd_rn(c, __fmul_rn(rx, rx));
    c = __fadd_rn(c, __fmul_rn(ry, ry));
  });
  const float s2 = __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty));
  float dzb;
  if (s2 < 1e-12f) dzb = 0.0f;
  else dzb = -__fdiv_rn(__fadd_rn(__fmul_rn(xb, tx), __fmul_rn(yb, ty)), s2);
  const float vt = __fdiv_rn(sig2, sdd);
  s9[0] = __fadd_rn(xb, __fmul_rn(tx, dzb));
  s9[1] = __fadd_rn(yb, __fmul_rn(ty, dzb));
  s9[2] = tx; s9[3] = ty;
  s9[4] = __fadd_rn(zb, dzb);
  s9[5] = __fadd_rn(__fdiv_rn(sig2, nf), __fmul_rn(__fmul_rn(dzb, dzb), vt));
  s9[6] = __fmul_rn(dzb, vt);
  s9[7] = vt;
  s9[8] = __fmul_rn(c, inv_s2);
}

template <int G>
__device__ void fit_fetch(const KernelArgs& a, PoolCtl& pool, FitTeam<G>& ts) {
  const uint32_t k = atomicAdd(&a.ws.counters[kCtrFitTicket], 1u);
  ts.event = k; ts.units = 0; ts.skip = 1;
  if (k >= a.n_events) return;
  // largest first, then smallest, second largest, ... (velo_order_kernel): the order only schedules
  const uint32_t e = a.ws.order[(k & 1u) ? (k >> 1) : a.n_events - 1u - (k >> 1)];
  ts.event = e;
  const EvInfo info = a.ws.ev_info[e];
  if (info.state == kEvDeferred) return;           // the slab kernel has written this event's counts
  if (info.state == kEvBig) return;                // velo_fit_big_kernel takes it
  if (info.state != kEvReady || info.ncand == 0) { a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0); return; }
  const FitLayout L = fit_layout(info.n, info.ncand, true);
  const uint32_t units = (L.bytes + kUnitBytes - 1u) / kUnitBytes;   // fits the pool: stage 1 checked fit_smem_bound
  const uint32_t first = pool_alloc(pool, units);
  ts.n = info.n; ts.cbase = info.cbase; ts.ncand = info.ncand;
  ts.o0 = a.event_offsets[e];
  ts.sb = sorted_base(ts.o0 - a.event_offsets[0], e);
  ts.units = units; ts.first_unit = first; ts.pool_off = first * kUnitBytes; ts.skip = 0;
}

// ---- one pipeline event, by one team ------------------------------------------------------------
template <int G, bool kTwoPlane = false, bool kCacheRows = false>
__device__ void fit_event(const KernelArgs& a, const float* mz, const float* mzb, FitTeam<G>& ts, unsigned char* blk,
                          uint32_t team, uint32_t tid, uint32_t& parity) {
  const velo_params_t& P = a.P;
  const uint32_t e = ts.event, n = ts.n, nt = ts.ncand, o0 = ts.o0;
  const FitLayout L = fit_layout(n, nt, kCacheRows);
  uint4* rowc = (uint4*)(blk + L.rowc);  // kCacheRows: candidate t's first 16 hit indices at rowc[2t], rowc[2t + 1]
  uint32_t* own = (uint32_t*)(blk + L.own);
  uint32_t* fbits = (uint32_t*)(blk + L.fbits);
  unsigned long long* tkey = (unsigned long long*)(blk + L.key);
  uint32_t* tmask = (uint32_t*)(blk + L.mask);
  uint8_t* tstate = blk + L.state;       // 0 dropped by O-10/O-12, 1 passed, 2 survives O-13
  const uint16_t* rows = a.ws.rows + (size_t)ts.cbase * 32u;
  const uint2* cmeta = a.ws.cmeta + ts.cbase;
  const float2* rows_xy = a.ws.rows_xy + (size_t)ts.cbase * kXyStride;
  float* cfit = a.ws.cfit + ts.cbase;    // plane k of candidate t: cfit[k * cand_total + t]
  const size_t cs = a.ws.cand_total;

  {
    const uint32_t* fb = a.ws.flag_bits + ((o0 - a.event_offsets[0]) >> 5) + e;
    for (uint32_t i = tid; i < ((n + 31u) >> 5); i += G) fbits[i] = fb[i];
  }
  team_sync<G>(team);
  // ---- O-10 ghost filter part 1 (reads the final flags) -------------------------------------------
  for (uint32_t t = tid; t < nt; t += G) {
    const uint2 cm = cmeta[t];
    uint2 r = make_uint2(0u, 0u);
    if (kCacheRows) {
      // both halves lie in one 32-byte sector: loaded together with cmeta, whatever the track's length
      const uint4* gr = reinterpret_cast<const uint4*>(rows + t * 32u);
      const uint4 r0 = gr[0], r1 = gr[1];
      rowc[2u * t] = r0; rowc[2u * t + 1u] = r1;
      r = make_uint2(r0.x, r0.y);
    }
    tmask[t] = cm.x;
    // the coordinate row this thread fits from in the next pass (64 bytes per 8 hits): on its way to L2 now
    prefetch_l2(rows_xy + t * kXyStride);
    if (__popc(cm.x) > 8) prefetch_l2(rows_xy + t * kXyStride + 8u);
    bool pass = true;
    if (__popc(cm.x) == 3) {
      if (!kCacheRows) r = *reinterpret_cast<const uint2*>(rows + t * 32u);
      const uint32_t h0 = r.x & 0xffffu, h1 = r.x >> 16, h2 = r.y & 0xffffu;
      const uint32_t f = ((fbits[h0 >> 5] >> (h0 & 31u)) | (fbits[h1 >> 5] >> (h1 & 31u)) | (fbits[h2 >> 5] >> (h2 & 31u))) & 1u;
      if (f || !(__uint_as_float(cm.y) <= P.max_scatter_weak)) pass = false;
    }
    tstate[t] = pass ? 1 : 0;
  }
  VELO_PH(a.ws.phase_clk, ts, 34);
  // ---- O-11 fit, O-12 chi2 cut, O-13 key -----------------------------------------------------------
  const float sig2 = __fmul_rn(P.sigma_hit, P.sigma_hit);
  const float inv_s2 = __fdiv_rn(1.0f, sig2);
  for (uint32_t t = tid; t < nt; t += G) {
    if (!tstate[t]) continue;
    const uint32_t mask = tmask[t], nh = (uint32_t)__popc(mask);
    float s9[9];
    fit_track<kTwoPlane>(rows_xy + t * kXyStride, mz, mzb, nh, mask, sig2, inv_s2, s9);
    const float lim = __fmul_rn(P.max_chi2_ndof, (float)(2 * (int)nh - 4));
    if (s9[8] > lim) { tstate[t] = 0; continue; }
    const uint32_t centre = kCacheRows ? rowc[2u * t].x >> 16 : (uint32_t)rows[t * 32u + 1u];
    tkey[t] = ((unsigned long long)(255u - nh) << 56) | ((unsigned long long)__float_as_uint(s9[8]) << 24) |
              (unsigned long long)centre;
#pragma unroll
    for (uint32_t k = 0; k < 9; ++k) cfit[k * cs + t] = s9[k];
    // O-13 owners, step 1: every passing candidate writes its id on its hits (plain stores: where
    // several share a hit, any one of them lands)
    for_hits_c<kCacheRows>(rowc + 2u * t, rows + t * 32u, nh, [&](uint32_t, uint32_t h) { own[h] = t; });
  }
  team_sync<G>(team);
  VELO_PH(a.ws.phase_clk, ts, 35);
  // ---- O-13 owners: owner[h] = the candidate with the smallest key among those that contain h ----
  // Step 2: a candidate that finds another id on one of its hits settles it with a compare-and-swap
  // on the 64-bit keys. Hits are shared rarely, so the common path has no atomics.
  VELO_PH(a.ws.phase_clk, ts, 36);
  for (uint32_t t = tid; t < nt; t += G) {
    if (!tstate[t]) continue;
    // first look at all hits at once (independent loads): most candidates own every hit of theirs
    const uint32_t nh = (uint32_t)__popc(tmask[t]);
    uint32_t contested = 0;
    for_hits_c<kCacheRows>(rowc + 2u * t, rows + t * 32u, nh, [&](uint32_t i, uint32_t h) { contested |= (own[h] != t) ? (1u << i) : 0u; });
    if (!contested) continue;
    const unsigned long long key = tkey[t];
    for_hits_c<kCacheRows>(rowc + 2u * t, rows + t * 32u, nh, [&](uint32_t i, uint32_t h) {
      if (!((contested >> i) & 1u)) return;
      uint32_t old = *(volatile uint32_t*)&own[h];
      while (old != t && key < tkey[old]) {
        const uint32_t seen = atomicCAS(&own[h], old, t);
        if (seen == old) break;
        old = seen;
      }
    });
  }
  team_sync<G>(team);
  VELO_PH(a.ws.phase_clk, ts, 37);
  // ---- O-13 clone filter; the event's counts --------------------------------------------------------
  uint32_t run_t = 0, run_h = 0;
  uint8_t* cstate = a.ws.cstate + ts.cbase;
  for (uint32_t t0 = 0; t0 < nt; t0 += G) {
    const uint32_t t = t0 + tid;
    uint32_t nh = 0, surv = 0;
    if (t < nt && tstate[t]) {
      nh = (uint32_t)__popc(tmask[t]);
      uint32_t lost = 0;
      for_hits_c<kCacheRows>(rowc + 2u * t, rows + t * 32u, nh, [&](uint32_t, uint32_t h) { lost += (own[h] != t) ? 1u : 0u; });
      surv = !((unsigned long long)lost * P.clone_den > (unsigned long long)nh * P.clone_num) ? 1u : 0u;
      if (!surv) nh = 0;
    }
    if (t < nt) cstate[t] = (uint8_t)surv;
    uint32_t tot_h, pre_t, tot_t;
    team_scan2<G>(nh, surv, ts.wsum, team, parity, &tot_h, &pre_t, &tot_t);
    run_t += tot_t; run_h += tot_h;
  }
  if (tid == 0) a.ws.ev_rec[e] = make_uint4(0, 0, run_t, run_h);
}

// ---- the fit kernel: one CTA per SM, kTeams teams of G threads ------------------------------------
template <int G, int kTeams, bool kTwoPlane>
__global__ void __launch_bounds__(G * kTeams, 1) velo_fit_kernel(const KernelArgs a, const uint32_t pool_units) {
  extern __shared__ __align__(16) unsigned char smem[];
  using Ctl = FitCtl<G, kTeams>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  Ctl& ctl = *reinterpret_cast<Ctl*>(smem);
  unsigned char* pool = smem + kCtl;
  const uint32_t team = threadIdx.x / G, tid = threadIdx.x % G;
  if (threadIdx.x == 0) pool_init(ctl.pool, pool_units);
  if (threadIdx.x < VELO_MAX_MODULES) { ctl.module_z[threadIdx.x] = a.module_z[threadIdx.x]; ctl.module_z_b[threadIdx.x] = a.module_z_b[threadIdx.x]; }
  FitTeam<G>& ts = ctl.team[team];
  __syncthreads();
  VELO_STAGE_BEGIN(a.ws.phase_clk, 2);
  uint32_t parity = 0;
  VELO_PH_START(ts);
  for (;;) {
    if (tid == 0) fit_fetch<G>(a, ctl.pool, ts);
    team_sync<G>(team);
    if (ts.event >= a.n_events) break;
    VELO_PH(a.ws.phase_clk, ts, 33);     // ticket, descriptors, pool
    if (!ts.skip) fit_event<G, kTwoPlane, true>(a, ctl.module_z, ctl.module_z_b, ts, pool + ts.pool_off, team, tid, parity);
    team_sync<G>(team);
    if (tid == 0 && ts.units) pool_free(ctl.pool, ts.first_unit, ts.units);
    VELO_PH(a.ws.phase_clk, ts, 38);     // clone filter, counts
    VELO_PH_COUNT(a.ws.phase_clk, 32, 1);
  }
  VELO_STAGE_END(a.ws.phase_clk, 2);
}

// ---- the same stage for the events of ws.big_list: one CTA of G threads per event, the per-event
// arrays (owner per hit, keys, masks) in the CTA's global slab (L2-resident) -------------------------
template <int G>
__global__ void __launch_bounds__(G, 1) velo_fit_big_kernel(const KernelArgs a) {
  __shared__ FitTeam<G> ts;
  __shared__ float module_z[VELO_MAX_MODULES];
  const uint32_t tid = threadIdx.x;
  if (tid < VELO_MAX_MODULES) module_z[tid] = a.module_z[tid];
  unsigned char* blk = a.ws.slabs + (size_t)blockIdx.x * slab_layout().bytes;
  uint32_t parity = 0;
  const uint32_t base = a.event_offsets[0];
  for (;;) {
    __syncthreads();
    if (tid == 0) {
      const uint32_t k = atomicAdd(&a.ws.counters[kCtrBigFitTicket], 1u);
      ts.units = k >= a.ws.counters[kCtrBigN];      // 1 = no more events
      ts.skip = 1;
      if (!ts.units) {
        const uint32_t e = a.ws.big_sorted[k];
        const EvInfo info = a.ws.ev_info[e];
        ts.event = e;
        if (info.state == kEvBig) {                  // else: the general kernel has written its counts
          if (info.ncand == 0) a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0);
          else {
            ts.n = info.n; ts.cbase = info.cbase; ts.ncand = info.ncand;
            ts.o0 = a.event_offsets[e]; ts.sb = sorted_base(ts.o0 - base, e); ts.skip = 0;
          }
        }
      }
    }
    __syncthreads();
    if (ts.units) break;
    if (!ts.skip) fit_event<G>(a, module_z, module_z, ts, blk, 0u, tid, parity);
  }
}

// ---- S7 write: one warp per event places its surviving tracks in the final arrays ----------------
// Offsets come from velo_offsets_kernel (event_track_offsets, ws.ev_hit_base). Candidates are in
// creation order, so a running count over them is the track's place inside the event.
template <int kWarps, int kMinBlocks>
__global__ void __launch_bounds__(32 * kWarps, kMinBlocks) velo_write_kernel(const KernelArgs a) {
  // the hit lists of 32 candidates at a time go through shared memory, so that the warp writes
  // track_hits as whole sectors instead of 32 scattered words per store
  __shared__ uint32_t stage_all[kWarps][32 * VELO_MAX_MODULES];
  uint32_t* stage = stage_all[threadIdx.x >> 5];
  const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t tot_t = a.event_track_offsets[a.n_events], tot_h = a.ws.ev_hit_base[a.n_events];
  if (tot_t > a.cap_tracks || tot_h > a.cap_track_hits) return;  // VELO_ERR_CAPACITY: nothing valid
  const size_t cs = a.cap_tracks, cc = a.ws.cand_total;
  const uint32_t obase = a.event_offsets[0];
  for (uint32_t e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; e < a.n_events; e += warps) {
    // the event's four descriptors in one round trip (a warp has one event: every round trip counts)
    const uint4 r = a.ws.ev_rec[e];
    const uint32_t dst_t = a.event_track_offsets[e], dst_h = a.ws.ev_hit_base[e];
    EvInfo info{0u, kEvDeferred, 0u, 0u};
    if (!a.all_deferred) info = a.ws.ev_info[e];
    const uint32_t o0 = a.event_offsets[e];
    if (r.z == 0) continue;
    if (info.state == kEvDeferred) {
      // tracks of the general kernel: temp block -> place (four independent loads per lane and trip)
      const uint32_t* src = a.ws.tmp_hits + r.y;
      uint32_t* dst = a.track_hits + dst_h;
      for (uint32_t k = lane; k < r.w; k += 128u) {
        uint32_t v[4];
#pragma unroll
        for (uint32_t q = 0; q < 4; ++q) v[q] = (k + 32u * q < r.w) ? src[k + 32u * q] : 0u;
#pragma unroll
        for (uint32_t q = 0; q < 4; ++q) if (k + 32u * q < r.w) dst[k + 32u * q] = v[q];
      }
      for (uint32_t k = lane; k < r.z; k += 32u) {
        float v[VELO_N_STATE];
        const uint32_t lo = a.ws.tmp_loff[r.x + k];
#pragma unroll
        for (int p = 0; p < VELO_N_STATE; ++p) v[p] = a.ws.tmp_states[(size_t)p * cs + r.x + k];
        a.track_hit_offsets[dst_t + k] = dst_h + lo;
#pragma unroll
        for (int p = 0; p < VELO_N_STATE; ++p) a.states[(size_t)p * cs + dst_t + k] = v[p];
      }
      continue;
    }
    if (info.state == kEvBig) continue;                 // velo_write_big_kernel: a CTA per such event
    const uint16_t* orig = a.ws.sorig + sorted_base(o0 - obase, e);
    const uint16_t* rows = a.ws.rows + (size_t)info.cbase * 32u;
    const uint2* cmeta = a.ws.cmeta + info.cbase;
    const uint8_t* cstate = a.ws.cstate + info.cbase;
    const float* cfit = a.ws.cfit + info.cbase;
    uint32_t run_t = 0, run_h = 0;
    // the event's index map, candidate masks and fates, and the first pass's rows and fit planes: on their way to L2
    for (uint32_t k = lane * 64u; k < info.n; k += 32u * 64u) prefetch_l2(orig + k);
    for (uint32_t k = lane * 16u; k < info.ncand; k += 32u * 16u) prefetch_l2(cmeta + k);
    if (lane * 128u < info.ncand) prefetch_l2(cstate + lane * 128u);
    if (lane < info.ncand) prefetch_l2(rows + lane * 32u);
    if (lane < 9u) prefetch_l2(cfit + lane * cc);
    for (uint32_t t0 = 0; t0 < info.ncand; t0 += 32u) {
      const uint32_t t = t0 + lane;
      if (t + 32u < info.ncand) {        // the next pass's candidates: their rows and fit planes on the way to L2
        prefetch_l2(rows + (t + 32u) * 32u);
        if (lane < 9u) prefetch_l2(cfit + lane * cc + t0 + 32u);
      }
      const bool surv = t < info.ncand && cstate[t] != 0;
      const uint32_t nh = surv ? (uint32_t)__popc(cmeta[t].x) : 0u;
      const uint32_t b = __ballot_sync(0xffffffffu, surv);
      uint32_t inc = nh;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= (uint32_t)d) inc += o; }
      const uint32_t lt = run_t + (uint32_t)__popc(b & ((1u << lane) - 1u)), lh = run_h + inc - nh;
      const uint32_t pass_h = __shfl_sync(0xffffffffu, inc, 31), pass_base = run_h;
      run_t += (uint32_t)__popc(b); run_h += pass_h;
      if (surv) {
        float s9[9];
#pragma unroll
        for (uint32_t k = 0; k < 9; ++k) s9[k] = cfit[k * cc + t];
        float* dst_s = a.states + dst_t + lt;
        dst_s[0] = s9[0]; dst_s[cs] = s9[1]; dst_s[2 * cs] = s9[2]; dst_s[3 * cs] = s9[3]; dst_s[4 * cs] = s9[4];
        dst_s[5 * cs] = s9[5]; dst_s[6 * cs] = s9[6]; dst_s[7 * cs] = s9[7];
        dst_s[8 * cs] = s9[5]; dst_s[9 * cs] = s9[6]; dst_s[10 * cs] = s9[7];
        dst_s[11 * cs] = s9[8]; dst_s[12 * cs] = __uint_as_float(nh);
        a.track_hit_offsets[dst_t + lt] = dst_h + lh;
        uint32_t* st = stage + (lh - pass_base);
        for_hits(rows + t * 32u, nh, [&](uint32_t i, uint32_t h) { st[i] = o0 + orig[h]; });
      }
      __syncwarp();
      uint32_t* dst = a.track_hits + dst_h + pass_base;
      for (uint32_t k = lane; k < pass_h; k += 32u) dst[k] = stage[k];
      __syncwarp();
    }
  }
}

// The same for the events of the one-event-per-CTA pipeline (thousands of tracks each): a CTA per
// event, a block-wide scan over its candidates instead of a warp's.
__global__ void __launch_bounds__(1024) velo_write_big_kernel(const KernelArgs a) {
  __shared__ unsigned long long warp_sums[33];
  const uint32_t tid = threadIdx.x;
  const uint32_t tot_t = a.event_track_offsets[a.n_events], tot_h = a.ws.ev_hit_base[a.n_events];
  if (tot_t > a.cap_tracks || tot_h > a.cap_track_hits) return;  // VELO_ERR_CAPACITY: nothing valid
  const size_t cs = a.cap_tracks, cc = a.ws.cand_total;
  const uint32_t obase = a.event_offsets[0], nb = a.ws.counters[kCtrBigN];
  for (uint32_t k = blockIdx.x; k < nb; k += gridDim.x) {
    const uint32_t e = a.ws.big_sorted[k];
    const EvInfo info = a.ws.ev_info[e];
    const uint4 r = a.ws.ev_rec[e];
    if (info.state != kEvBig || r.z == 0) continue;       // deferred on the way: the warp-per-event kernel copies its temp block
    const uint32_t dst_t = a.event_track_offsets[e], dst_h = a.ws.ev_hit_base[e];
    const uint32_t o0 = a.event_offsets[e];
    const uint16_t* orig = a.ws.sorig + sorted_base(o0 - obase, e);
    const uint16_t* rows = a.ws.rows + (size_t)info.cbase * 32u;
    const uint2* cmeta = a.ws.cmeta + info.cbase;
    const uint8_t* cstate = a.ws.cstate + info.cbase;
    const float* cfit = a.ws.cfit + info.cbase;
    uint32_t run_t = 0, run_h = 0;
    for (uint32_t t0 = 0; t0 < info.ncand; t0 += blockDim.x) {
      const uint32_t t = t0 + tid;
      const bool surv = t < info.ncand && cstate[t] != 0;
      const uint32_t nh = surv ? (uint32_t)__popc(cmeta[t].x) : 0u;
      unsigned long long tot;
      const unsigned long long pre = block_scan_excl(((unsigned long long)nh << 32) | (surv ? 1ull : 0ull), warp_sums, &tot);
      const uint32_t lt = run_t + (uint32_t)(pre & 0xffffffffu), lh = run_h + (uint32_t)(pre >> 32);
      run_t += (uint32_t)(tot & 0xffffffffu); run_h += (uint32_t)(tot >> 32);
      if (!surv) continue;
      float s9[9];
#pragma unroll
      for (uint32_t q = 0; q < 9; ++q) s9[q] = cfit[q * cc + t];
      float* dst_s = a.states + dst_t + lt;
      dst_s[0] = s9[0]; dst_s[cs] = s9[1]; dst_s[2 * cs] = s9[2]; dst_s[3 * cs] = s9[3]; dst_s[4 * cs] = s9[4];
      dst_s[5 * cs] = s9[5]; dst_s[6 * cs] = s9[6]; dst_s[7 * cs] = s9[7];
      dst_s[8 * cs] = s9[5]; dst_s[9 * cs] = s9[6]; dst_s[10 * cs] = s9[7];
      dst_s[11 * cs] = s9[8]; dst_s[12 * cs] = __uint_as_float(nh);
      a.track_hit_offsets[dst_t + lt] = dst_h + lh;
      uint32_t* dst = a.track_hits + dst_h + lh;
      for_hits(rows + t * 32u, nh, [&](uint32_t i, uint32_t h) { dst[i] = o0 + orig[h]; });
    }
  }
}

template <int G, int kTeams, bool kTwoPlane = false>
int launch_fit_t(const KernelArgs& a, cudaStream_t stream, uint32_t pool_units) {
  static_assert(G == 32 || kTeams <= 15, "named barriers 1..15");
  using Ctl = FitCtl<G, kTeams>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  const uint32_t smem = kCtl + pool_units * kUnitBytes;
  cudaError_t err = cudaFuncSetAttribute(velo_fit_kernel<G, kTeams, kTwoPlane>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err != cudaSuccess) return (int)err;
  const uint32_t sms = num_sms();
  const uint32_t want = (a.n_events + kTeams - 1) / kTeams;
  const uint32_t grid = want < sms ? (want ? want : 1u) : sms;
  velo_fit_kernel<G, kTeams, kTwoPlane><<<grid, G * kTeams, smem, stream>>>(a, pool_units);
  return (int)cudaGetLastError();
}

}  // namespace

int launch_fit(const KernelArgs& a, cudaStream_t stream, const PipeOpts& o) {
  if (a.n_events == 0) return 0;
  const uint32_t pu = o.pool_units ? (o.pool_units > kPoolUnitsMax ? kPoolUnitsMax : o.pool_units) : kPoolUnitsMax;
  const uint32_t mean = a.n_events ? a.n_hits / a.n_events : 0u;
  if (a.two_plane)                     // two sensor planes per module (L-1): the default team shapes only
    return mean < 768u ? launch_fit_t<64, 15, true>(a, stream, pu) : launch_fit_t<128, 8, true>(a, stream, pu);
  switch (o.fit_teams ? o.fit_teams : (mean < 768u ? 15u : 0u)) {   // small events: 15 teams of 64 threads
    case 4: return launch_fit_t<128, 4>(a, stream, pu);
    case 6: return launch_fit_t<128, 6>(a, stream, pu);
    case 8: return launch_fit_t<128, 8>(a, stream, pu);
    case 12: return launch_fit_t<64, 12>(a, stream, pu);
    case 15: return launch_fit_t<64, 15>(a, stream, pu);
    case 254: return launch_fit_t<256, 4>(a, stream, pu);
    // seven teams of 128 threads: 72 registers per thread instead of 64 (no spills in the fit), and the pool holds
    // seven events with their row copies more easily than eight (567 us; 8 teams: 575, 6 teams: 582)
    default: return launch_fit_t<128, 7>(a, stream, pu);
  }
}

int launch_fit_big(const KernelArgs& a, cudaStream_t stream) {
  const uint32_t sms = num_sms();
  const uint32_t grid = a.ws.n_slabs < sms ? a.ws.n_slabs : sms;
  if (grid == 0) return 0;
  velo_fit_big_kernel<1024><<<grid, 1024, 0, stream>>>(a);
  return (int)cudaGetLastError();
}

int launch_write(const KernelArgs& a, cudaStream_t stream) {
  if (a.n_events == 0) return 0;
  // a warp per event, four per CTA (1, 2 or 8 warps per CTA: 315, 309, 312 us against 305)
  velo_write_kernel<4, 8><<<(a.n_events + 3u) / 4u, 128, 0, stream>>>(a);
  if (a.big_path) velo_write_big_kernel<<<num_sms() * 2u, 1024, 0, stream>>>(a);
  return (int)cudaGetLastError();
}

}  // namespace velo
