// velo_track.cu — stage 2 of the pipeline: the O-6 module loop (S3 forwarding, S2 search-by-triplet
// seeding, hit flags) over the phi-sorted blocks that stage 1 left in global scratch (sm_100a).
//
// One persistent CTA per SM owns the SM's shared memory as a pool; a team of G threads (two warps for
// mu = 5 events, one for open-VELO events, four for events of several thousand hits) takes an event;
// its warps work side by side and meet twice per step (track_event_w). It holds, instead of the whole
// event, only what a step touches at random:
//   * a ring of four module slots fed by 1-D TMA bulk copies (cp.async.bulk + mbarrier): step s
//     reads modules s+1, s, s-1 while module s-2 is in flight, a full step ahead of its use;
//   * the list of ACTIVE tracks as self-contained 32-byte records (last two hits' coordinates,
//     phi and window starts of the latest hit, hit indices, module mask, candidate id), compacted
//     in place every step, so the lanes of the forwarding pass are always dense;
//   * one flag bit per hit, the first hit of every candidate, the list of unflagged centre hits.
// About 15 KB for a mu = 5 event of 1.9 k hits instead of the 34 KB of the whole sorted event, and
// only for the duration of the loop: the sort (stage 1) and the fit/filters/output (stage 3) run
// in their own kernels. Candidates leave as 64-byte rows of sorted hit indices plus {module mask,
// seed scatter}; the final flags leave as one bit per hit.
//
// Window scans never search: stage 1 stored with every hit where its window starts in the three
// modules a scan can target (records' words 2 and 3); a scan runs from there, three hits per trip
// with the loads issued first, until the window test fails. A window across +-pi first visits its
// low-phi run from position 0, so hits are always met in ascending sorted index and ties resolve
// to the lowest index by strict comparison (O-7, O-8). Step semantics: SURVEY.md §8(c) O-3 ... O-9;
// every float operation is a round-to-nearest intrinsic in the oracle's order (no FMA contraction).
#include "velo_device.cuh"
#include "velo_internal.h"
#include "velo_pool.cuh"

namespace velo {

namespace {

template <int G>
struct TrackTeam {
  unsigned long long mbar[4];        // one mbarrier per ring slot
  uint32_t wsum[2 * (G / 32)];
  uint32_t event, n, sb;             // event index, hits, first record in the sorted scratch
  uint32_t units, first_unit, pool_off, skip;
  uint32_t maxmod, cbase, tcap, acap;
  uint32_t defer;                    // set by any thread: the event continues in the general kernel
  uint32_t npairs;                   // one-event-per-CTA seeding: (centre, h0) pairs listed in this round
  uint32_t unpack;                   // packed input: decode the deferred event for the general kernel
  unsigned long long ph_last;        // phase clocks (-DVELO_TIMELINE builds)
  uint16_t mod_off[kModOffStride];
};

template <int G, int kTeams>
struct TrackCtl {
  PoolCtl pool;
  float module_z[VELO_MAX_MODULES];
  float module_z_b[VELO_MAX_MODULES];  // two-plane geometries (L-1): the modules' second sensor planes
  float tz[VELO_MAX_MODULES * 4];    // O-4's z ratio for a track whose latest hits are on modules mb and mb + 1 + gap,
                                     // forwarded to module mb - 1 - pend: [mb][gap][pend], gap and pend 0 or 1
  TrackTeam<G> team[kTeams];
};

__device__ __forceinline__ uint32_t al16(uint32_t v) { return (v + 15u) & ~15u; }

constexpr uint32_t kSlotPad = 3;      // sentinel records behind every module slot of the ring (scan_run)
constexpr uint32_t kPairCap = 8192;   // (centre, h0) pairs per round of the one-event-per-CTA seeding
struct TrackLayout { uint32_t ring, act, flags, th0, cl, keys, plist, bytes; };
__device__ __forceinline__ TrackLayout track_layout(uint32_t n, uint32_t maxmod, uint32_t tcap, uint32_t acap,
                                                    bool with_ring = true) {
  TrackLayout L;
  uint32_t o = 0;
  L.ring = o; o += with_ring ? 4u * 16u * (maxmod + kSlotPad) : 0u;
  L.act = o; o += 32u * acap;
  L.flags = o; o += al16(4u * ((n + 31u + kSlotPad) >> 5));      // a padded trip may test a bit or two past the event
  L.th0 = o; o += al16(2u * tcap);
  L.cl = o; o += al16(2u * maxmod);
  // one-event-per-CTA form only: the best (scatter, h0, h2) of every centre of a round as a 64-bit
  // key, and the round's list of (centre, h0) pairs
  L.keys = o; o += with_ring ? 0u : 8u * 1024u;
  L.plist = o; o += with_ring ? 0u : 4u * kPairCap;
  L.bytes = o;
  return L;
}

template <int G>
__device__ void track_fetch(const KernelArgs& a, PoolCtl& pool, TrackTeam<G>& ts) {
  const uint32_t k = atomicAdd(&a.ws.counters[kCtrTrackTicket], 1u);
  ts.event = k; ts.units = 0; ts.skip = 1; ts.defer = 0; ts.unpack = 0;
  if (k >= a.n_events) return;
  // tickets walk the size-sorted list from both ends in turn: largest, smallest, second largest, ...
  const uint32_t e = a.ws.order[(k & 1u) ? (k >> 1) : a.n_events - 1u - (k >> 1)];
  ts.event = e;
  const EvInfo info = a.ws.ev_info[e];
  if (info.state != kEvReady) return;
  const uint32_t n = info.n;
  const uint32_t maxmod = a.ws.mod_off[(size_t)e * kModOffStride + kModOffStride - 1];
  const uint32_t tcap = cand_capacity(n), acap = active_capacity(n);
  const TrackLayout L = track_layout(n, maxmod, tcap, acap);
  const uint32_t units = (L.bytes + kUnitBytes - 1u) / kUnitBytes;
  if (units > pool.units) {
    a.ws.ev_info[e].state = kEvDeferred;
    a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
    ts.unpack = a.pixel != nullptr;
    return;
  }
  ts.cbase = atomicAdd(&a.ws.counters[kCtrCandAlloc], tcap);
#ifdef VELO_TIMELINE
  { const uint32_t tid = 0; VELO_PH(a.ws.phase_clk, ts, 24); }     // ticket and descriptors; what follows in "fetch" is the pool
#endif
  const uint32_t first = pool_alloc(pool, units);
  ts.n = n; ts.sb = sorted_base(a.event_offsets[e] - a.event_offsets[0], e);
  ts.maxmod = maxmod; ts.tcap = tcap; ts.acap = acap;
  ts.units = units; ts.first_unit = first; ts.pool_off = first * kUnitBytes; ts.skip = 0;
}

// Visits positions j0, j0 + 1, ... of a module slot (nm hits) while they lie inside the wide window
// (lo16w, limw), a few per trip: the 16-byte loads of a trip are issued before its arithmetic.
// f(jj, rec, in) must be branch-free. kPad: the slot ends with three sentinel records (x = +inf: their
// scatter is +inf, no cut accepts them), so a trip reads past the module without clamping its indices;
// otherwise padding lanes repeat position nm - 1 with `in` false.
template <bool kPad, class F>
__device__ __forceinline__ void scan_run(const uint4* slot, uint32_t j0, uint32_t nm, uint32_t lo16w, uint32_t limw, F&& f) {
  // records per trip: a window holds 0.7 hits on average (mu = 5), so most scans end in their first trip;
  // three per trip from a ring slot (measured: 4 / 3 / 2 / 1 -> 1469 / 1448 / 1467 / 1514 us), four from L2
  constexpr uint32_t T = kPad ? 3u : 4u;
  static_assert(T - 1u <= kSlotPad, "a trip may read T - 1 records past the module");
  for (uint32_t j = j0; j < nm; j += T) {
    uint4 r[T]; uint32_t jj[T];
#pragma unroll
    for (uint32_t k = 0; k < T; ++k) { jj[k] = kPad ? j + k : min(j + k, nm - 1u); r[k] = slot[jj[k]]; }
    bool in = false;
#pragma unroll
    for (uint32_t k = 0; k < T; ++k) {
      in = kPad ? (r[k].z - lo16w <= limw) : ((j + k < nm) & (r[k].z - lo16w <= limw));
      f(jj[k], r[k], in);
    }
    if (!in) break;     // the last of the trip is outside (or past the module): so is everything after it
  }
}

// O-3 window about unsigned phi c with half-width W, as a test on the phi field of a record word.
struct Win { uint32_t lo16, lim; bool wrapped; };
__device__ __forceinline__ Win make_win(uint32_t c, int W) {
  Win q;
  if (2 * (long long)W + 1 >= 65536) { q.lo16 = 0; q.lim = 0xffffffffu; q.wrapped = false; return q; }
  const uint32_t lo = (c - (uint32_t)W) & 0xffffu, hi = (c + (uint32_t)W) & 0xffffu;
  q.lo16 = lo << 16; q.lim = ((2u * (uint32_t)W) << 16) | 0xffffu; q.wrapped = lo > hi;
  return q;
}

// ---- one event, by one CTA ----------------------------------------------------------------------
// The one-event-per-CTA form for events too large for a ring in shared memory: the module slots ARE
// the sorted records in global scratch (L2), nothing is copied; one list of active tracks, compacted
// over the whole team after every pass; the event ends in state kEvBig so that the per-event kernels
// of stage 3 leave it to velo_fit_big_kernel. (Events that fit a team: track_event_w below.)
template <int G, bool kSameW>
__device__ void track_event_big(const KernelArgs& a, const float* mz, const float* tzt, TrackTeam<G>& ts, unsigned char* blk,
                                uint32_t team, uint32_t tid, uint32_t& parity) {
  const uint32_t M = a.n_modules, n = ts.n, e = ts.event;
  const velo_params_t& P = a.P;
  const uint32_t tcap = ts.tcap, acap = ts.acap;
  const TrackLayout L = track_layout(n, ts.maxmod, tcap, acap, false);
  const TrackLayout& L_ = L;
  uint4* act = (uint4*)(blk + L.act);
  uint32_t* flags = (uint32_t*)(blk + L.flags);   // one bit per sorted hit
  auto flagged = [&](uint32_t h) -> bool { return (flags[h >> 5] >> (h & 31u)) & 1u; };
  auto set_flag = [&](uint32_t h) { atomicOr(&flags[h >> 5], 1u << (h & 31u)); };
  // Active tracks beyond the shared-memory list (rare: it holds 0.055 per hit + 24, the mean peak is
  // 0.07 per hit at mu = 5 but lasts a step or two) live in global scratch: stage 3's state planes,
  // which nothing reads before stage 3 writes them.
  uint4* act_ovf = reinterpret_cast<uint4*>(a.ws.cfit) + 2u * (size_t)ts.cbase;
  auto act_load = [&](uint32_t k, uint4& q0, uint4& q1) {
    if (k < acap) { q0 = act[k]; q1 = act[acap + k]; }
    else { q0 = __ldcg(act_ovf + 2u * (k - acap)); q1 = __ldcg(act_ovf + 2u * (k - acap) + 1u); }
  };
  auto act_store = [&](uint32_t k, const uint4& q0, const uint4& q1) {
    if (k < acap) { act[k] = q0; act[acap + k] = q1; }
    else { act_ovf[2u * (k - acap)] = q0; act_ovf[2u * (k - acap) + 1u] = q1; }
  };
  uint16_t* th0 = (uint16_t*)(blk + L.th0);
  uint16_t* cl = (uint16_t*)(blk + L.cl);
  const uint16_t* mo = ts.mod_off;
  const uint4* grec = a.ws.rec16 + ts.sb;
  uint16_t* rows = a.ws.rows + (size_t)ts.cbase * 32u;
  uint2* cmeta = a.ws.cmeta + ts.cbase;
  float2* rows_xy = a.ws.rows_xy + (size_t)ts.cbase * kXyStride;
  const int Wseed = P.phi_window_seed, Wfwd = P.phi_window_fwd;
  const int Wwide = Wseed > Wfwd ? Wseed : Wfwd;

  for (uint32_t i = tid; i < kModOffStride; i += G) ts.mod_off[i] = a.ws.mod_off[(size_t)e * kModOffStride + i];
  for (uint32_t i = tid; i < ((n + 31u + kSlotPad) >> 5); i += G) flags[i] = 0;
  team_sync<G>(team);

  VELO_PH(a.ws.phase_clk, ts, 18);       // descriptors, flags, first loads

  uint32_t nact = 0, ncand = 0;
  const float max_seed = P.max_scatter_seed;
  // one comparison per visited record, as in track_event_w: scatter < bound, the bound starting at the next float
  // above the (finite: velo_api.cu) cut
  const float fwd_bound = nextafterf(P.max_scatter_fwd, INFINITY), seed_bound = nextafterf(P.max_scatter_seed, INFINITY);
  constexpr uint32_t kNone = 0xffffffffu;
  for (uint32_t s = M - 2; s >= 1; --s) {
    const uint32_t u = s - 1;
    // No hit in modules 0 .. u: forwarding can only miss and seeding finds no third hit, in this step
    // and in all that follow, and what a miss changes (the miss count) is not read after the loop.
    if (mo[u + 1] == 0) break;
    VELO_PH(a.ws.phase_clk, ts, 19);
    const uint32_t off_u = mo[u], nu = (uint32_t)mo[u + 1] - off_u;
    const uint32_t off_s = mo[s], ns = (uint32_t)mo[s + 1] - off_s;
    const uint32_t off_p = mo[s + 1], np = (uint32_t)mo[s + 2] - off_p;
    const uint4* ring_u = grec + off_u;
    const uint4* ring_s = grec + off_s;
    const uint4* ring_p = grec + off_p;
    const float z2 = mz[u];

    // ---- (A) O-7 forwarding into module u of every track active at the start of the step ----------
    uint32_t wbase = 0;
    for (uint32_t p0 = 0; p0 < nact; p0 += G) {
      const uint32_t k = p0 + tid;
      bool alive = false;
      uint4 q0 = make_uint4(0, 0, 0, 0), q1 = q0;
      if (k < nact) {
        act_load(k, q0, q1);
        const float x0 = __uint_as_float(q0.x), y0 = __uint_as_float(q0.y);
        const float x1 = __uint_as_float(q0.z), y1 = __uint_as_float(q0.w);
        const uint32_t c = q1.x >> 16, id = q1.x & 0xffffu, w3 = q1.y, hab = q1.z, mask = q1.w;
        const uint32_t mb = __ffs(mask) - 1u, ma = __ffs(mask & (mask - 1u)) - 1u;
        const uint32_t gap = ma - mb - 1u, pend0 = mb - s;
        float tz;
        if ((gap | pend0) <= 1u) tz = tzt[mb * 4u + gap * 2u + pend0];        // the same quotient, taken once per CTA
        else { const float z1 = mz[mb], z0 = mz[ma]; tz = __fdiv_rn(__fsub_rn(z2, z1), __fsub_rn(z1, z0)); }
        const float px = __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, x0), tz));
        const float py = __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, y0), tz));
        const Win wx = make_win(c, Wfwd);
        uint32_t best = kNone; float best_sc = fwd_bound;
        auto visit = [&](uint32_t jj, const uint4& r, bool in) {
          const float ex = __fsub_rn(px, __uint_as_float(r.x)), ey = __fsub_rn(py, __uint_as_float(r.y));
          const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
          bool ok = in & (sc < best_sc);
          if (!kSameW) ok &= (r.z - wx.lo16 <= wx.lim);
          best = ok ? jj : best; best_sc = ok ? sc : best_sc;
        };
        const uint32_t pend = mb - s;      // modules already missed since the latest hit
        if (pend <= 1u) {
          const Win ww = kSameW ? wx : make_win(c, Wwide);
          if (ww.wrapped) scan_run<false>(ring_u, 0u, nu, ww.lo16, ww.lim, visit);          // low-phi run of a window across +-pi
          scan_run<false>(ring_u, pend ? (w3 & 0xffffu) : (w3 >> 16), nu, ww.lo16, ww.lim, visit);
        } else {
          // no stored start for a target this far from the latest hit (max_skipped >= 2): whole module
          for (uint32_t j = 0; j < nu; ++j) {
            const uint4 r = ring_u[j];
            const float ex = __fsub_rn(px, __uint_as_float(r.x)), ey = __fsub_rn(py, __uint_as_float(r.y));
            const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
            const bool ok = (r.z - wx.lo16 <= wx.lim) & (sc < best_sc);
            best = ok ? j : best; best_sc = ok ? sc : best_sc;
          }
        }
        if (best != kNone) {
          const uint4 r2 = ring_u[best];
          const uint32_t h2 = off_u + best, nh = (uint32_t)__popc(mask);
          rows[id * 32u + nh] = (uint16_t)h2;
          rows_xy[id * kXyStride + nh] = make_float2(__uint_as_float(r2.x), __uint_as_float(r2.y));
          // (B): forwarding never reads flags, so they can be set right away
          if (nh + 1u == 4u) { set_flag(th0[id]); set_flag(hab >> 16); set_flag(hab & 0xffffu); }
          if (nh + 1u >= 4u) set_flag(h2);
          q0 = make_uint4(q0.z, q0.w, r2.x, r2.y);
          q1 = make_uint4((r2.z & 0xffff0000u) | id, r2.w, (hab << 16) | h2, mask | (1u << u));
          alive = true;
        } else {
          alive = (mb - u) <= P.max_skipped;       // consecutive misses so far, this one included
          if (!alive && __popc(mask) > 3) cmeta[id].x = mask;
        }
      }
      uint32_t total;
      const uint32_t pos = team_scan_pred<G>(alive, ts.wsum, team, parity, &total);   // (also: every read of this pass is done)
      if (alive) act_store(wbase + pos, q0, q1);
      wbase += total;
    }
    nact = wbase;
    team_sync<G>(team);                  // flags and the compacted list are visible
    VELO_PH(a.ws.phase_clk, ts, 20);

    // ---- (C) O-8 seeding with centre module s -----------------------------------------------------
    // (C1) the unflagged centre hits, in ascending order (flags are final for this step)
    uint32_t ncl = 0;
    for (uint32_t c0 = 0; c0 < ns; c0 += G) {
      const uint32_t j = c0 + tid;
      const bool open = j < ns && !flagged(off_s + j);
      uint32_t total;
      const uint32_t pos = team_scan_pred<G>(open, ts.wsum, team, parity, &total);
      if (open) cl[ncl + pos] = (uint16_t)j;
      ncl += total;
    }
    team_sync<G>(team);
    VELO_PH(a.ws.phase_clk, ts, 21);
    // (C2) rounds of G unflagged centre hits: best (h0, h2) of a centre under (scatter, h0, h2)
    if (ncl) {
      const float zc0 = mz[s + 1], zc1 = mz[s];
      const float tz = __fdiv_rn(__fsub_rn(z2, zc1), __fsub_rn(zc1, zc0));
      for (uint32_t k0 = 0; k0 < ncl; k0 += (uint32_t)G) {
        const uint32_t k = k0 + tid;
        bool found = false; uint32_t b0 = 0, b2 = 0, j1 = 0; float best_sc = 0.0f;
        uint4 r1 = make_uint4(0, 0, 0, 0);
        bool by_pairs = false;
        {
          // Large events: a centre has tens of h0 candidates and each means a long scan of the h2
          // window, very unevenly over the centres. The round's (centre, h0) pairs are listed in shared
          // memory and dealt out one per lane; a centre's best triplet is the minimum of a 64-bit key
          // (scatter bits, h0, h2): the same lexicographic order, reached in any order.
          unsigned long long* keys = (unsigned long long*)(blk + L_.keys);
          uint32_t* plist = (uint32_t*)(blk + L_.plist);
          uint32_t* npairs = &ts.npairs;
          keys[tid] = ~0ull;
          if (tid == 0) *npairs = 0u;
          team_sync<G>(team);
          if (k < ncl) {
            j1 = cl[k];
            r1 = ring_s[j1];
            const uint32_t c = r1.z >> 16;
            const Win wx = make_win(c, Wseed);
            const Win ww = kSameW ? wx : make_win(c, Wwide);
            for (uint32_t run0 = ww.wrapped ? 0u : 1u; run0 < 2u; ++run0) {
              for (uint32_t j0 = run0 ? (r1.z & 0xffffu) : 0u; j0 < np; ++j0) {
                const uint4 r0 = ring_p[j0];
                if (!(r0.z - ww.lo16 <= ww.lim)) break;
                if (!kSameW && !(r0.z - wx.lo16 <= wx.lim)) continue;
                if (flagged(off_p + j0)) continue;
                const uint32_t slot = atomicAdd(npairs, 1u);
                if (slot < kPairCap) plist[slot] = (tid << 16) | j0;
              }
            }
          }
          team_sync<G>(team);
          const uint32_t T = *npairs;
          by_pairs = T <= kPairCap;        // else: the lane-per-centre search below
          if (by_pairs) {
            for (uint32_t p = tid; p < T; p += G) {
              const uint32_t pr = plist[p], kl = pr >> 16, j0 = pr & 0xffffu;
              const uint4 rc = ring_s[cl[k0 + kl]], r0 = ring_p[j0];
              const float x1 = __uint_as_float(rc.x), y1 = __uint_as_float(rc.y);
              const Win wx = make_win(rc.z >> 16, Wseed);
              const Win ww = kSameW ? wx : make_win(rc.z >> 16, Wwide);
              const float px = __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, __uint_as_float(r0.x)), tz));
              const float py = __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, __uint_as_float(r0.y)), tz));
              uint32_t bb2 = kNone; float bsc = seed_bound;
              auto visit2 = [&](uint32_t jj, const uint4& r, bool in) {
                const float ex = __fsub_rn(px, __uint_as_float(r.x)), ey = __fsub_rn(py, __uint_as_float(r.y));
                const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
                bool ok = in & !flagged(off_u + jj) & (sc < bsc);
                if (!kSameW) ok &= (r.z - wx.lo16 <= wx.lim);
                bb2 = ok ? jj : bb2; bsc = ok ? sc : bsc;
              };
              if (ww.wrapped) scan_run<false>(ring_u, 0u, nu, ww.lo16, ww.lim, visit2);
              scan_run<false>(ring_u, rc.w >> 16, nu, ww.lo16, ww.lim, visit2);
              if (bb2 != kNone) atomicMin(&keys[kl], ((unsigned long long)__float_as_uint(bsc) << 32) | ((unsigned long long)j0 << 16) | bb2);
            }
            team_sync<G>(team);
            const unsigned long long key = keys[tid];
            found = k < ncl && key != ~0ull;
            b0 = (uint32_t)(key >> 16) & 0xffffu; b2 = (uint32_t)key & 0xffffu; best_sc = __uint_as_float((uint32_t)(key >> 32));
          }
        }
        if (!by_pairs && k < ncl) {
          j1 = cl[k];
          r1 = ring_s[j1];
          const float x1 = __uint_as_float(r1.x), y1 = __uint_as_float(r1.y);
          const uint32_t c = r1.z >> 16;
          const Win wx = make_win(c, Wseed);
          const Win ww = kSameW ? wx : make_win(c, Wwide);
          for (uint32_t run0 = ww.wrapped ? 0u : 1u; run0 < 2u; ++run0) {
            for (uint32_t j0 = run0 ? (r1.z & 0xffffu) : 0u; j0 < np; ++j0) {
              const uint4 r0 = ring_p[j0];
              if (!(r0.z - ww.lo16 <= ww.lim)) break;
              if (!kSameW && !(r0.z - wx.lo16 <= wx.lim)) continue;
              if (flagged(off_p + j0)) continue;
              const float px = __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, __uint_as_float(r0.x)), tz));
              const float py = __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, __uint_as_float(r0.y)), tz));
              // h0 and h2 ascending: strict < keeps the lexicographic minimum; branch-free body
              auto visit2 = [&](uint32_t jj, const uint4& r, bool in) {
                const float ex = __fsub_rn(px, __uint_as_float(r.x)), ey = __fsub_rn(py, __uint_as_float(r.y));
                const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
                bool ok = in & !flagged(off_u + jj) & (sc <= max_seed) & (!found | (sc < best_sc));
                if (!kSameW) ok &= (r.z - wx.lo16 <= wx.lim);
                found |= ok; b0 = ok ? j0 : b0; b2 = ok ? jj : b2; best_sc = ok ? sc : best_sc;
              };
              if (ww.wrapped) scan_run<false>(ring_u, 0u, nu, ww.lo16, ww.lim, visit2);
              scan_run<false>(ring_u, r1.w >> 16, nu, ww.lo16, ww.lim, visit2);
            }
          }
        }
        uint32_t total;
        const uint32_t pos = team_scan_pred<G>(found, ts.wsum, team, parity, &total);
        if (found && ncand + pos < tcap) {
          const uint32_t id = ncand + pos;
          const uint32_t h0 = off_p + b0, h1 = off_s + j1, h2 = off_u + b2;
          const uint4 r2 = ring_u[b2];
          *reinterpret_cast<uint2*>(rows + id * 32u) = make_uint2(h0 | (h1 << 16), h2);
          const uint4 r0 = ring_p[b0];
          float4* rxy = reinterpret_cast<float4*>(rows_xy + id * kXyStride);
          rxy[0] = make_float4(__uint_as_float(r0.x), __uint_as_float(r0.y), __uint_as_float(r1.x), __uint_as_float(r1.y));
          rows_xy[id * kXyStride + 2u] = make_float2(__uint_as_float(r2.x), __uint_as_float(r2.y));
          cmeta[id] = make_uint2(7u << u, __float_as_uint(best_sc));
          th0[id] = (uint16_t)h0;
          act_store(nact + pos, make_uint4(r1.x, r1.y, r2.x, r2.y),
                    make_uint4((r2.z & 0xffff0000u) | id, r2.w, (h1 << 16) | h2, 7u << u));
        }
        ncand += total; nact += total;
      }
    }
    if (ncand > tcap) { if (tid == 0) ts.defer = 1; }
    team_sync<G>(team);                  // the new tracks are visible
    VELO_PH(a.ws.phase_clk, ts, 22);
    if (ts.defer) break;
  }
  if (ts.defer) {
    if (tid == 0) {
      a.ws.ev_info[e].state = kEvDeferred;
      a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
    }
    return;
  }
  // tracks still active take their final module mask; the final flags leave as bits
  for (uint32_t k = tid; k < nact; k += G) {
    uint4 q0, q1;
    act_load(k, q0, q1);
    if (__popc(q1.w) > 3) cmeta[q1.x & 0xffffu].x = q1.w;
  }
  {
    uint32_t* fb = a.ws.flag_bits + ((a.event_offsets[e] - a.event_offsets[0]) >> 5) + e;
    for (uint32_t i = tid; i < ((n + 31u) >> 5); i += G) fb[i] = flags[i];
  }
  if (tid == 0) {
    a.ws.ev_info[e] = EvInfo{n, kEvBig, ts.cbase, ncand};
    atomicAdd(&a.ws.counters[kCtrCand], ncand);
  }
}

// ---- one event, by one team whose warps work side by side ------------------------------------------
// The same step semantics as track_event (the form the one-event-per-CTA kernel keeps), dealt out so
// that the warps of a team meet twice per step instead of after every pass:
//   * every warp owns a share of the active-track list (the tracks it seeded): forwarding, the
//     compaction of its share (ballot) and the appends never leave the warp;
//   * every warp owns a contiguous share of the centre module's positions: it lists its unflagged
//     centres and searches their triplets on its own, parking what it finds where the new tracks'
//     records will be (the tail of its share of the list);
//   * barrier 1 follows forwarding (the flags of the step are final), barrier 2 follows the search:
//     the warps exchange how many seeds each found, which fixes the candidate ids in the order B1
//     (centre position ascending: warp 0's share precedes warp 1's), then each warp writes its own.
// kTwoPlane (DESIGN.md §2 L-1: two sensor planes per module): bit 15 of a record's last word says which
// plane the hit lies on, O-4's z ratio is taken per candidate plane, bits 31 and 30 of an active track's
// module mask hold the planes of its latest and previous hit, and the planes of all its hits leave in
// the last entry of its coordinate row (kSideSlot) for the fit.
template <int G, bool kSameW, bool kTwoPlane>
__device__ void track_event_w(const KernelArgs& a, const float* mz, const float* mzb, const float* tzt, TrackTeam<G>& ts,
                              unsigned char* blk, uint32_t team, uint32_t tid, uint32_t& phases) {
  constexpr uint32_t kMaskBits = kTwoPlane ? 0x3fffffffu : 0xffffffffu;
  constexpr uint32_t kStartBits = kTwoPlane ? 0x7fffu : 0xffffu;
  auto plane_of = [](const uint4& r) -> uint32_t { return (r.w >> 15) & 1u; };
  constexpr uint32_t W = G / 32;
  const uint32_t lane = tid & 31u, w = tid >> 5, lt = (1u << lane) - 1u;
  const uint32_t M = a.n_modules, n = ts.n, e = ts.event;
  const velo_params_t& P = a.P;
  const uint32_t tcap = ts.tcap, acap_w = ts.acap / W, ovf_w = tcap / W;
  const TrackLayout L = track_layout(n, ts.maxmod, tcap, ts.acap);
  const uint32_t slotcap = ts.maxmod + kSlotPad;
  uint4* ring = (uint4*)(blk + L.ring);
  uint4* act = (uint4*)(blk + L.act) + 2u * w * acap_w;       // this warp's share
  uint32_t* flags = (uint32_t*)(blk + L.flags);               // one bit per sorted hit
  auto flagged = [&](uint32_t h) -> bool { return (flags[h >> 5] >> (h & 31u)) & 1u; };
  auto set_flag = [&](uint32_t h) { atomicOr(&flags[h >> 5], 1u << (h & 31u)); };
  // beyond the shared-memory share: global scratch (stage 3's state planes, unused until stage 3)
  uint4* act_ovf = reinterpret_cast<uint4*>(a.ws.cfit) + 2u * ((size_t)ts.cbase + (size_t)w * ovf_w);
  auto act_load = [&](uint32_t k, uint4& q0, uint4& q1) {
    if (k < acap_w) { q0 = act[k]; q1 = act[acap_w + k]; }      // two planes of 16-byte halves: a warp's loads meet no bank twice
    else if (k - acap_w < ovf_w) { q0 = __ldcg(act_ovf + 2u * (k - acap_w)); q1 = __ldcg(act_ovf + 2u * (k - acap_w) + 1u); }
    else { q0 = make_uint4(0, 0, 0, 0); q1 = q0; }      // never stored (act_store): the event is being given up
  };
  auto act_store = [&](uint32_t k, const uint4& q0, const uint4& q1) {
    if (k < acap_w) { act[k] = q0; act[acap_w + k] = q1; }
    else if (k - acap_w < ovf_w) { act_ovf[2u * (k - acap_w)] = q0; act_ovf[2u * (k - acap_w) + 1u] = q1; }
    else ts.defer = 1;                 // a share this lopsided: the general kernel takes the event
  };
  uint16_t* th0 = (uint16_t*)(blk + L.th0);
  uint16_t* cl = (uint16_t*)(blk + L.cl);
  const uint16_t* mo = ts.mod_off;
  const uint4* grec = a.ws.rec16 + ts.sb;
  uint16_t* rows = a.ws.rows + (size_t)ts.cbase * 32u;
  uint2* cmeta = a.ws.cmeta + ts.cbase;
  float2* rows_xy = a.ws.rows_xy + (size_t)ts.cbase * kXyStride;
  const int Wseed = P.phi_window_seed, Wfwd = P.phi_window_fwd;
  const int Wwide = Wseed > Wfwd ? Wseed : Wfwd;

  for (uint32_t i = tid; i < kModOffStride; i += G) ts.mod_off[i] = a.ws.mod_off[(size_t)e * kModOffStride + i];
  for (uint32_t i = tid; i < ((n + 31u + kSlotPad) >> 5); i += G) flags[i] = 0;
  team_sync<G>(team);

  // ring: module m lives in slot m & 3; loads are issued and waited for in descending module order
  auto issue = [&](uint32_t m) {
    if (tid == 0) {
      const uint32_t bytes = 16u * ((uint32_t)mo[m + 1] - (uint32_t)mo[m]);
      mbar_arrive_expect_tx(&ts.mbar[m & 3u], bytes);
      if (bytes) tma_load_1d(ring + (m & 3u) * slotcap, grec + mo[m], bytes, &ts.mbar[m & 3u]);
      uint4* pad = ring + (m & 3u) * slotcap + (bytes >> 4);    // the sentinels behind the records (scan_run)
#pragma unroll
      for (uint32_t k = 0; k < kSlotPad; ++k) pad[k] = make_uint4(0x7f800000u, 0u, 0u, 0u);
    }
  };
  auto wait = [&](uint32_t m) {
    mbar_wait(&ts.mbar[m & 3u], (phases >> (m & 3u)) & 1u);
    phases ^= 1u << (m & 3u);
  };
  uint32_t issued = M, waited = M;       // lowest module issued / waited for so far
  for (uint32_t k = 0; k < 4 && issued > 0; ++k) issue(--issued);
  wait(--waited); wait(--waited);        // modules M-1 and M-2
  VELO_PH(a.ws.phase_clk, ts, 18);       // descriptors, flags, first loads

  uint32_t nact = 0, ncand = 0;          // nact: this warp's share
  // "scatter <= max and below the best so far" is kept as one comparison, scatter < bound, with the bound starting
  // at the next float above max (the cuts are finite here: velo_api.cu sends any other cut through the general
  // kernel); a match is found iff an index was taken. Ties still go to the first record met (strict <).
  const float fwd_bound = nextafterf(P.max_scatter_fwd, INFINITY), seed_bound = nextafterf(P.max_scatter_seed, INFINITY);
  constexpr uint32_t kNone = 0xffffffffu;
  for (uint32_t s = M - 2; s >= 1; --s) {
    const uint32_t u = s - 1;
    if (mo[u + 1] == 0) break;           // no hit in modules 0 .. u: nothing can change any more (see track_event)
    wait(--waited);                      // module u has landed
    VELO_PH(a.ws.phase_clk, ts, 19);
    const uint32_t off_u = mo[u], nu = (uint32_t)mo[u + 1] - off_u;
    const uint32_t off_s = mo[s], ns = (uint32_t)mo[s + 1] - off_s;
    const uint32_t off_p = mo[s + 1], np = (uint32_t)mo[s + 2] - off_p;
    const uint4* ring_u = ring + (u & 3u) * slotcap;
    const uint4* ring_s = ring + (s & 3u) * slotcap;
    const uint4* ring_p = ring + ((s + 1u) & 3u) * slotcap;
    const float z2 = mz[u];

    // ---- (A) O-7 forwarding into module u of this warp's share of the active tracks ----------------
    uint32_t wbase = 0;
    for (uint32_t p0 = 0; p0 < nact; p0 += 32u) {
      const uint32_t k = p0 + lane;
      bool alive = false;
      uint4 q0 = make_uint4(0, 0, 0, 0), q1 = q0;
      if (k < nact) {
        act_load(k, q0, q1);
        const float x0 = __uint_as_float(q0.x), y0 = __uint_as_float(q0.y);
        const float x1 = __uint_as_float(q0.z), y1 = __uint_as_float(q0.w);
        const uint32_t c = q1.x >> 16, id = q1.x & 0xffffu, w3 = q1.y, hab = q1.z, mask = q1.w & kMaskBits;
        const uint32_t mb = __ffs(mask) - 1u, ma = __ffs(mask & (mask - 1u)) - 1u;
        const uint32_t gap = ma - mb - 1u, pend = mb - s;     // pend: modules already missed since the latest hit
        float tz, px_b = 0.0f, py_b = 0.0f;                   // (px_b, py_b): the prediction on the module's second plane
        if constexpr (kTwoPlane) {
          const float z1 = (q1.w >> 31) ? mzb[mb] : mz[mb], z0 = ((q1.w >> 30) & 1u) ? mzb[ma] : mz[ma];
          const float den = __fsub_rn(z1, z0);
          tz = __fdiv_rn(__fsub_rn(z2, z1), den);
          const float tzb = __fdiv_rn(__fsub_rn(mzb[u], z1), den);
          px_b = __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, x0), tzb));
          py_b = __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, y0), tzb));
        } else if ((gap | pend) <= 1u) tz = tzt[mb * 4u + gap * 2u + pend];        // the same quotient, taken once per CTA
        else { const float z1 = mz[mb], z0 = mz[ma]; tz = __fdiv_rn(__fsub_rn(z2, z1), __fsub_rn(z1, z0)); }
        const float px = __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, x0), tz));
        const float py = __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, y0), tz));
        const Win wx = make_win(c, Wfwd);
        uint32_t best = kNone; float best_sc = fwd_bound;
        auto visit = [&](uint32_t jj, const uint4& r, bool in) {
          const bool pb = kTwoPlane && plane_of(r) != 0u;
          const float ex = __fsub_rn(pb ? px_b : px, __uint_as_float(r.x)), ey = __fsub_rn(pb ? py_b : py, __uint_as_float(r.y));
          const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
          bool ok = in & (sc < best_sc);
          if (!kSameW) ok &= (r.z - wx.lo16 <= wx.lim);
          best = ok ? jj : best; best_sc = ok ? sc : best_sc;
        };
        if (pend <= 1u) {
          const Win ww = kSameW ? wx : make_win(c, Wwide);
          if (ww.wrapped) scan_run<true>(ring_u, 0u, nu, ww.lo16, ww.lim, visit);          // low-phi run of a window across +-pi
          scan_run<true>(ring_u, pend ? (w3 & kStartBits) : (w3 >> 16), nu, ww.lo16, ww.lim, visit);
        } else {
          // no stored start for a target this far from the latest hit (max_skipped >= 2): whole module
          for (uint32_t j = 0; j < nu; ++j) {
            const uint4 r = ring_u[j];
            const bool pb = kTwoPlane && plane_of(r) != 0u;
            const float ex = __fsub_rn(pb ? px_b : px, __uint_as_float(r.x)), ey = __fsub_rn(pb ? py_b : py, __uint_as_float(r.y));
            const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
            const bool ok = (r.z - wx.lo16 <= wx.lim) & (sc < best_sc);
            best = ok ? j : best; best_sc = ok ? sc : best_sc;
          }
        }
        if (best != kNone) {
          const uint4 r2 = ring_u[best];
          const uint32_t h2 = off_u + best, nh = (uint32_t)__popc(mask);
          rows[id * 32u + nh] = (uint16_t)h2;
          rows_xy[id * kXyStride + nh] = make_float2(__uint_as_float(r2.x), __uint_as_float(r2.y));
          // (B): forwarding never reads flags, so they can be set right away
          if (nh + 1u == 4u) { set_flag(th0[id]); set_flag(hab >> 16); set_flag(hab & 0xffffu); }
          if (nh + 1u >= 4u) set_flag(h2);
          q0 = make_uint4(q0.z, q0.w, r2.x, r2.y);
          uint32_t nmask = mask | (1u << u);
          if constexpr (kTwoPlane) {
            const uint32_t p2 = plane_of(r2);
            nmask |= (p2 << 31) | ((q1.w >> 31) << 30);
            if (p2) atomicOr(reinterpret_cast<uint32_t*>(rows_xy + id * kXyStride + kSideSlot), 1u << u);
          }
          q1 = make_uint4((r2.z & 0xffff0000u) | id, r2.w, (hab << 16) | h2, nmask);
          alive = true;
        } else {
          alive = (mb - u) <= P.max_skipped;       // consecutive misses so far, this one included
          if (!alive && __popc(mask) > 3) cmeta[id].x = mask;
        }
      }
      const uint32_t b = __ballot_sync(0xffffffffu, alive);      // (also: every read of this pass is done)
      if (alive) act_store(wbase + (uint32_t)__popc(b & lt), q0, q1);
      wbase += (uint32_t)__popc(b);
    }
    nact = wbase;
    team_sync<G>(team);                  // barrier 1: the flags of this step are final
    VELO_PH(a.ws.phase_clk, ts, 20);
    if (ts.defer) break;                 // set before the barrier by a warp whose share overflowed: every warp sees it here

    // ---- (C) O-8 seeding with centre module s: this warp's share of the module's positions ----------
    const uint32_t c_lo = (w * ns) / W, c_hi = ((w + 1u) * ns) / W;
    uint16_t* clw = cl + c_lo;           // at most c_hi - c_lo entries: the share's unflagged centres
    // (C1) the unflagged centre hits, in ascending order
    uint32_t ncl = 0;
    for (uint32_t c0 = c_lo; c0 < c_hi; c0 += 32u) {
      const uint32_t j = c0 + lane;
      const bool open = j < c_hi && !flagged(off_s + j);
      const uint32_t b = __ballot_sync(0xffffffffu, open);
      if (open) clw[ncl + (uint32_t)__popc(b & lt)] = (uint16_t)j;
      ncl += (uint32_t)__popc(b);
    }
    __syncwarp();
    VELO_PH(a.ws.phase_clk, ts, 21);
    // (C2) L = 1, 2 or 4 adjacent lanes per centre (as many as the warp can seat at once), lane q taking
    // every L-th h0 of the window: best (h0, h2) under (scatter, h0, h2), reduced over the L lanes with
    // shuffles under the same lexicographic order
    uint32_t nfound = 0;
    if (ncl) {
      const float zc0 = mz[s + 1], zc1 = mz[s];
      const float tz = __fdiv_rn(__fsub_rn(z2, zc1), __fsub_rn(zc1, zc0));
      const uint32_t lsh = (4u * ncl <= 32u) ? 2u : (2u * ncl <= 32u) ? 1u : 0u;
      const uint32_t Ls = 1u << lsh;
      for (uint32_t k0 = 0; k0 < ncl; k0 += 32u >> lsh) {
        const uint32_t k = k0 + (lane >> lsh), q = lane & (Ls - 1u);
        uint32_t b0 = kNone, b2 = 0, j1 = 0; float best_sc = seed_bound;
        if (k < ncl) {
          j1 = clw[k];
          const uint4 r1 = ring_s[j1];
          const float x1 = __uint_as_float(r1.x), y1 = __uint_as_float(r1.y);
          const float z1c = (kTwoPlane && plane_of(r1)) ? mzb[s] : zc1;
          const uint32_t c = r1.z >> 16;
          const Win wx = make_win(c, Wseed);
          const Win ww = kSameW ? wx : make_win(c, Wwide);
          for (uint32_t run0 = ww.wrapped ? 0u : 1u; run0 < 2u; ++run0) {
            for (uint32_t j0 = (run0 ? (r1.z & 0xffffu) : 0u) + q; j0 < np; j0 += Ls) {
              const uint4 r0 = ring_p[j0];
              if (!(r0.z - ww.lo16 <= ww.lim)) break;
              if (!kSameW && !(r0.z - wx.lo16 <= wx.lim)) continue;
              if (flagged(off_p + j0)) continue;
              float tza = tz, tzb = 0.0f;
              if constexpr (kTwoPlane) {
                const float den = __fsub_rn(z1c, plane_of(r0) ? mzb[s + 1] : zc0);
                tza = __fdiv_rn(__fsub_rn(z2, z1c), den); tzb = __fdiv_rn(__fsub_rn(mzb[u], z1c), den);
              }
              const float px = __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, __uint_as_float(r0.x)), tza));
              const float py = __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, __uint_as_float(r0.y)), tza));
              const float px_b = kTwoPlane ? __fadd_rn(x1, __fmul_rn(__fsub_rn(x1, __uint_as_float(r0.x)), tzb)) : 0.0f;
              const float py_b = kTwoPlane ? __fadd_rn(y1, __fmul_rn(__fsub_rn(y1, __uint_as_float(r0.y)), tzb)) : 0.0f;
              // h0 and h2 ascending: strict < keeps the lexicographic minimum; branch-free body
              auto visit2 = [&](uint32_t jj, const uint4& r, bool in) {
                const bool pb = kTwoPlane && plane_of(r) != 0u;
                const float ex = __fsub_rn(pb ? px_b : px, __uint_as_float(r.x)), ey = __fsub_rn(pb ? py_b : py, __uint_as_float(r.y));
                const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
                bool ok = in & !flagged(off_u + jj) & (sc < best_sc);
                if (!kSameW) ok &= (r.z - wx.lo16 <= wx.lim);
                b0 = ok ? j0 : b0; b2 = ok ? jj : b2; best_sc = ok ? sc : best_sc;
              };
              if (ww.wrapped) scan_run<true>(ring_u, 0u, nu, ww.lo16, ww.lim, visit2);
              scan_run<true>(ring_u, r1.w >> 16, nu, ww.lo16, ww.lim, visit2);
            }
          }
        }
        bool found = b0 != kNone;
        for (uint32_t d = 1; d < Ls; d <<= 1) {
          const bool o_found = __shfl_xor_sync(0xffffffffu, (int)found, d) != 0;
          const float o_sc = __shfl_xor_sync(0xffffffffu, best_sc, d);
          const uint32_t o_b0 = __shfl_xor_sync(0xffffffffu, b0, d), o_b2 = __shfl_xor_sync(0xffffffffu, b2, d);
          const bool better = o_found & (!found | (o_sc < best_sc) |
                                         ((o_sc == best_sc) & ((o_b0 < b0) | ((o_b0 == b0) & (o_b2 < b2)))));
          found |= o_found; b0 = better ? o_b0 : b0; b2 = better ? o_b2 : b2; best_sc = better ? o_sc : best_sc;
        }
        found &= (q == 0u);                // one lane speaks for the centre
        const uint32_t b = __ballot_sync(0xffffffffu, found);
        if (found) {
          // parked where the new track's record will be: {x, y of h0, h0 << 16 | h2 (positions), scatter | centre}
          const uint4 r0 = ring_p[b0];
          act_store(nact + nfound + (uint32_t)__popc(b & lt), make_uint4(r0.x, r0.y, (b0 << 16) | b2, __float_as_uint(best_sc)),
                    make_uint4(j1, plane_of(r0), 0u, 0u));
        }
        nfound += (uint32_t)__popc(b);
      }
    }
    if (W > 1 && lane == 0) ts.wsum[w] = nfound;
    team_sync<G>(team);                  // barrier 2: every search is done (module s+1 has been read for the last
                                         // time); how many seeds each warp found fixes the candidate ids
    uint32_t base = ncand, total = nfound;
    if (W > 1) {
      total = 0;
#pragma unroll
      for (uint32_t k = 0; k < W; ++k) { const uint32_t c = ts.wsum[k]; if (k < w) base += c; total += c; }
    }
    if (issued > 0) issue(--issued);     // module s-3 into the slot of module s+1
    for (uint32_t f = lane; f < nfound; f += 32u) {
      const uint32_t id = base + f;
      if (id < tcap) {
        uint4 sb4, sb1;
        act_load(nact + f, sb4, sb1);
        const uint32_t j1 = sb1.x, b0 = sb4.z >> 16, b2 = sb4.z & 0xffffu;
        const uint32_t h0 = off_p + b0, h1 = off_s + j1, h2 = off_u + b2;
        const uint4 r1 = ring_s[j1], r2 = ring_u[b2];
        *reinterpret_cast<uint2*>(rows + id * 32u) = make_uint2(h0 | (h1 << 16), h2);
        float4* rxy = reinterpret_cast<float4*>(rows_xy + id * kXyStride);
        rxy[0] = make_float4(__uint_as_float(sb4.x), __uint_as_float(sb4.y), __uint_as_float(r1.x), __uint_as_float(r1.y));
        rows_xy[id * kXyStride + 2u] = make_float2(__uint_as_float(r2.x), __uint_as_float(r2.y));
        cmeta[id] = make_uint2(7u << u, sb4.w);
        th0[id] = (uint16_t)h0;
        uint32_t nmask = 7u << u;
        if constexpr (kTwoPlane) {
          const uint32_t p0 = sb1.y, p1 = plane_of(r1), p2 = plane_of(r2);
          nmask |= (p2 << 31) | (p1 << 30);
          rows_xy[id * kXyStride + kSideSlot] = make_float2(__uint_as_float((p0 << (s + 1u)) | (p1 << s) | (p2 << u)), 0.0f);
        }
        act_store(nact + f, make_uint4(r1.x, r1.y, r2.x, r2.y),
                  make_uint4((r2.z & 0xffff0000u) | id, r2.w, (h1 << 16) | h2, nmask));
      }
    }
    nact += nfound; ncand += total;
    __syncwarp();                        // the appended records and th0 are visible to the warp's other lanes
    VELO_PH(a.ws.phase_clk, ts, 22);
    if (ncand > tcap) { if (tid == 0) ts.defer = 1; break; }     // the same for every warp
  }
  // every load that was issued must land before the block can be freed
  while (waited > issued) wait(--waited);
  team_sync<G>(team);                    // a share that overflowed in the last step's appends is seen by every warp
  if (ts.defer) {
    if (tid == 0) {
      a.ws.ev_info[e].state = kEvDeferred;
      a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
    }
    return;
  }
  // tracks still active take their final module mask; the final flags leave as bits
  for (uint32_t k = lane; k < nact; k += 32u) {
    uint4 q0, q1;
    act_load(k, q0, q1);
    if (__popc(q1.w & kMaskBits) > 3) cmeta[q1.x & 0xffffu].x = q1.w & kMaskBits;
  }
  {
    uint32_t* fb = a.ws.flag_bits + ((a.event_offsets[e] - a.event_offsets[0]) >> 5) + e;
    for (uint32_t i = tid; i < ((n + 31u) >> 5); i += G) fb[i] = flags[i];
  }
  if (tid == 0) {
    a.ws.ev_info[e] = EvInfo{n, kEvReady, ts.cbase, ncand};
    atomicAdd(&a.ws.counters[kCtrCand], ncand);
  }
}

// ---- the kernel: one CTA per SM, kTeams teams of G threads ---------------------------------------
template <int G, int kTeams, bool kSameW, bool kTwoPlane>
__global__ void __launch_bounds__(G * kTeams, 1) velo_track_kernel(const KernelArgs a, const uint32_t pool_units) {
  extern __shared__ __align__(16) unsigned char smem[];
  using Ctl = TrackCtl<G, kTeams>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  Ctl& ctl = *reinterpret_cast<Ctl*>(smem);
  unsigned char* pool = smem + kCtl;
  const uint32_t team = threadIdx.x / G, tid = threadIdx.x % G;
  if (threadIdx.x == 0) pool_init(ctl.pool, pool_units);
  if (threadIdx.x < VELO_MAX_MODULES) { ctl.module_z[threadIdx.x] = a.module_z[threadIdx.x]; ctl.module_z_b[threadIdx.x] = a.module_z_b[threadIdx.x]; }
  if (threadIdx.x < VELO_MAX_MODULES * 4u) {
    const uint32_t mb = threadIdx.x >> 2, gap = (threadIdx.x >> 1) & 1u, pend = threadIdx.x & 1u, ma = mb + 1u + gap;
    float v = 0.0f;
    if (ma < a.n_modules && mb >= 1u + pend)
      v = __fdiv_rn(__fsub_rn(a.module_z[mb - 1u - pend], a.module_z[mb]), __fsub_rn(a.module_z[mb], a.module_z[ma]));
    ctl.tz[threadIdx.x] = v;
  }
  TrackTeam<G>& ts = ctl.team[team];
  if (tid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) mbar_init(&ts.mbar[k], 1u);
    mbar_fence_init();
  }
  __syncthreads();
  VELO_STAGE_BEGIN(a.ws.phase_clk, 1);
  uint32_t phases = 0;
  VELO_PH_START(ts);
  for (;;) {
    if (tid == 0) track_fetch<G>(a, ctl.pool, ts);
    team_sync<G>(team);
    if (ts.event >= a.n_events) break;
    VELO_PH(a.ws.phase_clk, ts, 17);     // ticket, descriptors, pool
    if (!ts.skip) track_event_w<G, kSameW, kTwoPlane>(a, ctl.module_z, ctl.module_z_b, ctl.tz, ts, pool + ts.pool_off, team, tid, phases);
    if (a.pixel && (ts.unpack || (!ts.skip && ts.defer))) unpack_event<G>(a, ts.event, tid);
    team_sync<G>(team);   // every thread is done with the block and with ts before the leader reuses them
    if (tid == 0 && ts.units) pool_free(ctl.pool, ts.first_unit, ts.units);
    VELO_PH(a.ws.phase_clk, ts, 23);     // tail: remaining loads, masks, flag bits
    VELO_PH_COUNT(a.ws.phase_clk, 16, 1);
  }
  VELO_STAGE_END(a.ws.phase_clk, 1);
}

// ---- the same stage for the events of ws.big_list: one CTA of G threads per event ------------------
template <int G, bool kSameW>
__global__ void __launch_bounds__(G, 1) velo_track_big_kernel(const KernelArgs a, const uint32_t smem_bytes) {
  extern __shared__ __align__(16) unsigned char smem[];
  using Ctl = TrackCtl<G, 1>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  Ctl& ctl = *reinterpret_cast<Ctl*>(smem);
  unsigned char* blk = smem + kCtl;
  const uint32_t tid = threadIdx.x;
  if (tid < VELO_MAX_MODULES) ctl.module_z[tid] = a.module_z[tid];
  if (threadIdx.x < VELO_MAX_MODULES * 4u) {
    const uint32_t mb = threadIdx.x >> 2, gap = (threadIdx.x >> 1) & 1u, pend = threadIdx.x & 1u, ma = mb + 1u + gap;
    float v = 0.0f;
    if (ma < a.n_modules && mb >= 1u + pend)
      v = __fdiv_rn(__fsub_rn(a.module_z[mb - 1u - pend], a.module_z[mb]), __fsub_rn(a.module_z[mb], a.module_z[ma]));
    ctl.tz[threadIdx.x] = v;
  }
  TrackTeam<G>& ts = ctl.team[0];
  uint32_t parity = 0;
  const uint32_t base = a.event_offsets[0];
  for (;;) {
    __syncthreads();
    if (tid == 0) {
      const uint32_t k = atomicAdd(&a.ws.counters[kCtrBigTrackTicket], 1u);
      ts.units = k >= a.ws.counters[kCtrBigN];      // 1 = no more events
      ts.skip = 1; ts.defer = 0; ts.unpack = 0;
      if (!ts.units) {
        const uint32_t e = a.ws.big_sorted[k];
        const EvInfo info = a.ws.ev_info[e];
        ts.event = e;
        if (info.state == kEvBig) {                  // else: stage 1 gave it to the general kernel
          const uint32_t n = info.n, maxmod = a.ws.mod_off[(size_t)e * kModOffStride + kModOffStride - 1];
          const uint32_t tcap = cand_capacity(n), acap = active_capacity(n);
          if (track_layout(n, maxmod, tcap, acap, false).bytes > smem_bytes - kCtl) {
            a.ws.ev_info[e].state = kEvDeferred;
            a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
            ts.unpack = a.pixel != nullptr;
          } else {
            ts.cbase = atomicAdd(&a.ws.counters[kCtrCandAlloc], tcap);
            ts.n = n; ts.sb = sorted_base(a.event_offsets[e] - base, e);
            ts.maxmod = maxmod; ts.tcap = tcap; ts.acap = acap; ts.skip = 0;
          }
        }
      }
    }
    __syncthreads();
    if (ts.units) break;
    if (!ts.skip) track_event_big<G, kSameW>(a, ctl.module_z, ctl.tz, ts, blk, 0u, tid, parity);
    if (a.pixel && (ts.unpack || (!ts.skip && ts.defer))) unpack_event<G>(a, ts.event, tid);
  }
}

template <int G>
int launch_track_big_t(const KernelArgs& a, cudaStream_t stream) {
  const uint32_t smem = 227u * 1024u;
  const bool same = a.P.phi_window_seed == a.P.phi_window_fwd;
  const uint32_t grid = num_sms();
  cudaError_t err;
  if (same) {
    err = cudaFuncSetAttribute(velo_track_big_kernel<G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return (int)err;
    velo_track_big_kernel<G, true><<<grid, G, smem, stream>>>(a, smem);
  } else {
    err = cudaFuncSetAttribute(velo_track_big_kernel<G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return (int)err;
    velo_track_big_kernel<G, false><<<grid, G, smem, stream>>>(a, smem);
  }
  return (int)cudaGetLastError();
}

template <int G, int kTeams, bool kSameW, bool kTwoPlane>
int launch_track_k(const KernelArgs& a, cudaStream_t stream, uint32_t pool_units) {
  static_assert(G == 32 || kTeams <= 15, "named barriers 1..15");
  using Ctl = TrackCtl<G, kTeams>;
  constexpr uint32_t kCtl = (sizeof(Ctl) + 127u) & ~127u;
  const uint32_t smem = kCtl + pool_units * kUnitBytes;
  const uint32_t sms = num_sms();
  const uint32_t want = (a.n_events + kTeams - 1) / kTeams;
  const uint32_t grid = want < sms ? (want ? want : 1u) : sms;
  auto* kern = velo_track_kernel<G, kTeams, kSameW, kTwoPlane>;
  const cudaError_t err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err != cudaSuccess) return (int)err;
  kern<<<grid, G * kTeams, smem, stream>>>(a, pool_units);
  return (int)cudaGetLastError();
}

template <int G, int kTeams>
int launch_track_t(const KernelArgs& a, cudaStream_t stream, uint32_t pool_units) {
  const bool same = a.P.phi_window_seed == a.P.phi_window_fwd;
  return same ? launch_track_k<G, kTeams, true, false>(a, stream, pool_units)
              : launch_track_k<G, kTeams, false, false>(a, stream, pool_units);
}

// Two sensor planes per module (L-1): the default team shapes only.
template <int G, int kTeams>
int launch_track_2p(const KernelArgs& a, cudaStream_t stream, uint32_t pool_units) {
  const bool same = a.P.phi_window_seed == a.P.phi_window_fwd;
  return same ? launch_track_k<G, kTeams, true, true>(a, stream, pool_units)
              : launch_track_k<G, kTeams, false, true>(a, stream, pool_units);
}

}  // namespace

int launch_track_big(const KernelArgs& a, cudaStream_t stream) { return launch_track_big_t<768>(a, stream); }

int launch_track(const KernelArgs& a, cudaStream_t stream, const PipeOpts& o) {
  const uint32_t pu = o.pool_units ? (o.pool_units > kPoolUnitsMax ? kPoolUnitsMax : o.pool_units) : kPoolUnitsMax;
  uint32_t g = o.track_group, t = o.track_teams;
  if (g == 0) {
    // two warps per event for mu = 5 sized events; more threads per event when the events are large
    const uint32_t mean = a.n_events ? a.n_hits / a.n_events : 0u;
    g = mean >= 6144u ? 128u : mean < 768u ? 32u : 64u;
    if (g == 32u && t == 0) t = 24;            // small events (open VELO): a warp per event, 24 in flight
  }
  if (a.two_plane) {
    if (g == 128) return launch_track_2p<128, 6>(a, stream, pu);
    if (g == 64) return launch_track_2p<64, 12>(a, stream, pu);
    return launch_track_2p<32, 24>(a, stream, pu);
  }
  if (g == 128) {
    if (t == 0) t = 6;
    switch (t) {
      case 4: return launch_track_t<128, 4>(a, stream, pu);
      case 8: return launch_track_t<128, 8>(a, stream, pu);
      default: return launch_track_t<128, 6>(a, stream, pu);
    }
  }
  if (g == 64) {
    if (t == 0) t = 12;
    switch (t) {
      case 8: return launch_track_t<64, 8>(a, stream, pu);
      case 15: return launch_track_t<64, 15>(a, stream, pu);
      default: return launch_track_t<64, 12>(a, stream, pu);
    }
  }
  if (t == 0) t = 16;
  switch (t) {
    case 8: return launch_track_t<32, 8>(a, stream, pu);
    case 12: return launch_track_t<32, 12>(a, stream, pu);
    case 20: return launch_track_t<32, 20>(a, stream, pu);
    case 24: return launch_track_t<32, 24>(a, stream, pu);
    default: return launch_track_t<32, 16>(a, stream, pu);
  }
}

}  // namespace velo
