// velo_event_smem.cu — the shared-memory event kernel of the VELO hot path (sm_100a).
//
// One persistent CTA per SM owns the SM's shared memory as a pool of 4 KB units. The CTA is cut
// into teams of 128 threads; a team takes the next event from a global ticket, allocates from the
// pool exactly what that event needs (events span 0 ... ~6 k hits at mu = 5, so a fixed slot per
// event would waste more than half of the SM), and runs the whole per-event path there: S0 decode
// (phi16), S1 phi sort, the module loop with S3 forwarding and S2 search-by-triplet seeding, S4
// ghost filter, S5 fit, S6 clone filter, and the staging of its tracks for S7. Teams synchronise
// with named barriers (bar.sync id, 128), never with the whole CTA, so ~5 independent events are
// in flight per SM and hide each other's shared-memory and barrier latency.
//
// Shared memory holds what the module loop touches at random: 12 bytes per hit (x, y, one packed
// word), the phi-bucket table and 21 bytes per candidate track. The candidates' hit lists (written
// once per appended hit, read back only after the loop) and fitted states live in a per-team
// scratch in global memory that stays L2-resident. Smaller blocks = more events in flight per SM,
// and events in flight are what hides the latency of the 24 dependent, barrier-separated steps.
//
// The team path keeps only 12 bytes per hit because it requires every hit
// to lie on its module plane, z[i] == module_z[module[i]] bit for bit (true for the detector:
// the geometry is what velo_geometry_load was given). Then z is a per-module constant and the
// z-ratio of O-4 is computed once per track and step instead of once per candidate. Events that
// break this, or that do not fit the pool, its 15-bit local indices or its candidate table, are
// appended to ws.large_list and reconstructed by the general slab kernel (velo_kernels.cu).
//
// Step semantics: SURVEY.md §8(c) O-1 ... O-14 (restated in DESIGN.md §3). Every float operation
// is a round-to-nearest intrinsic in the written order (no FMA contraction), so hit lists and
// states are bit-identical to the oracle's.
#include "velo_device.cuh"
#include "velo_internal.h"

namespace velo {

namespace {

#ifndef VELO_TEAM_THREADS
#define VELO_TEAM_THREADS 128
#endif
constexpr int kTeamThreads = VELO_TEAM_THREADS;   // tuning builds may try 64 or 256
constexpr int kTeamWarps = kTeamThreads / 32;
constexpr uint32_t kUnitBytes = 3456;       // pool allocation unit: 64 of them (one bitmap word) make
constexpr uint32_t kPoolUnits = 64;         //   216 KB of pool; + 8 KB of control = 224 KB per CTA
constexpr uint32_t kCtlBytes = 8192;
constexpr uint32_t kClChunk = 256;          // centre hits per seeding chunk (2 per thread)
constexpr uint32_t kMaxTeams = kTeamsPerCtaMax;
constexpr uint32_t kMaxTeamHits = kTeamMaxHits;   // <= 32767: the local original index is stored in 15 bits
#ifndef VELO_SEED_LANES
#define VELO_SEED_LANES 4
#endif
constexpr uint32_t kSeedLanes = VELO_SEED_LANES;   // lanes that share the search of one seed centre
constexpr uint32_t kMaxBinSlot = 2047;      // slot inside a phi bucket is stashed in 11 bits
constexpr uint32_t kFlagBit = 0x8000u;      // O-5 flag[h] inside the packed hit word

// Per-team control block (fixed place in the CTA's control unit).
struct TeamShared {
  uint32_t wsum[2][kTeamWarps];   // team_scan scratch, parity-toggled
  uint32_t wsum2[2][kTeamWarps];
  uint32_t event, n, o0;          // the team's current event: index, hits, first hit
  uint32_t pool_off;              // byte offset of its block inside the pool
  uint32_t units, first_unit;
  uint32_t defer;                 // != 0: the event goes to the slab path (or, bit 31, is bad input)
  uint32_t tbase, hbase;          // temp-block bases from the global counters
  uint32_t nt;                    // candidates so far (slot counter)
  uint32_t nact[2];               // lengths of the two active-track lists
  uint32_t ncl[2];                // length of cl[], double-buffered by chunk parity
  uint32_t sstart[VELO_MAX_MODULES + 1];   // sstart[s] = candidates created before step s seeds
  uint16_t cl[kClChunk];          // unflagged centre hits of the current chunk
};

struct Control {
  unsigned long long bitmap;      // 1 = unit in use
  uint32_t alloc_next, alloc_serving;   // FIFO ticket lock around the allocator: no starvation
  float module_z[VELO_MAX_MODULES];
  TeamShared team[kMaxTeams];
};
static_assert(sizeof(Control) <= kCtlBytes, "control block must fit its units");

// Phase timing for tuning builds (-DVELO_PHASE_CLOCKS): the team leader adds the SM clocks spent
// since the previous mark to ws.phase_clk[i]. Compiled out of the product library.
#ifdef VELO_PHASE_CLOCKS
#define VELO_PHASE(i)                                                                  \
  do {                                                                                 \
    if (tid == 0) {                                                                    \
      const long long now_ = clock64();                                                \
      atomicAdd(&a.ws.phase_clk[i], (unsigned long long)(now_ - ph_last));             \
      ph_last = now_;                                                                  \
    }                                                                                  \
  } while (0)
#ifdef VELO_PHASE_COUNTS
#define VELO_COUNT(i, v) atomicAdd(&a.ws.phase_clk[i], (unsigned long long)(v))
#else
#define VELO_COUNT(i, v) do { } while (0)
#endif
// finer marks inside a phase (leader only): clocks since the previous VELO_SUB / VELO_SUB_START
#define VELO_SUB_START() long long sub_last_ = clock64()
#define VELO_SUB(i)                                                                    \
  do {                                                                                 \
    if (tid == 0) {                                                                    \
      const long long now_ = clock64();                                                \
      atomicAdd(&a.ws.phase_clk[i], (unsigned long long)(now_ - sub_last_));           \
      sub_last_ = now_;                                                                \
    }                                                                                  \
  } while (0)
#else
#define VELO_PHASE(i) do { } while (0)
#define VELO_COUNT(i, v) do { } while (0)
#define VELO_SUB_START() do { } while (0)
#define VELO_SUB(i) do { } while (0)
#endif

__device__ __forceinline__ void team_sync(uint32_t team) {
  asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(kTeamThreads) : "memory");
}

// Exclusive scan of one u32 per thread over the team (and of a second value in the same pass).
// `parity` alternates the scratch buffer so that one barrier per call suffices.
__device__ __forceinline__ uint32_t team_scan2(uint32_t v, uint32_t v2, TeamShared& ts, uint32_t team, uint32_t& parity,
                                               uint32_t* total, uint32_t* prefix2, uint32_t* total2) {
  const uint32_t lane = threadIdx.x & 31u, wid = (threadIdx.x & (kTeamThreads - 1)) >> 5;
  uint32_t inc = v, inc2 = v2;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d), o2 = __shfl_up_sync(0xffffffffu, inc2, d);
    if (lane >= (uint32_t)d) { inc += o; inc2 += o2; }
  }
  const uint32_t p = parity & 1u;
  parity ^= 1u;
  if (lane == 31) { ts.wsum[p][wid] = inc; ts.wsum2[p][wid] = inc2; }
  team_sync(team);
  uint32_t base = 0, base2 = 0, tot = 0, tot2 = 0;
#pragma unroll
  for (uint32_t k = 0; k < (uint32_t)kTeamWarps; ++k) {
    const uint32_t s = ts.wsum[p][k], s2 = ts.wsum2[p][k];
    if (k < wid) { base += s; base2 += s2; }
    tot += s; tot2 += s2;
  }
  *total = tot; *total2 = tot2; *prefix2 = base2 + inc2 - v2;
  return base + inc - v;
}

// Byte layout of one event's block in the pool.
struct Layout {
  uint32_t xy, w, bins, u;   // offsets: float2[n], u32[n], packed u16 bucket table, union region
  uint32_t tcap;             // candidate-table capacity
  uint32_t bytes;
};
__device__ __forceinline__ uint32_t align16(uint32_t v) { return (v + 15u) & ~15u; }
constexpr uint32_t kTrackBytes = 21;   // shared-memory bytes per candidate slot (see Ev)
__device__ __forceinline__ Layout event_layout(uint32_t n, uint32_t M) {
  Layout L;
  uint32_t o = 0;
  L.xy = o; o += align16(8u * n);
  L.w = o; o += align16(4u * n);
  L.bins = o; o += align16(2u * (M * kBinsPerModule + 2u));
  L.u = o;
  L.tcap = ((n >> 3) + 32u + 15u) & ~15u;   // candidates ~0.106/hit (max seen 0.157): n/8 + 32, else deferred
  const uint32_t sortb = 4u * n, trkb = kTrackBytes * L.tcap;
  o += align16(sortb > trkb ? sortb : trkb);
  L.bytes = o;
  return L;
}
static_assert(kTeamMaxHits / 8 + 48 <= kTeamMaxTracks, "team scratch rows must cover the candidate table");

// The arrays of one event.
struct Ev {
  // shared memory
  float2* xy;            // sorted hit coordinates
  uint32_t* w;           // packed: (phi16 + 32768) << 16 | flag << 15 | original local index;
                         // after the module loop the upper half becomes the O-13 owner (track id)
  const uint16_t* bo;    // bucket offsets, bo[m * 64 + b], bo[M * 64] = n
  uint32_t* stash;       // sort scratch (dead after S1), aliased by the candidate table:
  uint32_t* tmask;       // modules of the track's hits, bit m
  uint32_t* tl;          // last two hits: older << 16 | latest         } reused as the
  float* tseed;          // seed scatter                                  } 64-bit tkey[t]
  uint16_t* tcentre;     // sorted index of the seed's centre hit
  uint16_t* th0;         // the seed's first hit (row[0]); with tl it flags a track that reaches 4 hits
  uint16_t* act;         // two lists of tcap active-track ids; after the loop: order[] (creation order)
  uint8_t* tmiss;        // consecutive misses; after the loop: pass state (hits on a track = popc(tmask))
  uint32_t tcap;
  // per-team scratch in global memory (L2-resident)
  uint16_t* rows;        // rows[t * 32 + k] = k-th hit (sorted index) of candidate t
  float* st;             // st[k * kTeamMaxTracks + t], k < 9: fitted state of candidate t
};

// ---- O-3 window of module m around unsigned phi `c`: at most two runs of sorted indices, in
// ascending order, and a modular test ((pu - lo) & 0xffff) <= span for the hits inside them.
// lo and span are kept shifted to the phi field of the packed hit word: lo16 = lo << 16,
// lim = span << 16 | 0xffff, so that the test is one subtract and one compare on the whole word.
struct Window { uint32_t b0, e0, b1, e1, lo16, lim; };
__device__ __forceinline__ Window make_window(const uint16_t* bo_m, uint32_t c, int W) {
  Window q;
  q.b1 = q.e1 = 0;
  if (W < 0) { q.b0 = q.e0 = 0; q.lo16 = 0; q.lim = 0; return q; }
  if (2 * (long long)W + 1 >= 65536) { q.b0 = bo_m[0]; q.e0 = bo_m[kBinsPerModule]; q.lo16 = 0; q.lim = 0xffffffffu; return q; }
  const uint32_t lo = (c - (uint32_t)W) & 0xffffu, hi = (c + (uint32_t)W) & 0xffffu;
  q.lo16 = lo << 16; q.lim = (2u * (uint32_t)W) << 16 | 0xffffu;
  if (lo <= hi) { q.b0 = bo_m[lo >> kBinShift]; q.e0 = bo_m[(hi >> kBinShift) + 1]; }
  else if ((lo >> kBinShift) <= (hi >> kBinShift)) {  // wraps and the two runs would overlap: whole module
    q.b0 = bo_m[0]; q.e0 = bo_m[kBinsPerModule];
  } else {  // wraps: the low-phi run has the lower sorted indices and is visited first
    q.b0 = bo_m[0]; q.e0 = bo_m[(hi >> kBinShift) + 1];
    q.b1 = bo_m[lo >> kBinShift]; q.e1 = bo_m[kBinsPerModule];
  }
  return q;
}
__device__ __forceinline__ bool in_window(const Window& q, uint32_t wj) { return wj - q.lo16 <= q.lim; }

// Visits the sorted indices [b, e) in ascending order, four per trip: the eight shared-memory
// loads of a trip are issued before any of its arithmetic, so a trip costs one load latency
// instead of four (the scans are latency-bound, not bandwidth-bound). f(j, w, xy, valid) must be
// branch-free; for the padding lanes of the last trip valid is false and j repeats e - 1.
template <class F>
__device__ __forceinline__ void scan4(const Ev& ev, uint32_t b, uint32_t e, F&& f) {
  for (uint32_t j = b; j < e; j += 4u) {
    uint32_t jj[4], wj[4]; float2 pj[4];
#pragma unroll
    for (uint32_t k = 0; k < 4; ++k) { jj[k] = min(j + k, e - 1u); wj[k] = ev.w[jj[k]]; pj[k] = ev.xy[jj[k]]; }
#pragma unroll
    for (uint32_t k = 0; k < 4; ++k) f(jj[k], wj[k], pj[k], j + k < e);
  }
}

// Calls f(i, h) for the hits h (sorted indices) of candidate t in discovery order, i = 0 .. n-1.
// One 16-byte load per 8 hits from the team's row scratch.
template <class F>
__device__ __forceinline__ void for_hits(const Ev& ev, uint32_t t, uint32_t n, F&& f) {
  const uint4* row = reinterpret_cast<const uint4*>(ev.rows + t * 32u);
  for (uint32_t g = 0; g * 8u < n; ++g) {
    const uint4 v = row[g];
    const uint32_t q[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (uint32_t j = 0; j < 8; ++j) {
      if (g * 8u + j < n) f(g * 8u + j, (q[j >> 1] >> ((j & 1u) * 16u)) & 0xffffu);
    }
  }
}

// ---- O-11 straight-line fit of candidate t with z taken from the module planes ---------------
// s9 = x, y, tx, ty, z, cxx, cxtx, vt, chi2 (the 13 state words repeat cxx, cxtx, vt for y and add n).
// Hits are visited in discovery order = decreasing module = the set bits of `mask` from the top.
__device__ __forceinline__ void fit_track(const Ev& ev, const float* mz, uint32_t t, uint32_t n, uint32_t mask,
                                          float sig2, float inv_s2, float* s9) {
  float sz = 0.0f, sx = 0.0f, sy = 0.0f;
  uint32_t mk = mask;
  for_hits(ev, t, n, [&](uint32_t, uint32_t h) {
    const uint32_t m = 31u - __clz(mk); mk &= ~(1u << m);
    const float2 p = ev.xy[h];
    sz = __fadd_rn(sz, mz[m]); sx = __fadd_rn(sx, p.x); sy = __fadd_rn(sy, p.y);
  });
  const float nf = (float)n;
  const float zb = __fdiv_rn(sz, nf), xb = __fdiv_rn(sx, nf), yb = __fdiv_rn(sy, nf);
  float sdd = 0.0f, sdx = 0.0f, sdy = 0.0f;
  mk = mask;
  for_hits(ev, t, n, [&](uint32_t, uint32_t h) {
    const uint32_t m = 31u - __clz(mk); mk &= ~(1u << m);
    const float2 p = ev.xy[h];
    const float d = __fsub_rn(mz[m], zb);
    sdd = __fadd_rn(sdd, __fmul_rn(d, d));
    sdx = __fadd_rn(sdx, __fmul_rn(d, __fsub_rn(p.x, xb)));
    sdy = __fadd_rn(sdy, __fmul_rn(d, __fsub_rn(p.y, yb)));
  });
  const float tx = __fdiv_rn(sdx, sdd), ty = __fdiv_rn(sdy, sdd);
  float c = 0.0f;
  mk = mask;
  for_hits(ev, t, n, [&](uint32_t, uint32_t h) {
    const uint32_t m = 31u - __clz(mk); mk &= ~(1u << m);
    const float2 p = ev.xy[h];
    const float d = __fsub_rn(mz[m], zb);
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

__device__ __forceinline__ void set_status(uint32_t* counters, int code) {
  atomicCAS(&counters[kCtrStatus], 0u, (uint32_t)code);   // first error wins
}

__device__ __forceinline__ void defer_to_slab(const KernelArgs& a, uint32_t e) {
  a.ws.large_list[atomicAdd(&a.ws.counters[kCtrLargeN], 1u)] = e;
}

// ---- pool allocator (called by a team's leader thread only) ------------------------------------
__device__ __forceinline__ uint32_t pool_alloc(Control& ctl, uint32_t units) {
  const uint32_t my = atomicAdd(&ctl.alloc_next, 1u);
  volatile uint32_t* serving = &ctl.alloc_serving;
  while (*serving != my) __nanosleep(1500);
  volatile unsigned long long* bm = &ctl.bitmap;
  const unsigned long long all = kPoolUnits >= 64u ? ~0ull : (1ull << (kPoolUnits & 63u)) - 1ull;
  uint32_t first;
  unsigned long long seen = ~0ull;
  for (;;) {
    const unsigned long long used = *bm;
    if (used == seen) { __nanosleep(1500); continue; }   // nothing was freed since the last failed try
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
__device__ __forceinline__ void pool_free(Control& ctl, uint32_t first, uint32_t units) {
  const unsigned long long claim = ((units >= 64u ? ~0ull : ((1ull << units) - 1ull)) << first);
  atomicAnd(&ctl.bitmap, ~claim);
}

// Leader: take the next event and a pool block for it. ts.defer != 0 means "nothing to do here".
__device__ void leader_fetch(const KernelArgs& a, Control& ctl, TeamShared& ts) {
  const uint32_t k = atomicAdd(&a.ws.counters[kCtrTicket], 1u);
  ts.event = k; ts.units = 0; ts.defer = 1; ts.n = 0;
  if (k >= a.n_events) return;
  // tickets walk the size-sorted list from both ends in turn: largest, smallest, second largest, ...
  const uint32_t e = a.ws.order[(k & 1u) ? (k >> 1) : a.n_events - 1u - (k >> 1)];
  ts.event = e;
  const uint32_t o0 = a.event_offsets[e], o1 = a.event_offsets[e + 1];
  if (o1 < o0 || o1 - o0 > VELO_MAX_EVENT_HITS) {
    set_status(a.ws.counters, VELO_ERR_INPUT); a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0); return;
  }
  const uint32_t n = o1 - o0;
  if (n == 0) { a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0); return; }
  if (n > a.team_max_hits) { defer_to_slab(a, e); return; }
  const Layout L = event_layout(n, a.n_modules);
  const uint32_t units = (L.bytes + kUnitBytes - 1u) / kUnitBytes;
  if (units > kPoolUnits) { defer_to_slab(a, e); return; }
  const uint32_t first = pool_alloc(ctl, units);
  ts.n = n; ts.o0 = o0; ts.units = units; ts.first_unit = first; ts.pool_off = first * kUnitBytes; ts.defer = 0;
}

// ---- one event, by one team -----------------------------------------------------------------------
__device__ void team_event(const KernelArgs& a, Control& ctl, TeamShared& ts, unsigned char* pool,
                           unsigned char* scratch, uint32_t team, uint32_t tid, uint32_t& parity, long long& ph_last) {
  (void)ph_last;
  const uint32_t lane = tid & 31u, wid = tid >> 5;
  const uint32_t M = a.n_modules, nbins = M * kBinsPerModule;
  const velo_params_t& P = a.P;
  const uint32_t e = ts.event, n = ts.n, o0 = ts.o0;
  const float* mz = ctl.module_z;
  const Layout L = event_layout(n, M);
  unsigned char* blk = pool + ts.pool_off;
  Ev ev;
  ev.xy = (float2*)(blk + L.xy); ev.w = (uint32_t*)(blk + L.w);
  uint32_t* binsw = (uint32_t*)(blk + L.bins);
  uint16_t* bins16 = (uint16_t*)binsw;
  ev.bo = bins16;
  ev.stash = (uint32_t*)(blk + L.u);
  const uint32_t T = L.tcap;
  ev.tcap = T;
  {
    unsigned char* q = blk + L.u;
    ev.tmask = (uint32_t*)q; q += 4u * T;
    ev.tl = (uint32_t*)q; q += 4u * T;
    ev.tseed = (float*)q; q += 4u * T;
    ev.tcentre = (uint16_t*)q; q += 2u * T;
    ev.th0 = (uint16_t*)q; q += 2u * T;
    ev.act = (uint16_t*)q; q += 4u * T;
    ev.tmiss = q;
  }
  ev.rows = (uint16_t*)scratch;
  ev.st = (float*)(scratch + (size_t)kTeamMaxTracks * 64u);
  unsigned long long* tkey = (unsigned long long*)ev.tl;   // 8 bytes per track over (tl, tseed), used after O-10
  const size_t g0 = (size_t)(o0 - a.hit_base);
  const float* gx = a.x + g0; const float* gy = a.y + g0; const float* gz = a.z + g0;
  const uint8_t* gm = a.module + g0;

  // ---- S0 decode: phi16, bucket histogram (O-1); the plane check of the team path ---------------
  const uint32_t nwords = nbins / 2u;
  for (uint32_t b = tid; b <= nwords; b += kTeamThreads) binsw[b] = 0;
  team_sync(team);
  {
    uint32_t trouble = 0;
    constexpr uint32_t U = 4;   // hits in flight per thread: the loads of a group are issued together
    for (uint32_t i0 = tid; i0 < n; i0 += U * kTeamThreads) {
      float x[U], y[U], z[U]; uint32_t m[U];
#pragma unroll
      for (uint32_t k = 0; k < U; ++k) {
        const uint32_t i = i0 + k * kTeamThreads;
        const bool ok = i < n;
        x[k] = ok ? gx[i] : 1.0f; y[k] = ok ? gy[i] : 0.0f; z[k] = ok ? gz[i] : 0.0f; m[k] = ok ? (uint32_t)gm[i] : 0xffffffffu;
      }
#pragma unroll
      for (uint32_t k = 0; k < U; ++k) {
        const uint32_t i = i0 + k * kTeamThreads;
        if (i >= n) continue;
        if (m[k] >= M) { trouble |= 0x80000000u; continue; }
        if (__float_as_uint(z[k]) != __float_as_uint(mz[m[k]])) trouble |= 1u;
        const uint32_t pu = (uint32_t)(phi16(x[k], y[k]) + 32768);
        const uint32_t bin = m[k] * kBinsPerModule + (pu >> kBinShift);
        const uint32_t sh = (bin & 1u) * 16u;
        const uint32_t slot = (atomicAdd(&binsw[bin >> 1], 1u << sh) >> sh) & 0xffffu;
        if (slot > kMaxBinSlot) trouble |= 1u;
        ev.stash[i] = (m[k] << 27) | (pu << 11) | (slot & kMaxBinSlot);
      }
    }
    if (trouble) atomicOr(&ts.defer, trouble);
  }
  team_sync(team);
  VELO_PHASE(1);   // S0 decode
  if (ts.defer) {
    if (tid == 0) {
      if (ts.defer & 0x80000000u) { set_status(a.ws.counters, VELO_ERR_INPUT); a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0); }
      else defer_to_slab(a, e);
    }
    return;
  }
  // exclusive scan of the packed histogram -> bucket offsets; bo[nbins] = n
  {
    const uint32_t per = (nwords + kTeamThreads - 1) / kTeamThreads;
    const uint32_t w0 = min(tid * per, nwords), w1 = min(w0 + per, nwords);
    uint32_t s = 0;
    for (uint32_t k = w0; k < w1; ++k) { const uint32_t v = binsw[k]; s += (v & 0xffffu) + (v >> 16); }
    uint32_t tot, p2, t2;
    uint32_t run = team_scan2(s, 0u, ts, team, parity, &tot, &p2, &t2);
    for (uint32_t k = w0; k < w1; ++k) {
      const uint32_t v = binsw[k], c0 = v & 0xffffu, c1 = v >> 16;
      binsw[k] = run | ((run + c0) << 16);
      run += c0 + c1;
    }
    if (tid == 0) bins16[nbins] = (uint16_t)n;
  }
  team_sync(team);
  VELO_PHASE(2);   // bucket scan
  // ---- S1 phi sort (O-2): group by bucket in w[], rank inside the bucket by (phi16, index), place ---
  for (uint32_t i = tid; i < n; i += kTeamThreads) {
    const uint32_t st = ev.stash[i], pu = (st >> 11) & 0xffffu;
    const uint32_t bin = (st >> 27) * kBinsPerModule + (pu >> kBinShift);
    ev.w[(uint32_t)bins16[bin] + (st & kMaxBinSlot)] = (pu << 16) | i;
  }
  team_sync(team);
  for (uint32_t i = tid; i < n; i += kTeamThreads) {
    const uint32_t st = ev.stash[i], pu = (st >> 11) & 0xffffu;
    const uint32_t bin = (st >> 27) * kBinsPerModule + (pu >> kBinShift);
    const uint32_t item = (pu << 16) | i;
    const uint32_t lo = bins16[bin], hi = bins16[bin + 1];
    uint32_t r = lo;
    for (uint32_t j = lo; j < hi; ++j) r += (ev.w[j] < item) ? 1u : 0u;
    ev.stash[i] = (pu << 16) | r;   // r <= 32767
  }
  team_sync(team);   // every rank is known: w[] can take its final content
  {
    constexpr uint32_t U = 4;
    for (uint32_t i0 = tid; i0 < n; i0 += U * kTeamThreads) {
      float x[U], y[U];
#pragma unroll
      for (uint32_t k = 0; k < U; ++k) {
        const uint32_t i = i0 + k * kTeamThreads;
        x[k] = i < n ? gx[i] : 0.0f; y[k] = i < n ? gy[i] : 0.0f;   // second read of x, y: L2
      }
#pragma unroll
      for (uint32_t k = 0; k < U; ++k) {
        const uint32_t i = i0 + k * kTeamThreads;
        if (i >= n) continue;
        const uint32_t st = ev.stash[i], r = st & 0xffffu;
        ev.xy[r] = make_float2(x[k], y[k]);
        ev.w[r] = (st & 0xffff0000u) | i;
      }
    }
  }
  team_sync(team);   // the sort scratch is dead from here on: the candidate table takes its place
  VELO_PHASE(3);   // S1 sort

  // ---- O-6 module loop ---------------------------------------------------------------------------
  // Dense work lists keep the lanes busy: act[] = the tracks still forwarding (order irrelevant:
  // every decision of a phase reads only state from before the phase), cl[] = the unflagged
  // centre hits of a chunk. Slots of new candidates come from an atomic counter, so the table
  // order is arbitrary; the creation order is restored once, after the loop (sstart[], order[]).
  if (tid == 0) { ts.nt = 0; ts.nact[0] = ts.nact[1] = 0; ts.ncl[0] = ts.ncl[1] = 0; ts.sstart[M - 1] = 0; }
  uint32_t cur = 0, cpar = 0;
  team_sync(team);
  for (uint32_t s = M - 2; s >= 1; --s) {
    const uint32_t u = s - 1, nxt = cur ^ 1u;
    // No hit in modules 0 .. u: forwarding can only miss and seeding finds no third hit, in this step
    // and in all that follow, and what a miss changes (the miss counter) is not read after the loop.
    if (ev.bo[(u + 1) * kBinsPerModule] == 0) {
      for (uint32_t r = tid + 1u; r <= s; r += kTeamThreads) ts.sstart[r] = ts.nt;   // nothing is created any more
      break;
    }
    VELO_SUB_START();
    // (A) O-7 forwarding into module u of every track active at the start of the step
    {
      const uint32_t nact = ts.nact[cur];
      const float z2 = mz[u];
      const float max_fwd = P.max_scatter_fwd;
      const uint16_t* bo_u = ev.bo + u * kBinsPerModule;
      const uint16_t* act = ev.act + cur * T;
      uint16_t* act_next = ev.act + nxt * T;
      for (uint32_t k0 = wid * 32u; k0 < nact; k0 += kTeamThreads) {
        const uint32_t k = k0 + lane;
        bool alive = false;
        uint32_t t = 0;
        if (k < nact) {
          t = act[k];
          const uint32_t l = ev.tl[t], ha = l >> 16, hb = l & 0xffffu;
          const uint32_t mask = ev.tmask[t];
          const uint32_t mb = __ffs(mask) - 1u, ma = __ffs(mask & (mask - 1u)) - 1u;
          const float2 p1 = ev.xy[hb], p0 = ev.xy[ha];
          const uint32_t whb = ev.w[hb], c = whb >> 16;
          const float z1 = mz[mb], z0 = mz[ma];
          VELO_SUB(24);   // list entry, track words, hit words
          const float tz = __fdiv_rn(__fsub_rn(z2, z1), __fsub_rn(z1, z0));
          const float px = __fadd_rn(p1.x, __fmul_rn(__fsub_rn(p1.x, p0.x), tz));
          const float py = __fadd_rn(p1.y, __fmul_rn(__fsub_rn(p1.y, p0.y), tz));
          const Window q = make_window(bo_u, c, P.phi_window_fwd);
          VELO_SUB(25);   // prediction, window
          // branch-free visits (the loops are latency-bound: a taken branch costs more than the math)
          bool found = false; uint32_t best = 0, best_w = 0; float best_sc = 0.0f;
          auto visit = [&](uint32_t j, uint32_t wj, float2 p2, bool valid) {
            const float ex = __fsub_rn(px, p2.x), ey = __fsub_rn(py, p2.y);
            const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
            const bool better = valid & in_window(q, wj) & (sc <= max_fwd) & (!found | (sc < best_sc));
            found |= better; best = better ? j : best; best_w = better ? wj : best_w; best_sc = better ? sc : best_sc;
          };
          scan4(ev, q.b0, q.e0, visit);
          scan4(ev, q.b1, q.e1, visit);   // second run: only for a window across +-pi
          VELO_SUB(26);   // visits
          VELO_COUNT(16, 1); VELO_COUNT(17, (q.e0 - q.b0) + (q.e1 - q.b1));
          if (found) {
            const uint32_t nh = (uint32_t)__popc(mask);   // one hit per module: the mask counts them
            ev.rows[t * 32u + nh] = (uint16_t)best;
            ev.tmiss[t] = 0;
            ev.tl[t] = (hb << 16) | best;
            ev.tmask[t] = mask | (1u << u);
            // (B): forwarding never reads flags, so they can be set right away
            // (the words of hb and best are in registers: the other bits of a hit word never change
            // during the loop, so a plain store of word | flag is as good as a read-modify-write)
            if (nh + 1 == 4) { ev.w[ev.th0[t]] |= kFlagBit; ev.w[ha] |= kFlagBit; ev.w[hb] = whb | kFlagBit; }
            if (nh + 1 >= 4) ev.w[best] = best_w | kFlagBit;
            alive = true;
          } else {
            const uint32_t miss = (uint32_t)ev.tmiss[t] + 1u;
            ev.tmiss[t] = (uint8_t)miss;
            alive = miss <= P.max_skipped;
          }
        }
        VELO_SUB(27);   // track update, flags
        const uint32_t ballot = __ballot_sync(0xffffffffu, alive);
        if (ballot) {
          uint32_t base = 0;
          if (lane == 0) base = atomicAdd(&ts.nact[nxt], (uint32_t)__popc(ballot));
          base = __shfl_sync(0xffffffffu, base, 0);
          if (alive) act_next[base + __popc(ballot & ((1u << lane) - 1u))] = (uint16_t)t;
        }
      }
    }
    VELO_SUB(28);   // list append
    team_sync(team);
    VELO_SUB(29);   // barrier
    VELO_PHASE(4);   // (A) forwarding
    if (tid == 0) { ts.nact[cur] = 0; ts.sstart[s] = ts.nt; }   // nact[cur] was read by everyone before the barrier
    // (C) O-8 seeding with centre module s, in chunks of 2 x 128 centre hits
    {
      const uint32_t c_begin = ev.bo[s * kBinsPerModule], c_end = ev.bo[(s + 1) * kBinsPerModule];
      const float z0 = mz[s + 1], z1 = mz[s], z2 = mz[u];
      const float tz = __fdiv_rn(__fsub_rn(z2, z1), __fsub_rn(z1, z0));
      const float max_seed = P.max_scatter_seed;
      const uint16_t* bo_0 = ev.bo + (s + 1) * kBinsPerModule;
      const uint16_t* bo_2 = ev.bo + u * kBinsPerModule;
      uint16_t* act_next = ev.act + nxt * T;
      for (uint32_t c0 = c_begin; c0 < c_end; c0 += kClChunk) {
        // (C1) the chunk's unflagged centre hits -> cl[] (flags are final for this step: (A) is done)
#pragma unroll
        for (uint32_t r = 0; r < kClChunk / kTeamThreads; ++r) {
          const uint32_t h1 = c0 + r * kTeamThreads + tid;
          const bool open = h1 < c_end && !(ev.w[h1] & kFlagBit);
          const uint32_t ballot = __ballot_sync(0xffffffffu, open);
          if (ballot) {
            uint32_t base = 0;
            if (lane == 0) base = atomicAdd(&ts.ncl[cpar], (uint32_t)__popc(ballot));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (open) ts.cl[base + __popc(ballot & ((1u << lane) - 1u))] = (uint16_t)h1;
          }
        }
        team_sync(team);
        VELO_PHASE(5);   // (C1) unflagged centre hits
        const uint32_t ncl = ts.ncl[cpar];
        if (tid == 0) ts.ncl[cpar ^ 1u] = 0;   // the other counter: last read before the barrier above
        cpar ^= 1u;
        // (C2) four lanes per unflagged centre hit: lane `sub` takes every 4th h0 of the window; the
        // quad's best (h0, h2) under (scatter, h0, h2) is reduced with shuffles
        for (uint32_t k0 = 0; k0 < ncl; k0 += kTeamThreads / kSeedLanes) {
          const uint32_t k = k0 + tid / kSeedLanes, sub = tid % kSeedLanes;
          bool found = false; uint32_t b0 = 0, b2 = 0, h1 = 0; float best_sc = 0.0f;
          if (k < ncl) {
            h1 = ts.cl[k];
            const uint32_t w1 = ev.w[h1];
            const float2 p1 = ev.xy[h1];
            const Window q0 = make_window(bo_0, w1 >> 16, P.phi_window_seed);
            const Window q2 = make_window(bo_2, w1 >> 16, P.phi_window_seed);
            const uint32_t end0 = q0.e0 + (q0.e1 - q0.b1);
            VELO_COUNT(18, 1); VELO_COUNT(19, end0 - q0.b0);
            for (uint32_t jo = q0.b0 + sub; jo < end0; jo += kSeedLanes) {
              const uint32_t h0 = jo < q0.e0 ? jo : jo - q0.e0 + q0.b1;
              const uint32_t w0 = ev.w[h0];
              if ((w0 & kFlagBit) || !in_window(q0, w0)) continue;
              VELO_COUNT(20, 1); VELO_COUNT(21, (q2.e0 - q2.b0) + (q2.e1 - q2.b1));
              const float2 p0 = ev.xy[h0];
              const float px = __fadd_rn(p1.x, __fmul_rn(__fsub_rn(p1.x, p0.x), tz));
              const float py = __fadd_rn(p1.y, __fmul_rn(__fsub_rn(p1.y, p0.y), tz));
              // h0 and h2 ascending: strict < keeps this lane's lexicographic minimum; branch-free body
              auto visit2 = [&](uint32_t h2, uint32_t w2, float2 p2, bool valid) {
                const float ex = __fsub_rn(px, p2.x), ey = __fsub_rn(py, p2.y);
                const float sc = __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
                const bool better = valid & !(w2 & kFlagBit) & in_window(q2, w2) & (sc <= max_seed) & (!found | (sc < best_sc));
                found |= better; b0 = better ? h0 : b0; b2 = better ? h2 : b2; best_sc = better ? sc : best_sc;
              };
              scan4(ev, q2.b0, q2.e0, visit2);
              scan4(ev, q2.b1, q2.e1, visit2);
            }
          }
#pragma unroll
          for (uint32_t d = 1; d < kSeedLanes; d <<= 1) {   // minimum over the group, ties: lowest h0, then lowest h2
            const bool of = __shfl_xor_sync(0xffffffffu, (int)found, d) != 0;
            const float osc = __shfl_xor_sync(0xffffffffu, best_sc, d);
            const uint32_t ob0 = __shfl_xor_sync(0xffffffffu, b0, d), ob2 = __shfl_xor_sync(0xffffffffu, b2, d);
            const bool take = of & (!found | (osc < best_sc) | ((osc == best_sc) & ((ob0 < b0) | ((ob0 == b0) & (ob2 < b2)))));
            found |= of; b0 = take ? ob0 : b0; b2 = take ? ob2 : b2; best_sc = take ? osc : best_sc;
          }
          if (found && sub == 0) {
            const uint32_t slot = atomicAdd(&ts.nt, 1u);
            if (slot < T) {
              *reinterpret_cast<uint2*>(ev.rows + slot * 32u) = make_uint2(b0 | (h1 << 16), b2);
              ev.th0[slot] = (uint16_t)b0;
              ev.tmiss[slot] = 0;
              ev.tl[slot] = (h1 << 16) | b2;
              ev.tmask[slot] = 7u << u;
              ev.tseed[slot] = best_sc; ev.tcentre[slot] = (uint16_t)h1;
              act_next[atomicAdd(&ts.nact[nxt], 1u)] = (uint16_t)slot;
            }
          }
        }
        team_sync(team);   // cl[] may be refilled; after the last chunk: the new tracks are visible
        VELO_PHASE(6);   // (C2) seeding
        if (tid == 0) { VELO_COUNT(22, 1); }
      }
      if (c_begin >= c_end) team_sync(team);   // no chunk ran: still order this step's resets before the next step
    }
    if (ts.nt > T) {   // candidate table too small for this event: the general path takes it
      if (tid == 0) defer_to_slab(a, e);
      return;
    }
    cur = nxt;
  }
  const uint32_t nt = ts.nt;
  // creation order (O-8: step descending, then sorted index of the centre hit) of the table entries
  uint16_t* order = ev.act;   // the work lists are dead
  if (tid == 0) ts.sstart[0] = nt;
  team_sync(team);
  for (uint32_t t = tid; t < nt; t += kTeamThreads) {
    const uint32_t sc = 30u - __clz(ev.tmask[t]);            // centre module = step of creation
    const uint32_t a0 = ts.sstart[sc], a1 = ts.sstart[sc - 1];
    const uint32_t centre = ev.tcentre[t];
    uint32_t r = a0;
    for (uint32_t j = a0; j < a1; ++j) r += (ev.tcentre[j] < centre) ? 1u : 0u;
    order[r] = (uint16_t)t;
  }
  // (visible to the scan below after the barriers of the phases in between)
  VELO_PHASE(7);   // creation order

  // ---- O-10 ghost filter part 1 (reads the final flags); tmiss[t] becomes the pass state ---------
  for (uint32_t t = tid; t < nt; t += kTeamThreads) {
    bool pass = true;
    if (__popc(ev.tmask[t]) == 3) {
      const uint32_t l = ev.tl[t];   // never extended: still (centre, third hit)
      const uint32_t f = ev.w[ev.th0[t]] | ev.w[l >> 16] | ev.w[l & 0xffffu];
      if ((f & kFlagBit) || !(ev.tseed[t] <= P.max_scatter_weak)) pass = false;
    }
    ev.tmiss[t] = pass ? 1 : 0;
  }
  team_sync(team);
  // ---- O-11 fit, O-12 chi2 cut, O-13 key --------------------------------------------------------
  // (tkey[t] overlays tl/tseed of other tracks: every thread has read those above)
  const float sig2 = __fmul_rn(P.sigma_hit, P.sigma_hit);
  const float inv_s2 = __fdiv_rn(1.0f, sig2);
  for (uint32_t t = tid; t < nt; t += kTeamThreads) {
    if (!ev.tmiss[t]) continue;
    const uint32_t nh = (uint32_t)__popc(ev.tmask[t]);
    const uint32_t centre = ev.tcentre[t];
    float s9[9];
    fit_track(ev, mz, t, nh, ev.tmask[t], sig2, inv_s2, s9);
    const float lim = __fmul_rn(P.max_chi2_ndof, (float)(2 * (int)nh - 4));
    if (s9[8] > lim) { ev.tmiss[t] = 0; continue; }
    tkey[t] = ((unsigned long long)(255u - nh) << 56) | ((unsigned long long)__float_as_uint(s9[8]) << 24) |
              (unsigned long long)centre;
#pragma unroll
    for (uint32_t k = 0; k < 9; ++k) ev.st[k * kTeamMaxTracks + t] = s9[k];
  }
  team_sync(team);
  VELO_PHASE(8);   // O-10, fit, keys
  // ---- O-13 owners: owner[h] = the candidate with the smallest key among those that contain h ----
  // Step 1: every passing candidate writes its id on its hits (plain 16-bit stores: where several
  // candidates share a hit, any one of them lands). Step 2: a candidate that finds another id on
  // one of its hits settles it with a compare-and-swap on the 64-bit keys. Hits are shared rarely,
  // so the common path has no atomics and no dependent chain.
  {
    uint16_t* own = reinterpret_cast<uint16_t*>(ev.w);   // own[2h + 1] = upper half of w[h]
    for (uint32_t t = tid; t < nt; t += kTeamThreads) {
      if (!ev.tmiss[t]) continue;
      for_hits(ev, t, (uint32_t)__popc(ev.tmask[t]), [&](uint32_t, uint32_t h) { own[2u * h + 1u] = (uint16_t)t; });
    }
    team_sync(team);
    for (uint32_t t = tid; t < nt; t += kTeamThreads) {
      if (!ev.tmiss[t]) continue;
      const unsigned long long key = tkey[t];
      for_hits(ev, t, (uint32_t)__popc(ev.tmask[t]), [&](uint32_t, uint32_t h) {
        uint32_t* wp = &ev.w[h];
        uint32_t old = *(volatile uint32_t*)wp;
        while ((old >> 16) != t && key < tkey[old >> 16]) {
          const uint32_t seen = atomicCAS(wp, old, (t << 16) | (old & 0xffffu));
          if (seen == old) break;
          old = seen;
        }
      });
    }
  }
  team_sync(team);
  VELO_PHASE(9);   // owners
  // ---- O-13 clone filter, then the event's survivors in creation order (exclusive scans) ---------
  uint32_t* pl = ev.tl;                 // per-track output position inside the event: track index and
  uint32_t* ph = (uint32_t*)ev.tseed;   // hit offset (tkey, which overlays both, is dead after the owners phase)
  uint32_t run_t = 0, run_h = 0;
  for (uint32_t k0 = 0; k0 < nt; k0 += kTeamThreads) {
    const uint32_t k = k0 + tid;
    const uint32_t t = k < nt ? order[k] : 0u;   // the k-th candidate in creation order
    uint32_t nh = 0, surv = 0;
    if (k < nt && ev.tmiss[t]) {
      nh = (uint32_t)__popc(ev.tmask[t]);
      uint32_t lost = 0;
      for_hits(ev, t, nh, [&](uint32_t, uint32_t h) { lost += ((ev.w[h] >> 16) != t) ? 1u : 0u; });
      surv = !((unsigned long long)lost * P.clone_den > (unsigned long long)nh * P.clone_num) ? 1u : 0u;
      if (!surv) nh = 0;
    }
    uint32_t tot_h, pre_t, tot_t;
    const uint32_t pre_h = team_scan2(nh, surv, ts, team, parity, &tot_h, &pre_t, &tot_t);
    if (k < nt) { ev.tmiss[t] = (uint8_t)(surv ? 2 : 0); pl[t] = run_t + pre_t; ph[t] = run_h + pre_h; }
    run_t += tot_t; run_h += tot_h;
  }
  const uint32_t ev_nt = run_t, ev_nh = run_h;
  VELO_PHASE(10);  // clone filter + scans
  // ---- S7 part 1: allocate the event's temp block; stage the hit lists; coalesced copy out -------
  if (tid == 0) {
    ts.tbase = atomicAdd(&a.ws.counters[kCtrTracks], ev_nt);
    ts.hbase = atomicAdd(&a.ws.counters[kCtrHits], ev_nh);
    atomicAdd(&a.ws.counters[kCtrCand], nt);
    a.ws.ev_rec[e] = make_uint4(ts.tbase, ts.hbase, ev_nt, ev_nh);
  }
  team_sync(team);
  const uint32_t tbase = ts.tbase, hbase = ts.hbase;
  const bool fits = (unsigned long long)tbase + ev_nt <= a.cap_tracks &&
                    (unsigned long long)hbase + ev_nh <= a.cap_track_hits;
  if (!fits) return;   // VELO_ERR_CAPACITY is raised by the offsets kernel; nothing valid to write
  uint32_t* stage = (uint32_t*)ev.xy;          // coordinates are dead after the fit: 2n words
  const bool staged = ev_nh <= 2u * n;
  for (uint32_t t = tid; t < nt; t += kTeamThreads) {
    if (ev.tmiss[t] != 2) continue;
    const uint32_t nh = (uint32_t)__popc(ev.tmask[t]), lt = pl[t], lh = ph[t];
    float s9[9];
#pragma unroll
    for (uint32_t k = 0; k < 9; ++k) s9[k] = ev.st[k * kTeamMaxTracks + t];
    float* st = a.ws.tmp_states + tbase + lt;
    const size_t cs = a.cap_tracks;
    st[0] = s9[0]; st[cs] = s9[1]; st[2 * cs] = s9[2]; st[3 * cs] = s9[3]; st[4 * cs] = s9[4];
    st[5 * cs] = s9[5]; st[6 * cs] = s9[6]; st[7 * cs] = s9[7];
    st[8 * cs] = s9[5]; st[9 * cs] = s9[6]; st[10 * cs] = s9[7];
    st[11 * cs] = s9[8]; st[12 * cs] = __uint_as_float(nh);
    a.ws.tmp_loff[tbase + lt] = lh;
    uint32_t* dst = staged ? stage + lh : a.ws.tmp_hits + hbase + lh;
    for_hits(ev, t, nh, [&](uint32_t i, uint32_t h) { dst[i] = o0 + (ev.w[h] & 0x7fffu); });
  }
  if (staged) {
    team_sync(team);
    for (uint32_t j = tid; j < ev_nh; j += kTeamThreads) a.ws.tmp_hits[hbase + j] = stage[j];
  }
  VELO_PHASE(11);  // output
}

// ---- the kernel: one CTA per SM, kTeams teams, events by ticket ---------------------------------
// The launch bound is one team more than the CTA has: it caps the registers (80 for 5 teams) so
// that about 14 k registers per SM stay free and the small kernels around the event kernel (order,
// deferred-event list, offsets, compaction) of the neighbouring batches run beside it instead of
// waiting for a whole SM.
template <int kTeams>
__global__ void __launch_bounds__((kTeams + 1) * kTeamThreads > 1024 ? 1024 : (kTeams + 1) * kTeamThreads, 1)
    velo_event_team_kernel(const KernelArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  Control& ctl = *reinterpret_cast<Control*>(smem);
  unsigned char* pool = smem + kCtlBytes;
  const uint32_t team = threadIdx.x / kTeamThreads, tid = threadIdx.x % kTeamThreads;
  if (threadIdx.x == 0) { ctl.bitmap = 0ull; ctl.alloc_next = 0; ctl.alloc_serving = 0; }
  if (threadIdx.x < VELO_MAX_MODULES) ctl.module_z[threadIdx.x] = a.module_z[threadIdx.x];
  __syncthreads();
  TeamShared& ts = ctl.team[team];
  unsigned char* scratch = a.ws.team_scratch + ((size_t)blockIdx.x * kMaxTeams + team) * kTeamScratchBytes;
  uint32_t parity = 0;
  long long ph_last = clock64();
  (void)ph_last;
  for (;;) {
    if (tid == 0) leader_fetch(a, ctl, ts);
    team_sync(team);
    if (ts.event >= a.n_events) break;
    VELO_PHASE(0);   // ticket + pool allocation (waiting for shared memory)
    if (!ts.defer) team_event(a, ctl, ts, pool, scratch, team, tid, parity, ph_last);
    team_sync(team);   // every thread is done with the block and with ts before the leader reuses them
    if (tid == 0 && ts.units) pool_free(ctl, ts.first_unit, ts.units);
    VELO_PHASE(12);  // last barrier + free
  }
}

template <int kTeams>
int launch_teams(const KernelArgs& a, cudaStream_t stream) {
  static_assert(kTeams <= (int)kMaxTeams && kTeams <= 15, "named barriers 1..15");
  if constexpr (kTeams * kTeamThreads > 1024) {
    return launch_teams<1024 / kTeamThreads>(a, stream);
  } else {
  const uint32_t smem = kCtlBytes + kPoolUnits * kUnitBytes;
  cudaError_t err = cudaFuncSetAttribute(velo_event_team_kernel<kTeams>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err != cudaSuccess) return (int)err;   // per device and cheap: set on every launch
  const uint32_t sms = num_sms();
  const uint32_t want = (a.n_events + kTeams - 1) / kTeams;
  const uint32_t grid = want < sms ? (want ? want : 1u) : sms;
  velo_event_team_kernel<kTeams><<<grid, kTeams * kTeamThreads, smem, stream>>>(a);
  return (int)cudaGetLastError();
  }
}

}  // namespace

int launch_event_smem(const KernelArgs& a, cudaStream_t stream, uint32_t teams) {
  if (teams == 0) {
    // Default: as many teams as mean-sized events fit the pool (about 16 bytes per hit + 5 KB per
    // event), less one because blocks of unequal size never pack perfectly: 5 for mu = 5 events of
    // 1.9 k hits, 8 for the 0.3 k-hit events of the open VELO. More teams would only wait for memory.
    const uint32_t mean = a.n_events ? a.n_hits / a.n_events : 0u;
    const uint32_t fit = (kPoolUnits * kUnitBytes) / (16u * mean + 5120u);
    teams = fit <= 5u ? 5u : (fit - 1u > kMaxTeams ? kMaxTeams : fit - 1u);
  }
  switch (teams) {
    case 1: return launch_teams<1>(a, stream);
    case 2: return launch_teams<2>(a, stream);
    case 3: return launch_teams<3>(a, stream);
    case 4: return launch_teams<4>(a, stream);
    case 6: return launch_teams<6>(a, stream);
    case 7: return launch_teams<7>(a, stream);
    case 8: return launch_teams<8>(a, stream);
    case 5:
    default: return launch_teams<5>(a, stream);
  }
}

}  // namespace velo
