// velo_kernels.cu — the general kernel of the VELO hot path and the small kernels between the stages
// of the pipeline (sm_100a; SURVEY.md §8(a) S0 ... S7).
//
// velo_event_slab_kernel: one CTA reconstructs one event at a time with every per-event array in a
// slab in global memory: S0 decode (phi16, bucket key), S1 phi sort, the 24-step module loop with S3
// forwarding and S2 search-by-triplet seeding, S4 ghost filter, S5 straight-line fit, S6 clone filter,
// then writes its surviving tracks into a temp block allocated with one atomic per event (the write
// kernel of velo_fit.cu moves it into place). It takes any legal input and the events the three-stage
// pipeline (velo_sort.cu, velo_track.cu, velo_fit.cu) gives up. Also here: velo_order_kernel (the
// order in which stages 2 and 3 take the events), velo_big_order_kernel, velo_offsets_kernel (S7:
// counts -> offsets), the workspace layout and the launch sequence of a batch.
// Step semantics: SURVEY.md §8(c) O-1 ... O-14 (restated in DESIGN.md §2); the paper itself
// (§5) names the objects but gives no step.
#include "velo_device.cuh"
#include "velo_internal.h"

namespace velo {

namespace {

constexpr int kThreads = 256;            // CTA size of the slab kernel when it takes every event of a batch
constexpr int kThreadsLarge = 1024;      // ... and when it takes the events the pipeline deferred: those are
                                         // the large ones, and a batch waits for the latency of its largest event
constexpr unsigned kInactive = 255u;     // tmiss value of a track that stopped forwarding

// Per-event arrays (sorted-hit order) and the candidate-track table. The pointers address either
// shared memory (small events) or the CTA's slab in global memory (large events).
struct Ev {
  float *sx, *sy, *sz;       // sorted hit coordinates
  int16_t* phi;              // sorted phi16
  uint16_t* perm;            // sorted position -> original event-local index
  uint8_t* flag;             // O-5 flag[h]
  unsigned long long* owner; // O-13 owner[h]
  uint32_t *stash, *tmp;     // sort scratch
  uint16_t* th;              // candidate hits, th[k * tcap + t] = k-th hit of track t (sorted idx)
  uint8_t *tn, *tmiss;       // hits on the track; consecutive misses (kInactive = stopped)
  uint16_t* tcentre;         // sorted index of the seed's centre hit
  float* tseed;              // seed scatter
  unsigned long long* tkey;  // O-13 key
  uint8_t* tpass;            // 0 dropped by O-10/O-12, 1 passed, 2 survives O-13
  uint32_t tcap;             // capacity of the track table
};

struct Shared {
  unsigned long long warp_sums[33];
  uint32_t mod_off[VELO_MAX_MODULES + 1];
  uint32_t ticket, bad, ntracks, tbase, hbase;
};

// Visits, in ascending sorted index, every hit j of module m with |int16(phi[j] - c)| <= W (O-3).
template <int kShift, class F>
__device__ __forceinline__ void for_window(const Ev& ev, const uint32_t* binoff, int m, int c, int W, F&& f) {
  if (W < 0) return;
  const uint32_t* bo = binoff + m * (65536 >> kShift);
  if (2 * (long long)W + 1 >= 65536) {
    for (uint32_t j = bo[0]; j < bo[(65536 >> kShift)]; ++j) f(j);
    return;
  }
  const int lo = c + 32768 - W, hi = c + 32768 + W;  // unsigned-phi interval, may leave [0, 65535]
  auto seg = [&](int a, int b) {
    const uint32_t j1 = bo[(b >> kShift) + 1];
    for (uint32_t j = bo[a >> kShift]; j < j1; ++j) {
      const int pu = (int)ev.phi[j] + 32768;
      if (pu >= a && pu <= b) f(j);
    }
  };
  if (lo < 0) { seg(0, hi); seg(lo + 65536, 65535); }
  else if (hi > 65535) { seg(0, hi - 65536); seg(lo, 65535); }
  else seg(lo, hi);
}

// O-11 straight-line fit of the hits of candidate t; writes the 13 state words to st[].
__device__ __forceinline__ void fit_track(const Ev& ev, uint32_t t, uint32_t n, float sig2, float inv_s2,
                                          float* st) {
  float sz = 0.0f, sx = 0.0f, sy = 0.0f;
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t h = ev.th[i * ev.tcap + t];
    sz = __fadd_rn(sz, ev.sz[h]); sx = __fadd_rn(sx, ev.sx[h]); sy = __fadd_rn(sy, ev.sy[h]);
  }
  const float nf = (float)n;
  const float zb = __fdiv_rn(sz, nf), xb = __fdiv_rn(sx, nf), yb = __fdiv_rn(sy, nf);
  float sdd = 0.0f, sdx = 0.0f, sdy = 0.0f;
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t h = ev.th[i * ev.tcap + t];
    const float d = __fsub_rn(ev.sz[h], zb);
    sdd = __fadd_rn(sdd, __fmul_rn(d, d));
    sdx = __fadd_rn(sdx, __fmul_rn(d, __fsub_rn(ev.sx[h], xb)));
    sdy = __fadd_rn(sdy, __fmul_rn(d, __fsub_rn(ev.sy[h], yb)));
  }
  const float tx = __fdiv_rn(sdx, sdd), ty = __fdiv_rn(sdy, sdd);
  float c = 0.0f;
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t h = ev.th[i * ev.tcap + t];
    const float d = __fsub_rn(ev.sz[h], zb);
    const float rx = __fsub_rn(__fsub_rn(ev.sx[h], xb), __fmul_rn(tx, d));
    const float ry = __fsub_rn(__fsub_rn(ev.sy[h], yb), __fmul_rn(ty, d));
    c = __fadd_rn(c, __fmul_rn(rx, rx));
    c = __fadd_rn(c, __fmul_rn(ry, ry));
  }
  const float chi2 = __fmul_rn(c, inv_s2);
  const float s2 = __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty));
  float dzb;
  if (s2 < 1e-12f) dzb = 0.0f;
  else dzb = -__fdiv_rn(__fadd_rn(__fmul_rn(xb, tx), __fmul_rn(yb, ty)), s2);
  const float vt = __fdiv_rn(sig2, sdd);
  const float cxtx = __fmul_rn(dzb, vt);
  const float cxx = __fadd_rn(__fdiv_rn(sig2, nf), __fmul_rn(__fmul_rn(dzb, dzb), vt));
  st[0] = __fadd_rn(xb, __fmul_rn(tx, dzb));
  st[1] = __fadd_rn(yb, __fmul_rn(ty, dzb));
  st[2] = tx; st[3] = ty;
  st[4] = __fadd_rn(zb, dzb);
  st[5] = cxx; st[6] = cxtx; st[7] = vt;
  st[8] = cxx; st[9] = cxtx; st[10] = vt;
  st[11] = chi2;
  st[12] = __uint_as_float(n);
}

__device__ __forceinline__ void set_status(uint32_t* counters, int code) {
  // first error wins; VELO_OK is 0
  atomicCAS(&counters[kCtrStatus], 0u, (uint32_t)code);
}

// Reconstructs event e with the CTA's arrays `ev`. Called by all threads of the CTA.
// binoff: histogram, then exclusive offsets of the phi buckets (kMaxBins + 1 words, in shared memory
// or in the CTA's slab).
// kShift: phi units per bucket = 1 << kShift (1024 for ordinary events; 256 for batches of large
// events, whose buckets would otherwise hold ~50 hits each and every window scan ~100).
template <int kShift>
__device__ void process_event(const KernelArgs& a, const Ev& ev, Shared& sh, uint32_t* binoff, uint32_t e) {
  constexpr uint32_t kBins = 65536u >> kShift;   // buckets per module
  const uint32_t tid = threadIdx.x, nthr = blockDim.x;
  const uint32_t M = a.n_modules;
  const uint32_t o0 = a.event_offsets[e], o1 = a.event_offsets[e + 1];
  const uint32_t nbins = M * kBins;
  const velo_params_t& P = a.P;

  // ---- input checks (VELO_ERR_INPUT): the event then contributes zero tracks -------------------
  const uint32_t obase = a.event_offsets[0];
  if (o1 < o0 || o0 < obase || o1 - obase > a.n_hits || o1 - o0 > VELO_MAX_EVENT_HITS) {   // stays inside the batch
    if (tid == 0) { set_status(a.ws.counters, VELO_ERR_INPUT); a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0); }
    return;
  }
  const uint32_t n = o1 - o0;
  // packed input: the team that deferred the event left its fp32 coordinates in the workspace
  const size_t g0 = a.pixel ? (size_t)(o0 - obase) : (size_t)(o0 - a.hit_base);
  const float* gx = (a.pixel ? a.ws.ux : a.x) + g0; const float* gy = (a.pixel ? a.ws.uy : a.y) + g0;
  const float* gz = (a.pixel ? a.ws.uz : a.z) + g0;
  const uint8_t* gm = (a.pixel ? a.ws.umod : a.module) + g0;

  // ---- S0 decode: phi16 and bucket histogram (O-1) ---------------------------------------------
  for (uint32_t b = tid; b <= nbins; b += nthr) binoff[b] = 0;
  if (tid == 0) { sh.bad = 0; sh.ntracks = 0; }
  __syncthreads();
  for (uint32_t i = tid; i < n; i += nthr) {
    const uint32_t m = gm[i];
    if (m >= M) { sh.bad = 1; continue; }
    const uint32_t pu = (uint32_t)(phi16(gx[i], gy[i]) + 32768);
    const uint32_t slot = atomicAdd(&binoff[m * kBins + (pu >> kShift)], 1u);
    ev.stash[i] = (pu << 16) | slot;
  }
  __syncthreads();
  if (sh.bad) {
    if (tid == 0) { set_status(a.ws.counters, VELO_ERR_INPUT); a.ws.ev_rec[e] = make_uint4(0, 0, 0, 0); }
    __syncthreads();
    return;
  }
  // exclusive scan of the histogram -> bucket offsets; binoff[nbins] = n
  {
    const uint32_t per = (nbins + nthr - 1) / nthr;
    const uint32_t b0 = tid * per, b1 = min(b0 + per, nbins);
    uint32_t s = 0;
    for (uint32_t b = b0; b < b1; ++b) s += binoff[b];
    unsigned long long tot;
    uint32_t run = (uint32_t)block_scan_excl(s, sh.warp_sums, &tot);
    for (uint32_t b = b0; b < b1; ++b) { const uint32_t c = binoff[b]; binoff[b] = run; run += c; }
    if (tid == 0) binoff[nbins] = n;
  }
  __syncthreads();
  for (uint32_t m = tid; m <= M; m += nthr) sh.mod_off[m] = binoff[m * kBins];

  // ---- S1 phi sort (O-2): group by bucket, then rank inside the bucket by (phi16, index) -------
  for (uint32_t i = tid; i < n; i += nthr) {
    const uint32_t st = ev.stash[i], pu = st >> 16;
    const uint32_t bin = (uint32_t)gm[i] * kBins + (pu >> kShift);
    ev.tmp[binoff[bin] + (st & 0xffffu)] = (pu << 16) | i;
  }
  __syncthreads();
  for (uint32_t i = tid; i < n; i += nthr) {
    const uint32_t pu = ev.stash[i] >> 16;
    const uint32_t bin = (uint32_t)gm[i] * kBins + (pu >> kShift);
    const uint32_t item = (pu << 16) | i;
    const uint32_t lo = binoff[bin], hi = binoff[bin + 1];
    uint32_t r = lo;
    for (uint32_t j = lo; j < hi; ++j) r += (ev.tmp[j] < item) ? 1u : 0u;
    ev.sx[r] = gx[i]; ev.sy[r] = gy[i]; ev.sz[r] = gz[i];
    ev.phi[r] = (int16_t)((int)pu - 32768);
    ev.perm[r] = (uint16_t)i;
    ev.flag[r] = 0;
    ev.owner[r] = ~0ull;
  }
  __syncthreads();

  // ---- O-6 module loop --------------------------------------------------------------------------
  for (uint32_t s = M - 2; s >= 1; --s) {
    const uint32_t u = s - 1;
    // (A) O-7 forwarding into module u of every track active at the start of the step
    const uint32_t nt0 = sh.ntracks;
    for (uint32_t t = tid; t < nt0; t += nthr) {
      const uint32_t miss = ev.tmiss[t];
      if (miss == kInactive) continue;
      const uint32_t nh = ev.tn[t];
      const uint32_t ha = ev.th[(nh - 2) * ev.tcap + t], hb = ev.th[(nh - 1) * ev.tcap + t];
      const float x1 = ev.sx[hb], y1 = ev.sy[hb], z1 = ev.sz[hb];
      const float dx = __fsub_rn(x1, ev.sx[ha]), dy = __fsub_rn(y1, ev.sy[ha]), dz = __fsub_rn(z1, ev.sz[ha]);
      bool found = false; uint32_t best = 0; float best_sc = 0.0f;
      for_window<kShift>(ev, binoff, (int)u, (int)ev.phi[hb], P.phi_window_fwd, [&](uint32_t c) {
        const float sc = scatter(dx, dy, dz, x1, y1, z1, ev.sx[c], ev.sy[c], ev.sz[c]);
        if (sc <= P.max_scatter_fwd && (!found || sc < best_sc)) { found = true; best = c; best_sc = sc; }
      });
      if (found) {
        ev.th[nh * ev.tcap + t] = (uint16_t)best;
        ev.tn[t] = (uint8_t)(nh + 1);
        ev.tmiss[t] = 0;
        if (nh + 1 == 4) { for (uint32_t i = 0; i < 3; ++i) ev.flag[ev.th[i * ev.tcap + t]] = 1; }
        if (nh + 1 >= 4) ev.flag[best] = 1;   // (B): forwarding never reads flags, so set them now
      } else {
        ev.tmiss[t] = (miss + 1 > P.max_skipped) ? (uint8_t)kInactive : (uint8_t)(miss + 1);
      }
    }
    __syncthreads();
    // (C) O-8 seeding with centre module s; one thread per centre hit, tracks numbered by a scan
    const uint32_t c_begin = sh.mod_off[s], c_end = sh.mod_off[s + 1];
    for (uint32_t c0 = c_begin; c0 < c_end; c0 += nthr) {
      const uint32_t h1 = c0 + tid;
      bool found = false; uint32_t b0 = 0, b2 = 0; float best_sc = 0.0f;
      if (h1 < c_end && !ev.flag[h1]) {
        const float x1 = ev.sx[h1], y1 = ev.sy[h1], z1 = ev.sz[h1];
        const int c = (int)ev.phi[h1];
        for_window<kShift>(ev, binoff, (int)s + 1, c, P.phi_window_seed, [&](uint32_t h0) {
          if (ev.flag[h0]) return;
          const float dx = __fsub_rn(x1, ev.sx[h0]), dy = __fsub_rn(y1, ev.sy[h0]), dz = __fsub_rn(z1, ev.sz[h0]);
          for_window<kShift>(ev, binoff, (int)s - 1, c, P.phi_window_seed, [&](uint32_t h2) {
            if (ev.flag[h2]) return;
            const float sc = scatter(dx, dy, dz, x1, y1, z1, ev.sx[h2], ev.sy[h2], ev.sz[h2]);
            if (sc <= P.max_scatter_seed && (!found || sc < best_sc)) { found = true; b0 = h0; b2 = h2; best_sc = sc; }
          });
        });
      }
      unsigned long long tot;
      const uint32_t slot = sh.ntracks + (uint32_t)block_scan_excl(found ? 1ull : 0ull, sh.warp_sums, &tot);
      if (found && slot < ev.tcap) {
        ev.th[0 * ev.tcap + slot] = (uint16_t)b0;
        ev.th[1 * ev.tcap + slot] = (uint16_t)h1;
        ev.th[2 * ev.tcap + slot] = (uint16_t)b2;
        ev.tn[slot] = 3; ev.tmiss[slot] = 0;
        ev.tseed[slot] = best_sc; ev.tcentre[slot] = (uint16_t)h1;
      }
      __syncthreads();
      if (tid == 0) sh.ntracks += (uint32_t)tot;
      __syncthreads();
    }
    __syncthreads();
  }
  const uint32_t nt = sh.ntracks;  // candidates never exceed the centre hits, hence never tcap (slab)

  // ---- O-10 ghost filter, O-11 fit, O-12 chi2 cut, O-13 owners ----------------------------------
  const float sig2 = __fmul_rn(P.sigma_hit, P.sigma_hit);
  const float inv_s2 = __fdiv_rn(1.0f, sig2);
  for (uint32_t t = tid; t < nt; t += nthr) {
    const uint32_t nh = ev.tn[t];
    bool pass = true;
    if (nh == 3) {
      if (ev.flag[ev.th[t]] || ev.flag[ev.th[ev.tcap + t]] || ev.flag[ev.th[2 * ev.tcap + t]]) pass = false;
      if (!(ev.tseed[t] <= P.max_scatter_weak)) pass = false;
    }
    unsigned long long key = 0;
    if (pass) {
      float st[VELO_N_STATE];
      fit_track(ev, t, nh, sig2, inv_s2, st);
      const float lim = __fmul_rn(P.max_chi2_ndof, (float)(2 * (int)nh - 4));
      if (st[11] > lim) pass = false;
      key = ((unsigned long long)(255u - nh) << 56) | ((unsigned long long)__float_as_uint(st[11]) << 24) |
            (unsigned long long)ev.tcentre[t];
    }
    ev.tpass[t] = pass ? 1 : 0;
    ev.tkey[t] = key;
    if (pass) for (uint32_t i = 0; i < nh; ++i) atomicMin(&ev.owner[ev.th[i * ev.tcap + t]], key);
  }
  __syncthreads();
  // ---- O-13 clone filter; per-thread totals of survivors --------------------------------------
  uint32_t my_t = 0, my_h = 0;
  for (uint32_t t = tid; t < nt; t += nthr) {
    if (!ev.tpass[t]) continue;
    const uint32_t nh = ev.tn[t];
    const unsigned long long key = ev.tkey[t];
    uint32_t lost = 0;
    for (uint32_t i = 0; i < nh; ++i) lost += (ev.owner[ev.th[i * ev.tcap + t]] != key) ? 1u : 0u;
    if (!((unsigned long long)lost * P.clone_den > (unsigned long long)nh * P.clone_num)) {
      ev.tpass[t] = 2; my_t += 1; my_h += nh;
    }
  }
  // ---- S7 part 1: allocate the event's temp block, write survivors in creation order -----------
  unsigned long long tot;
  block_scan_excl(((unsigned long long)my_h << 32) | my_t, sh.warp_sums, &tot);
  const uint32_t ev_nt = (uint32_t)(tot & 0xffffffffu), ev_nh = (uint32_t)(tot >> 32);
  if (tid == 0) {
    sh.tbase = atomicAdd(&a.ws.counters[kCtrTracks], ev_nt);
    sh.hbase = atomicAdd(&a.ws.counters[kCtrHits], ev_nh);
    atomicAdd(&a.ws.counters[kCtrCand], nt);
    a.ws.ev_rec[e] = make_uint4(sh.tbase, sh.hbase, ev_nt, ev_nh);
  }
  __syncthreads();
  const uint32_t tbase = sh.tbase, hbase = sh.hbase;
  const bool fits = (unsigned long long)tbase + ev_nt <= a.cap_tracks &&
                    (unsigned long long)hbase + ev_nh <= a.cap_track_hits;
  unsigned long long run = 0;  // (hits << 32 | tracks) written so far
  for (uint32_t t0 = 0; t0 < nt; t0 += nthr) {
    const uint32_t t = t0 + tid;
    const bool surv = t < nt && ev.tpass[t] == 2;
    const uint32_t nh = surv ? ev.tn[t] : 0;
    unsigned long long ctot;
    const unsigned long long pre = run + block_scan_excl(surv ? (((unsigned long long)nh << 32) | 1ull) : 0ull,
                                                         sh.warp_sums, &ctot);
    run += ctot;
    if (surv && fits) {
      const uint32_t lt = (uint32_t)(pre & 0xffffffffu), lh = (uint32_t)(pre >> 32);
      float st[VELO_N_STATE];
      fit_track(ev, t, nh, sig2, inv_s2, st);
#pragma unroll
      for (int k = 0; k < VELO_N_STATE; ++k) a.ws.tmp_states[(size_t)k * a.cap_tracks + tbase + lt] = st[k];
      a.ws.tmp_loff[tbase + lt] = lh;
      for (uint32_t i = 0; i < nh; ++i) a.ws.tmp_hits[hbase + lh + i] = o0 + ev.perm[ev.th[i * ev.tcap + t]];
    }
  }
  __syncthreads();
}

// ---- event kernel, slab variant: persistent CTAs pull events from a ticket counter -------------
// from_list = 0: every event of the batch; 1: the events the shared-memory kernel deferred (ws.large_list).
// kBinsInSlab: the bucket table lives in the slab too, so that the CTA needs almost no shared memory
// and fits beside the pipeline kernels of the next batch (the usual case: nothing was deferred).
template <int kCta, bool kBinsInSlab, int kShift>
__global__ void __launch_bounds__(kCta) velo_event_slab_kernel(const KernelArgs a, const int from_list) {
  static_assert(!kBinsInSlab || kShift == kBinShift, "the slab's bucket table is sized for the default buckets");
  __shared__ Shared sh;
  __shared__ uint32_t bins_smem[kBinsInSlab ? 1 : VELO_MAX_MODULES * (65536 >> kShift) + 1];
  const SlabLayout L = slab_layout();
  unsigned char* slab = a.ws.slabs + (size_t)blockIdx.x * L.bytes;
  Ev ev;
  ev.sx = (float*)(slab + L.sx); ev.sy = (float*)(slab + L.sy); ev.sz = (float*)(slab + L.sz);
  ev.phi = (int16_t*)(slab + L.phi); ev.perm = (uint16_t*)(slab + L.perm); ev.flag = slab + L.flag;
  ev.owner = (unsigned long long*)(slab + L.owner);
  ev.stash = (uint32_t*)(slab + L.stash); ev.tmp = (uint32_t*)(slab + L.tmp);
  ev.th = (uint16_t*)(slab + L.th); ev.tn = slab + L.tn; ev.tmiss = slab + L.tmiss;
  ev.tcentre = (uint16_t*)(slab + L.tcentre); ev.tseed = (float*)(slab + L.tseed);
  ev.tkey = (unsigned long long*)(slab + L.tkey); ev.tpass = slab + L.tpass;
  ev.tcap = kSlabHits;
  const uint32_t limit = from_list ? a.ws.counters[kCtrLargeN] : a.n_events;
  for (;;) {
    if (threadIdx.x == 0) sh.ticket = atomicAdd(&a.ws.counters[from_list ? kCtrLargeTicket : kCtrTicket], 1u);
    __syncthreads();
    const uint32_t k = sh.ticket;
    __syncthreads();
    if (k >= limit) break;
    process_event<kShift>(a, ev, sh, kBinsInSlab ? (uint32_t*)(slab + L.bins) : bins_smem, from_list ? a.ws.large_list[k] : k);
  }
}

// ---- processing order for stages 2 and 3: event ids by ascending size class ------------------------
// Events of a batch differ in size by more than 10x. Stages 2 and 3 hand out the sorted list
// from both ends in turn (largest, smallest, second largest, ...), so the handful of events that
// share an SM's shared memory at any time add up to about the same bytes and the pool neither
// overflows (teams waiting for memory) nor sits half empty. Counting sort by n_hits / 64: the counts
// per class come from stage 1 (its team leaders add one per event to ws.size_hist), every CTA here
// scans the 256 counts for itself and places its own 256 events behind the class's global cursor
// (one CTA doing all of it took 37 us per 25 000-event batch with the other 147 SMs idle).
// The order only schedules: results and their placement do not depend on it.
__global__ void __launch_bounds__(kSizeClasses) velo_order_kernel(const KernelArgs a) {
  __shared__ uint32_t base[kSizeClasses];
  __shared__ uint32_t wsum[kSizeClasses / 32];
  const uint32_t tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5, ne = a.n_events;
  const uint32_t v = a.ws.size_hist[tid];
  uint32_t inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= (uint32_t)d) inc += o; }
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  uint32_t before = 0;
#pragma unroll
  for (uint32_t k = 0; k < kSizeClasses / 32; ++k) before += k < wid ? wsum[k] : 0u;
  base[tid] = before + inc - v;
  __syncthreads();
  const uint32_t e = blockIdx.x * kSizeClasses + tid;
  if (e >= ne) return;
  const uint32_t c = size_class(a.event_offsets[e], a.event_offsets[e + 1]);
  a.ws.order[base[c] + atomicAdd(&a.ws.size_hist[kSizeClasses + c], 1u)] = e;
}

// ---- S7 part 2: exclusive scans of the per-event counts -----------------------------------------
// CTA c owns events [c * chunk, (c + 1) * chunk), chunk = 256 * per. It first adds up the counts of every
// event before its chunk (its own copy of the prefix: the loads are independent and come from L2, so no CTA
// waits for another; 25 000 events: 98 CTAs, at most 97 loads per thread), then scans its chunk. One CTA
// scanning the whole batch was a chain of global-memory latencies: 48 us per batch with 147 SMs idle.
constexpr uint32_t kOffsetsThreads = 256;
__device__ __forceinline__ unsigned long long ev_counts(const uint4* ev_rec, uint32_t e) {   // {tracks, track hits}
  const uint2 r = *reinterpret_cast<const uint2*>(reinterpret_cast<const uint32_t*>(ev_rec + e) + 2);
  return ((unsigned long long)r.y << 32) | r.x;
}
__global__ void __launch_bounds__(kOffsetsThreads) velo_offsets_kernel(const KernelArgs a, const uint32_t per) {
  __shared__ unsigned long long warp_sums[33];
  const uint32_t tid = threadIdx.x, ne = a.n_events;
  const uint32_t c0 = min(blockIdx.x * kOffsetsThreads * per, ne);
  unsigned long long s = 0;
#pragma unroll 8
  for (uint32_t e = tid; e < c0; e += kOffsetsThreads) s += ev_counts(a.ws.ev_rec, e);
  unsigned long long before;
  block_scan_excl(s, warp_sums, &before);
  const uint32_t e0 = min(c0 + tid * per, ne), e1 = min(e0 + per, ne);
  s = 0;
  for (uint32_t e = e0; e < e1; ++e) s += ev_counts(a.ws.ev_rec, e);
  unsigned long long tot;
  unsigned long long run = before + block_scan_excl(s, warp_sums, &tot);
  for (uint32_t e = e0; e < e1; ++e) {
    a.event_track_offsets[e] = (uint32_t)(run & 0xffffffffu);
    a.ws.ev_hit_base[e] = (uint32_t)(run >> 32);
    run += ev_counts(a.ws.ev_rec, e);
  }
  if (blockIdx.x == gridDim.x - 1 && tid == 0) {     // the last chunk ends the batch: totals, summary
    tot += before;
    const uint32_t n_tracks = (uint32_t)(tot & 0xffffffffu), n_hits = (uint32_t)(tot >> 32);
    a.event_track_offsets[ne] = n_tracks;
    a.ws.ev_hit_base[ne] = n_hits;
    uint32_t status = a.ws.counters[kCtrStatus];
    const bool over = n_tracks > a.cap_tracks || n_hits > a.cap_track_hits;
    if (status == 0 && over) status = (uint32_t)VELO_ERR_CAPACITY;
    if (!over) a.track_hit_offsets[n_tracks] = n_hits;
    a.summary[0] = n_tracks; a.summary[1] = n_hits; a.summary[2] = status;
    a.summary[3] = a.ws.counters[kCtrCand];
    a.summary[4] = a.ws.counters[kCtrLargeN];
    a.summary[5] = a.ws.counters[kCtrBigN];
    a.summary[6] = a.summary[7] = 0;
  }
}

// The events of the one-event-per-CTA pipeline, largest first: an event's time grows faster than its
// size, so the longest must start first. Rank by counting (a few hundred events; one CTA).
__global__ void __launch_bounds__(1024) velo_big_order_kernel(const KernelArgs a) {
  const uint32_t nb = a.ws.counters[kCtrBigN];
  for (uint32_t i = threadIdx.x; i < nb; i += blockDim.x) {
    const uint32_t e = a.ws.big_list[i], n = a.event_offsets[e + 1] - a.event_offsets[e];
    uint32_t rank = 0;
    for (uint32_t j = 0; j < nb; ++j) {
      const uint32_t ej = a.ws.big_list[j], nj = a.event_offsets[ej + 1] - a.event_offsets[ej];
      rank += (nj > n || (nj == n && j < i)) ? 1u : 0u;
    }
    a.ws.big_sorted[rank] = e;
  }
}

// Packed input on the slab-only path: every event is decoded into the workspace planes first.
__global__ void __launch_bounds__(256) velo_unpack_kernel(const KernelArgs a) {
  for (uint32_t e = blockIdx.x; e < a.n_events; e += gridDim.x) {
    const uint32_t base = a.event_offsets[0], o0 = a.event_offsets[e], o1 = a.event_offsets[e + 1];
    if (o1 < o0 || o0 < base || o1 - base > a.n_hits) continue;       // reported by the event kernel
    unpack_event<256>(a, e, threadIdx.x);
  }
}

}  // namespace

// ---- host side -----------------------------------------------------------------------------------
uint32_t num_sms() {
  int dev = 0, sms = 0;   // per current device (a process may use several GPUs); the query is cheap
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
    cudaGetLastError();
    return 148u;
  }
  return (uint32_t)sms;
}

uint32_t default_n_slabs() { return num_sms() * 2u; }   // two 1024-thread CTAs of the general kernel fit an SM

Workspace carve_workspace(void* base, uint32_t n_events, uint32_t n_hits, uint32_t cap_tracks, uint32_t cap_track_hits,
                          uint32_t n_slabs) {
  Workspace w{};
  size_t o = 0;
  unsigned char* b = (unsigned char*)base;
  auto take = [&](size_t bytes) { size_t r = o; o += ((bytes + 255) / 256) * 256; return b + r; };
  w.counters = (uint32_t*)take(sizeof(uint32_t) * kNumCounters);                 // offset 0
  w.phase_clk = (unsigned long long*)take(sizeof(unsigned long long) * kNumPhaseClocks);   // offset 256
  w.size_hist = (uint32_t*)take(sizeof(uint32_t) * 2 * kSizeClasses);   // offset 768: one memset covers counters .. size_hist
  w.ev_info = (EvInfo*)take(sizeof(EvInfo) * ((size_t)n_events + 1));
  w.ev_rec = (uint4*)take(sizeof(uint4) * ((size_t)n_events + 1));
  w.ev_hit_base = (uint32_t*)take(4 * ((size_t)n_events + 1));
  w.large_list = (uint32_t*)take(4 * ((size_t)n_events + 1));
  w.big_list = (uint32_t*)take(4 * ((size_t)n_events + 1));
  w.big_sorted = (uint32_t*)take(4 * ((size_t)n_events + 1));
  w.order = (uint32_t*)take(4 * ((size_t)n_events + 1));
  const size_t sc = sorted_capacity(n_events, n_hits);
  w.rec16 = (uint4*)take(16 * sc);
  w.sorig = (uint16_t*)take(2 * sc);
  w.mod_off = (uint16_t*)take(2 * (size_t)kModOffStride * ((size_t)n_events + 1));
  w.flag_bits = (uint32_t*)take(4 * flag_words(n_events, n_hits));
  w.cand_total = (size_t)(n_hits >> 3) + (n_hits >> 4) + 48ull * n_events + 64ull;   // >= sum of cand_capacity(n_e)
  w.rows = (uint16_t*)take(64 * w.cand_total);
  w.rows_xy = (float2*)take(sizeof(float2) * kXyStride * w.cand_total);
  w.cmeta = (uint2*)take(8 * w.cand_total);
  w.cfit = (float*)take(4 * 9 * w.cand_total);
  w.cstate = (uint8_t*)take(w.cand_total);
  w.ux = (float*)take(4 * ((size_t)n_hits + 1)); w.uy = (float*)take(4 * ((size_t)n_hits + 1));
  w.uz = (float*)take(4 * ((size_t)n_hits + 1)); w.umod = (uint8_t*)take((size_t)n_hits + 1);
  w.tmp_loff = (uint32_t*)take(4 * ((size_t)cap_tracks + 1));
  w.tmp_hits = (uint32_t*)take(4 * ((size_t)cap_track_hits + 1));
  w.tmp_states = (float*)take(4 * (size_t)VELO_N_STATE * ((size_t)cap_tracks + 1));
  w.n_slabs = n_slabs;
  w.slabs = take((size_t)n_slabs * slab_layout().bytes);
  w.bytes = o;
  return w;
}

int launch_reconstruct(const KernelArgs& a_in, cudaStream_t stream, void* const* stage_events, uint32_t path,
                       const PipeOpts& po) {
  KernelArgs a = a_in;
  a.all_deferred = path == kPathSlabOnly ? 1u : 0u;
  // The one-event-per-CTA kernels are launched only for batches that can hold events above the pool's
  // reach (a mean event above a quarter of kPipeMaxHits): three launches that a mu = 5 batch would only
  // pay for. Without them such events take the general kernel, with the same results.
  // (not with two sensor planes per module: the records' plane bit needs modules of fewer than 32768 hits)
  a.big_path = path != kPathSlabOnly && !a.two_plane && a.n_events > 0 &&
               (unsigned long long)a.n_hits * 4ull > (unsigned long long)kPipeMaxHits * a.n_events ? 1u : 0u;
  auto mark = [&](int k) { if (stage_events && stage_events[k]) cudaEventRecord((cudaEvent_t)stage_events[k], stream); };
  cudaError_t err = cudaMemsetAsync(a.ws.counters, 0, (size_t)((unsigned char*)(a.ws.size_hist + 2 * kSizeClasses) - (unsigned char*)a.ws.counters), stream);
  if (err != cudaSuccess) return (int)err;
#ifdef VELO_TIMELINE
  cudaMemsetAsync(a.ws.phase_clk, 0, sizeof(unsigned long long) * kNumPhaseClocks, stream);
#endif
  mark(0);
  const uint32_t grid = a.n_events ? (a.ws.n_slabs < a.n_events ? a.ws.n_slabs : a.n_events) : 0u;
  const bool large_events = a.n_events && a.n_hits / a.n_events >= 4096u;
  if (a.n_events > 0) {
    if (path == kPathSlabOnly) {
      if (a.pixel) velo_unpack_kernel<<<num_sms() * 8u, 256, 0, stream>>>(a);
      mark(1);
      velo_event_slab_kernel<kThreads, false, kBinShift><<<grid, kThreads, 0, stream>>>(a, 0);
    } else {
      // stage 1: sort; stage 2: module loop (events by size, largest first); then the general kernel
      // for whatever the pipeline deferred (usually nothing: its CTAs come and go); stage 3 below
      int rc = launch_sort(a, stream, po);
      if (rc != 0) return rc;
      if (a.big_path) {
        if ((rc = launch_sort_big(a, stream)) != 0) return rc;
        velo_big_order_kernel<<<1, 1024, 0, stream>>>(a);
      }
      velo_order_kernel<<<(a.n_events + kSizeClasses - 1u) / kSizeClasses, kSizeClasses, 0, stream>>>(a);
      mark(1);
      rc = launch_track(a, stream, po);
      if (rc != 0) return rc;
      if (a.big_path && (rc = launch_track_big(a, stream)) != 0) return rc;
      if (large_events) velo_event_slab_kernel<kThreadsLarge, false, 8><<<grid, kThreadsLarge, 0, stream>>>(a, 1);
      else velo_event_slab_kernel<kThreads, true, kBinShift><<<grid, kThreads, 0, stream>>>(a, 1);
    }
  } else {
    mark(1);
  }
  mark(2);
  if (path != kPathSlabOnly) {
    int rc = launch_fit(a, stream, po);   // fit and filters: per-candidate results, per-event counts
    if (rc != 0) return rc;
    if (a.big_path && a.n_events > 0 && (rc = launch_fit_big(a, stream)) != 0) return rc;
  }
  mark(3);
  {
    // counts -> event_track_offsets, summary: at most one CTA per SM, a thread takes `per` events
    const uint32_t per = (a.n_events + kOffsetsThreads * num_sms() - 1u) / (kOffsetsThreads * num_sms());
    const uint32_t chunk = kOffsetsThreads * (per ? per : 1u);
    const uint32_t ctas = (a.n_events + chunk - 1u) / chunk;
    velo_offsets_kernel<<<ctas ? ctas : 1u, kOffsetsThreads, 0, stream>>>(a, per ? per : 1u);
  }
  mark(4);
  const int rc = launch_write(a, stream);          // every final array, once
  mark(5);
  return rc != 0 ? rc : (int)cudaGetLastError();
}

}  // namespace velo
