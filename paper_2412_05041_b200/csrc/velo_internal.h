// velo_internal.h — host/device shared declarations of libvelo (workspace layout, kernel
// arguments, launchers). Internal to paper_2412_05041_b200/csrc.
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/velo.h"

namespace velo {

// Phi bins per module of the per-event bucket table (S1 sort and the O-3 window lookup):
// bin = module * kBinsPerModule + ((phi16 + 32768) >> kBinShift).
constexpr int kBinShift = 10;
constexpr int kBinsPerModule = 65536 >> kBinShift;  // 64
constexpr int kMaxBins = VELO_MAX_MODULES * kBinsPerModule;

// ---- large-event slab: per-CTA scratch in global memory (L2-resident in practice) -------------
// One slab holds every per-event array of the path for an event of up to kSlabHits hits.
constexpr uint32_t kSlabHits = 65536;  // >= VELO_MAX_EVENT_HITS, and a multiple of 64
struct SlabLayout {                    // byte offsets inside a slab
  size_t sx, sy, sz, phi, perm, flag, owner, stash, tmp;            // per sorted hit
  size_t th, tn, tmiss, tcentre, tseed, tkey, tpass;                // per candidate track
  size_t bins;                                                      // phi-bucket table (when not in shared memory)
  size_t bytes;
};
__host__ __device__ inline SlabLayout slab_layout() {
  SlabLayout L{};
  size_t o = 0;
  const size_t H = kSlabHits;
  auto take = [&](size_t elem) { size_t r = o; o += ((elem * H + 255) / 256) * 256; return r; };
  L.sx = take(4); L.sy = take(4); L.sz = take(4); L.phi = take(2); L.perm = take(2); L.flag = take(1);
  L.owner = take(8); L.stash = take(4); L.tmp = take(4);
  L.th = take(2 * VELO_MAX_MODULES); L.tn = take(1); L.tmiss = take(1); L.tcentre = take(2);
  L.tseed = take(4); L.tkey = take(8); L.tpass = take(1);
  L.bins = o; o += ((sizeof(uint32_t) * (kMaxBins + 1) + 255) / 256) * 256;
  L.bytes = o;
  return L;
}

// ---- workspace layout (device) ---------------------------------------------------------------
// counters: u32[16]: 0 tracks allocated, 1 track-hits allocated, 2 status, 3 candidates,
//           4 event ticket, 5 large-event list length, 6 large-event ticket
enum { kCtrTracks = 0, kCtrHits = 1, kCtrStatus = 2, kCtrCand = 3, kCtrTicket = 4, kCtrLargeN = 5,
       kCtrLargeTicket = 6, kCtrSortTicket = 7, kCtrTrackTicket = 8, kCtrFitTicket = 9, kCtrCandAlloc = 10,
       kCtrBigN = 11, kCtrBigSortTicket = 12, kCtrBigTrackTicket = 13, kCtrBigFitTicket = 14,
       kNumCounters = 16, kNumPhaseClocks = 64,
       kSizeClasses = 256 };   // events by n_hits / 64 (velo_order_kernel); ws.size_hist: counts, then cursors

// ---- the three-stage pipeline (velo_sort.cu -> velo_track.cu -> velo_fit.cu) ---------------------
// Stage 1 writes every event's phi-sorted hits to global scratch; stage 2 streams them module by
// module into shared memory (TMA) and writes candidate tracks; stage 3 fits, filters and writes the
// final arrays. Scratch index of sorted hit h of event e: sorted_base(e) + h, with sorted_base(e) =
// align8(event_offsets[e] - event_offsets[0]) + 16 e: disjoint slots whose 2-, 8- and 16-byte
// element arrays all start 16-byte aligned and leave room to round a bulk copy up to 16 bytes.
__host__ __device__ inline uint32_t sorted_base(uint32_t o0_local, uint32_t e) { return ((o0_local + 7u) & ~7u) + 16u * e; }
__host__ __device__ inline size_t sorted_capacity(uint32_t n_events, uint32_t n_hits) { return (size_t)n_hits + 16ull * n_events + 32ull; }
// Flag bits of event e start at word (o0_local >> 5) + e (disjoint for consecutive events).
__host__ __device__ inline size_t flag_words(uint32_t n_events, uint32_t n_hits) { return (size_t)(n_hits >> 5) + n_events + 2ull; }
// Candidate-table capacity of an event of n hits in the pipeline path (candidates ~0.107/hit at
// mu = 5, 0.19/hit for the open VELO; an event that needs more is deferred to the general kernel).
__host__ __device__ inline uint32_t cand_capacity(uint32_t n) { return ((n >> 3) + (n >> 4) + 32u + 15u) & ~15u; }
// Shared-memory part of the active-track list (tracks alive at the same time: 0.07/hit at the peak
// of a mean mu = 5 event, 0.104/hit at most in 600 events of configs[1]): what does not fit spills
// to global scratch (velo_track.cu), so this capacity trades shared memory against rare L2 trips.
__host__ __device__ inline uint32_t active_capacity(uint32_t n) { return (((n * 7u) >> 7) + 24u + 7u) & ~7u; }
// Size class of an event for the scheduling order of stages 2 and 3 (velo_order_kernel): n_hits / 64, capped.
__host__ __device__ inline uint32_t size_class(uint32_t o0, uint32_t o1) {
  const uint32_t c = (o1 >= o0 ? o1 - o0 : 0u) >> 6;
  return c < (uint32_t)kSizeClasses - 1u ? c : (uint32_t)kSizeClasses - 1u;
}
constexpr uint32_t kModOffStride = 40;   // u16 per event: mod_off[0 .. M] (M <= 32), [39] = largest module
constexpr uint32_t kPipeMaxHits = 12000; // largest event the pipeline path takes (stage 1: 17 B/hit, stage 3: ~18 B/hit of shared memory)
// Upper bound of stage 3's shared-memory block for an event of n hits (velo_fit.cu: fit_layout with
// every candidate slot used): stage 1 defers an event to the general kernel if this does not fit.
__host__ __device__ inline uint32_t fit_smem_bound(uint32_t n) { return 4u * n + (n >> 3) + 45u * cand_capacity(n) + 256u; }
// (x, y) of a candidate's hits in discovery order, written by stage 2 as it appends them: stage 3
// fits from these rows and needs no gather. kXyStride float2 per candidate (16-byte aligned rows).
constexpr uint32_t kXyStride = VELO_MAX_MODULES;
// Two-plane geometries (at most 30 modules, so at most 30 hits per candidate): the row's last entry holds,
// as a bit pattern, which of its module's two planes each hit lies on (bit m = side of the hit in module m).
constexpr uint32_t kSideSlot = kXyStride - 1u;
constexpr uint32_t kTwoPlaneMaxModules = 30;
// per-event state written by stage 1, updated by stage 2
// kEvBig: an event of more than kPipeMaxHits hits. It runs through the same three stages in their
// one-event-per-CTA form (velo_*_big_kernel: the sort's and the fit's per-event arrays in a global
// slab instead of shared memory, the module loop reading the sorted records from L2 instead of a ring).
enum { kEvEmpty = 0, kEvReady = 1, kEvDeferred = 2, kEvBad = 3, kEvBig = 4 };
struct EvInfo { uint32_t n, state, cbase, ncand; };   // cbase: first candidate slot; ncand: candidates created

struct Workspace {
  uint32_t* counters;     // kNumCounters
  EvInfo* ev_info;        // n_events
  uint4* rec16;           // sorted_capacity: {x, y, phi16u << 16 | start(m+1), start(m-1) << 16 | start(m-2)}
  float2* rows_xy;        // cand_total * kXyStride: (x, y) of the candidates' hits, discovery order
  uint16_t* sorig;        // sorted_capacity: sorted position -> original event-local index
  uint16_t* mod_off;      // n_events * kModOffStride
  uint32_t* flag_bits;    // flag_words: final O-5 flags, one bit per sorted hit
  uint16_t* rows;         // cand_total * 32: hit lists (sorted indices) of the candidates
  uint2* cmeta;           // cand_total: {module mask of the hits, seed scatter bits}
  size_t cand_total;      // capacity of rows / cmeta in candidates
  float* cfit;            // 9 planes of cand_total: fitted state words of the candidates (stage 3)
  uint8_t* cstate;        // cand_total: 1 = the candidate survives every filter
  unsigned long long* phase_clk;  // kNumPhaseClocks SM-clock accumulators (written only by -DVELO_PHASE_CLOCKS builds)
  uint4* ev_rec;          // n_events: {temp track base, temp hit base, n_tracks, n_track_hits}
  uint32_t* ev_hit_base;  // n_events+1: exclusive scan of n_track_hits over events
  uint32_t* large_list;   // n_events: events deferred to the slab path
  uint32_t* big_list;     // n_events: events of more than kPipeMaxHits hits (the one-event-per-CTA pipeline)
  uint32_t* big_sorted;   // n_events: the same, largest first (stages 2 and 3 take them in this order)
  uint32_t* order;        // n_events: event ids by ascending size class (velo_order_kernel)
  uint32_t* size_hist;    // 2 * kSizeClasses: events per size class (counted by stage 1's leaders), placement cursors
  float *ux, *uy, *uz;    // n_hits: fp32 coordinates of deferred events when the input is packed pixels
  uint8_t* umod;          //   (index = absolute hit index - event_offsets[0])
  uint32_t* tmp_loff;     // cap_tracks: hit offset of a track inside its event's hit block
  uint32_t* tmp_hits;     // cap_track_hits
  float* tmp_states;      // VELO_N_STATE * cap_tracks
  unsigned char* slabs;   // n_slabs * slab bytes
  uint32_t n_slabs;
  size_t bytes;
};
Workspace carve_workspace(void* base, uint32_t n_events, uint32_t n_hits, uint32_t cap_tracks, uint32_t cap_track_hits,
                          uint32_t n_slabs);
uint32_t default_n_slabs();
uint32_t num_sms();  // SM count of the current device (148 on B200); 148 if no device is present

struct KernelArgs {
  // input
  const float *x, *y, *z;
  const uint8_t* module;
  const uint32_t* pixel;             // packed pixel addresses instead of x, y, z, module (velo_pixel_hits_t), or NULL
  double pitch, half_shift_x;        //   their format (velo_pixel_format_t)
  const uint32_t* event_offsets;
  uint32_t n_events, n_modules;
  uint32_t n_hits;                   // host knowledge of the batch size: sizes the scratch, steers launch heuristics
  uint32_t hit_base;                 // x, y, z, module point at absolute hit index hit_base (0 for velo_reconstruct)
  uint32_t team_max_hits;            // events with more hits go to the general kernel
  uint32_t all_deferred;             // slab-only path: every event was reconstructed by the general kernel
  uint32_t big_path;                 // events above team_max_hits take the one-event-per-CTA pipeline (else the general kernel)
  float module_z[VELO_MAX_MODULES];  // geometry: the shared-memory path requires z[i] == module_z[module[i]]
  float module_z_b[VELO_MAX_MODULES];// ... or, with two_plane, == module_z_b[module[i]] (the station's second sensor: side 1)
  uint32_t two_plane;
  velo_params_t P;
  // output
  uint32_t* event_track_offsets;
  uint32_t* track_hit_offsets;
  uint32_t* track_hits;
  float* states;
  uint32_t cap_tracks, cap_track_hits;
  uint32_t* summary;
  Workspace ws;
};

#ifdef __CUDACC__
}  // namespace velo
#include "velo_device.cuh"
namespace velo {
// Packed input: an event that leaves the pipeline for the general kernel is first decoded into the
// workspace's fp32 planes by the team that gives it up (G threads, thread `tid`).
template <int G>
__device__ inline void unpack_event(const KernelArgs& a, uint32_t e, uint32_t tid) {
  const uint32_t base = a.event_offsets[0], o0 = a.event_offsets[e], n = a.event_offsets[e + 1] - o0;
  const uint32_t* src = a.pixel + (size_t)(o0 - a.hit_base);
  const size_t d0 = (size_t)(o0 - base);
  for (uint32_t i = tid; i < n; i += G) {
    uint32_t m; float x, y;
    pixel_decode(src[i], a.pitch, a.half_shift_x, m, x, y);
    a.ws.ux[d0 + i] = x; a.ws.uy[d0 + i] = y;
    a.ws.uz[d0 + i] = m < a.n_modules ? a.module_z[m] : 0.0f;
    a.ws.umod[d0 + i] = (uint8_t)(m < 256u ? m : 255u);
  }
}
#endif

// Which event kernel(s) a batch runs through (velo_launch_options_t.path).
enum { kPathDefault = 0,     // three-stage pipeline, slab kernel for the events it defers
       kPathSlabOnly = 1 };  // slab kernel for every event (the general path on its own)

// Launch geometry of the pipeline kernels (0 = default), from velo_launch_options_t.
struct PipeOpts { uint32_t track_group, track_teams, fit_teams, sort_teams, pool_units; };
int launch_sort(const KernelArgs& a, cudaStream_t stream, const PipeOpts& o);
int launch_track(const KernelArgs& a, cudaStream_t stream, const PipeOpts& o);
int launch_fit(const KernelArgs& a, cudaStream_t stream, const PipeOpts& o);
int launch_write(const KernelArgs& a, cudaStream_t stream);
// The same stages for the events on ws.big_list: one event per CTA.
int launch_sort_big(const KernelArgs& a, cudaStream_t stream);
int launch_track_big(const KernelArgs& a, cudaStream_t stream);
int launch_fit_big(const KernelArgs& a, cudaStream_t stream);

// Enqueues the whole path for one batch on `stream`. Returns a cudaError_t as int.
int launch_reconstruct(const KernelArgs& a, cudaStream_t stream, void* const* stage_events, uint32_t path,
                       const PipeOpts& po);

}  // namespace velo
struct velo_geometry {
  uint32_t n_modules;
  float module_z[VELO_MAX_MODULES];
  float module_z_b[VELO_MAX_MODULES];
  uint32_t two_plane;
  float r_in, r_out, pitch, half_shift_x;
};
namespace velo {

// velo_reconstruct with the hit planes pointing at absolute hit index `hit_base` instead of 0 (the
// scheduler's device buffers hold one batch's slice; emitted track_hits stay absolute indices).
int reconstruct_impl(const velo_geometry_t* g, const velo_hits_t* hits, const velo_params_t* params,
                     velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream,
                     const velo_launch_options_t* opts, uint32_t hit_base);
// The same over packed pixel addresses (hits->pixel points at absolute hit index `hit_base`).
int reconstruct_pixels_impl(const velo_geometry_t* g, const velo_pixel_hits_t* hits, const velo_pixel_format_t* fmt,
                            const velo_params_t* params, velo_tracks_t* out, void* workspace, size_t workspace_bytes,
                            void* stream, const velo_launch_options_t* opts, uint32_t hit_base);

}  // namespace velo
