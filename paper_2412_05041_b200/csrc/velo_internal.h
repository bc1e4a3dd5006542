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

// ---- per-team scratch of the shared-memory team kernel (velo_event_smem.cu) --------------------
// The candidates' hit lists (32 x u16 per candidate) and fitted states (9 x f32) of the event a
// team is working on. Rewritten for every event, so it stays L2-resident.
constexpr uint32_t kTeamMaxHits = 13312;                       // largest event the team path takes
constexpr uint32_t kTeamMaxTracks = kTeamMaxHits / 8 + 64;     // >= its candidate-table capacity
constexpr uint32_t kTeamScratchBytes = kTeamMaxTracks * (64 + 36);
constexpr uint32_t kTeamsPerCtaMax = 8;

// ---- workspace layout (device) ---------------------------------------------------------------
// counters: u32[16]: 0 tracks allocated, 1 track-hits allocated, 2 status, 3 candidates,
//           4 event ticket, 5 large-event list length, 6 large-event ticket
enum { kCtrTracks = 0, kCtrHits = 1, kCtrStatus = 2, kCtrCand = 3, kCtrTicket = 4, kCtrLargeN = 5,
       kCtrLargeTicket = 6, kNumCounters = 16, kNumPhaseClocks = 32 };

struct Workspace {
  uint32_t* counters;     // kNumCounters
  unsigned long long* phase_clk;  // kNumPhaseClocks SM-clock accumulators (written only by -DVELO_PHASE_CLOCKS builds)
  uint4* ev_rec;          // n_events: {temp track base, temp hit base, n_tracks, n_track_hits}
  uint32_t* ev_hit_base;  // n_events+1: exclusive scan of n_track_hits over events
  uint32_t* large_list;   // n_events: events deferred to the slab path
  uint32_t* order;        // n_events: event ids by ascending size class (velo_order_kernel)
  uint32_t* tmp_loff;     // cap_tracks: hit offset of a track inside its event's hit block
  uint32_t* tmp_hits;     // cap_track_hits
  float* tmp_states;      // VELO_N_STATE * cap_tracks
  unsigned char* team_scratch;  // num_sms * kTeamsPerCtaMax * kTeamScratchBytes
  unsigned char* slabs;   // n_slabs * slab bytes
  uint32_t n_slabs;
  size_t bytes;
};
Workspace carve_workspace(void* base, uint32_t n_events, uint32_t cap_tracks, uint32_t cap_track_hits,
                          uint32_t n_slabs);
uint32_t default_n_slabs();
uint32_t num_sms();  // SM count of the current device (148 on B200); 148 if no device is present

struct KernelArgs {
  // input
  const float *x, *y, *z;
  const uint8_t* module;
  const uint32_t* event_offsets;
  uint32_t n_events, n_modules;
  uint32_t n_hits;                   // host knowledge of the batch size: only steers launch heuristics
  uint32_t team_max_hits;            // events with more hits go to the general kernel
  float module_z[VELO_MAX_MODULES];  // geometry: the shared-memory path requires z[i] == module_z[module[i]]
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

// Which event kernel(s) a batch runs through (velo_launch_options_t.path).
enum { kPathDefault = 0,   // shared-memory team kernel, slab kernel for the events it defers
       kPathSlabOnly = 1 };  // slab kernel for every event (the general path on its own)

// Enqueues the whole path for one batch on `stream`. Returns a cudaError_t as int.
int launch_reconstruct(const KernelArgs& a, cudaStream_t stream, cudaEvent_t ev_start, cudaEvent_t ev_stop,
                       uint32_t path, uint32_t teams);

// velo_event_smem.cu: the shared-memory event kernel (persistent, one CTA per SM, `teams` teams of
// 128 threads). Events it cannot hold are appended to ws.large_list. Returns a cudaError_t as int.
int launch_event_smem(const KernelArgs& a, cudaStream_t stream, uint32_t teams);

}  // namespace velo
