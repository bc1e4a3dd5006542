/* velo.h — C-ABI of libvelo: B200-native (sm_100a) VELO pixel-detector track reconstruction.
 *
 * What the library computes. The data-parallel core of the GPU first-stage trigger (HLT1) of
 * arxiv/paper_2412_05041: reconstruction of "VELO tracks", the objects that the paper's forward
 * tracking and seeding-matching consume (§5), over batches of independent events
 * (30 MHz event stream, §3). The paper says only that HLT1 uses "a more simplified
 * pattern recognition algorithm" and "simplified track fitting" (§5); the steps
 * (per-module phi sort, search-by-triplet seeding, forwarding, ghost/clone filter, straight-line
 * least-squares fit to the state at closest approach to the beamline) are named by
 * BASELINE.json:north_star and made precise in SURVEY.md §8(c) items O-1 ... O-17, restated in
 * DESIGN.md §2. Coordinates: origin at the nominal interaction point, z along the beam, y up
 * (§2); lengths in mm.
 *
 * Conventions.
 *  - Every function returns VELO_OK (0) or a negative error code; nothing throws or aborts.
 *  - "DEVICE" pointers are CUDA device pointers of the current device; "HOST" pointers are plain
 *    host pointers. The caller owns every buffer it passes. The library allocates device memory
 *    only inside velo_scheduler_create.
 *  - velo_reconstruct is asynchronous on `stream`: no allocation, no host synchronisation, no
 *    use of the default stream. Its return value reports synchronous failures only (bad
 *    arguments, workspace too small, launch error). Data-dependent failures are written to
 *    out->summary[2] on the device (see velo_tracks_t).
 *  - Concurrent calls on different streams with different workspaces and outputs are allowed.
 *  - Inputs must be finite; NaN/Inf coordinates are undefined behaviour.
 *  - There is no CPU fallback: without a CUDA device every compute entry point returns
 *    VELO_ERR_CUDA.
 */
#ifndef VELO_H_
#define VELO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  VELO_OK = 0,
  VELO_ERR_ARG = -1,       /* null pointer, zero capacity, inconsistent sizes                   */
  VELO_ERR_GEOMETRY = -2,  /* n_modules outside 3..32, module_z not strictly increasing          */
  VELO_ERR_WORKSPACE = -3, /* workspace_bytes < velo_workspace_bytes(...)                        */
  VELO_ERR_CUDA = -4,      /* a CUDA runtime call or a kernel launch failed                      */
  VELO_ERR_CAPACITY = -5,  /* (device status) tracks or track-hits exceed the output capacities  */
  VELO_ERR_INPUT = -6,     /* (device status) module id >= n_modules, non-monotone offsets, or   */
                           /* an event with more than VELO_MAX_EVENT_HITS hits                   */
  VELO_ERR_STATIC_LIMIT = -7 /* sizes beyond the fixed maximum of a *_static entry point         */
};

#define VELO_MAX_MODULES 32
#define VELO_MAX_EVENT_HITS 65535u /* event-local hit indices are 16-bit inside the kernels     */
#define VELO_N_STATE 13            /* words per track state, see velo_tracks_t.states           */
#define VELO_N_SUMMARY 8           /* words of velo_tracks_t.summary                            */

/* ---- geometry (BASELINE.json:configs[0], configs[3]) ---------------- */
typedef struct velo_geometry velo_geometry_t; /* opaque, host-resident, immutable after load    */

typedef struct {           /* HOST POD, copied by velo_geometry_load                             */
  uint32_t n_modules;      /* 26 in the paper's detector; must be 3..VELO_MAX_MODULES            */
  const float* module_z;   /* HOST, n_modules, strictly increasing (mm)                          */
  float r_in, r_out;       /* active annulus 5.1 .. 42.0 mm (informational)                      */
  float pitch;             /* pixel pitch 0.055 mm; sets the default sigma_hit = pitch/sqrt(12)  */
  float half_shift_x;      /* 0 closed; 24.5 = the 2023 49 mm opening (§2)           */
  const float* module_z_b; /* HOST, n_modules, or NULL. The 52-sensor layout (DESIGN.md §2 L-1): */
                           /* a station's second sensor plane; module_z is then the first one's. */
                           /* Every plane of module m must lie below every plane of module m+1;  */
                           /* needs n_modules <= 30. A hit on either plane takes the pipeline;   */
                           /* any other z is legal and takes the general kernel (as with NULL).  */
} velo_geometry_desc_t;

/* Validates and copies the description. *out is set to a new handle (free it with
 * velo_geometry_free) or left untouched on error. Needs no CUDA device. */
int velo_geometry_load(const velo_geometry_desc_t* desc, velo_geometry_t** out);
void velo_geometry_free(velo_geometry_t* g);
uint32_t velo_geometry_n_modules(const velo_geometry_t* g);

/* ---- parameters (SURVEY.md §8(c) O-3, O-4, O-7, O-8, O-10 ... O-13; defaults A5 ... A13) ---- */
typedef struct {           /* HOST POD                                                           */
  int32_t phi_window_seed; /* O-8 window half-width, phi16 units (1 unit = pi/32768 rad); 300    */
  int32_t phi_window_fwd;  /* O-7 window half-width; 300                                         */
  float max_scatter_seed;  /* O-8 accept sc <= this (mm^2); 0.1                                  */
  float max_scatter_fwd;   /* O-7; 0.1                                                           */
  float max_scatter_weak;  /* O-10: 3-hit tracks need seed scatter <= this; 0.05                 */
  uint32_t max_skipped;    /* O-7: consecutive missed modules a track survives; 1                */
  float sigma_hit;         /* O-11: (float)(pitch/sqrt(12)) = 0x1.042186p-6 for 55 um pixels     */
  float max_chi2_ndof;     /* O-12; 100                                                          */
  uint32_t clone_num, clone_den; /* O-13: killed iff lost*den > n*num; 1, 3                      */
} velo_params_t;

/* Fills *p with the defaults above (sigma_hit from the geometry's pitch). */
void velo_params_default(const velo_geometry_t* g, velo_params_t* p);

/* ---- input: hits of a batch of events, structure of arrays ------ */
typedef struct {
  const float *x, *y, *z;        /* global-frame hit coordinates (mm). Indexed by ABSOLUTE hit    */
                                 /* index, i.e. the same index space as event_offsets.            */
  const uint8_t* module;         /* module id of each hit, 0 .. n_modules-1 (by increasing z)     */
  const uint32_t* event_offsets; /* n_events+1, non-decreasing. Event e owns hits                 */
                                 /* [event_offsets[e], event_offsets[e+1]). event_offsets[0] may  */
                                 /* be non-zero: a batch is a slice of a larger array.            */
  uint32_t n_events;
  uint32_t n_hits;               /* = event_offsets[n_events] - event_offsets[0] (host knowledge) */
} velo_hits_t;
/* Hit order inside an event is arbitrary; there is no alignment or padding requirement. An event
 * holds at most VELO_MAX_EVENT_HITS hits. Empty events and empty modules are legal (A15). */

/* ---- output: VELO tracks = hit lists + beamline states (§5; O-11, O-14) --------- */
typedef struct {
  uint32_t* event_track_offsets; /* n_events+1. Tracks of event e are                             */
                                 /* [event_track_offsets[e], event_track_offsets[e+1]).           */
  uint32_t* track_hit_offsets;   /* cap_tracks+1; [n_tracks] = n_track_hits                       */
  uint32_t* track_hits;          /* cap_track_hits; ABSOLUTE hit indices (same index space as     */
                                 /* hits.x), in discovery order = decreasing module               */
  float* states;                 /* VELO_N_STATE planes of cap_tracks words (plane stride =       */
                                 /* cap_tracks): x, y, tx, ty, z at the point of closest approach */
                                 /* to the z axis; cxx, cxtx, ctxtx, cyy, cyty, ctyty; chi2; and  */
                                 /* n_hits stored as the bit pattern of a uint32                  */
  uint32_t cap_tracks, cap_track_hits;
  uint32_t* summary;             /* u32[VELO_N_SUMMARY]: n_tracks, n_track_hits, status (VELO_OK  */
                                 /* or a negative code as two's complement), n_candidates (before */
                                 /* the filters), n_deferred (events the pipeline handed to the   */
                                 /* general slab kernel), n_big (events above 12 000 hits, run in  */
                                 /* the one-event-per-CTA pipeline), then two reserved zeros      */
} velo_tracks_t;
/* If the batch needs more than cap_tracks tracks or cap_track_hits track-hits, summary[2] =
 * VELO_ERR_CAPACITY, summary[0..1] hold the REQUIRED sizes and the other output arrays are
 * unspecified: results are never silently truncated. On VELO_ERR_INPUT the offending events
 * contribute zero tracks. cap_tracks = n_hits and cap_track_hits = n_modules * n_hits can never
 * overflow; cap_tracks = n_hits/4 + n_events and cap_track_hits = 2*n_hits is ample for the
 * BASELINE.json workloads. Tracks of an event are emitted in creation order: seeding step
 * (centre module) descending, then sorted position of the seed's centre hit. */

/* Bytes of DEVICE workspace velo_reconstruct needs for a batch of this shape. */
size_t velo_workspace_bytes(uint32_t n_events, uint32_t n_hits, uint32_t cap_tracks,
                            uint32_t cap_track_hits);

/* Reconstructs one batch. hits/out hold DEVICE pointers; geometry, params and the two structs
 * themselves are HOST memory read before the call returns. workspace: DEVICE, 256-byte aligned,
 * used until the work enqueued on `stream` completes. `stream` is a cudaStream_t passed as
 * void* so that this header needs no CUDA include. */
int velo_reconstruct(const velo_geometry_t* g, const velo_hits_t* hits, const velo_params_t* params,
                     velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream);

/* Same call with launch options, for measurement and tuning. opts may be NULL (= velo_reconstruct).
 * stage_events: cudaEvent_t handles (or NULL) recorded on `stream` at the stage boundaries of the
 * batch, so that a benchmark can time every stage on the stream it runs on: [0] before stage 1,
 * [1] after stage 1 (sort: S0, S1), [2] after stage 2 (module loop: S2, S3, and the general kernel
 * for deferred events), [3] after stage 3 (fit and filters: S4, S5, S6), [4] after the offsets scan,
 * [5] after the write kernel (S7).
 * path: VELO_PATH_DEFAULT = the three-stage pipeline, with the general slab kernel for the events it
 * defers (hits off their module plane, events too large for one SM's shared memory);
 * VELO_PATH_SLAB_ONLY = the general slab kernel for every event. Both give identical results.
 * ctas_per_sm: persistent CTAs per SM of the slab kernel, 0 = library default; the workspace must
 * have been sized for the default or for velo_workspace_bytes_opts with the same value. */
enum { VELO_PATH_DEFAULT = 0, VELO_PATH_SLAB_ONLY = 1 };
#define VELO_N_STAGE_EVENTS 6
typedef struct {
  void* stage_events[VELO_N_STAGE_EVENTS];
  uint32_t ctas_per_sm;
  uint32_t path;
  uint32_t track_group;   /* threads per event in the module-loop kernel: 32, 64 or 128; 0 = default  */
  uint32_t track_teams;   /* events in flight per persistent CTA of the module-loop kernel; 0 = default */
  uint32_t fit_teams;     /* ... of the fit/output kernel; 0 = default                                  */
  uint32_t sort_teams;    /* ... of the sort kernel; 0 = default                                        */
  uint32_t pool_units;    /* shared-memory pool per CTA in units of 1728 bytes, 1..128; 0 = 128         */
} velo_launch_options_t;
size_t velo_workspace_bytes_opts(uint32_t n_events, uint32_t n_hits, uint32_t cap_tracks,
                                 uint32_t cap_track_hits, const velo_launch_options_t* opts);
int velo_reconstruct_opts(const velo_geometry_t* g, const velo_hits_t* hits, const velo_params_t* params,
                          velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream,
                          const velo_launch_options_t* opts);

/* ---- event-batch scheduler on streams (§3) ------------------ */
/* Owns n_streams CUDA streams, each with device input, output and workspace buffers for batches
 * of up to max_batch_events events / max_batch_hits hits, and pinned staging for the summaries. */
typedef struct velo_scheduler velo_scheduler_t;
int velo_scheduler_create(const velo_geometry_t* g, uint32_t n_streams, uint32_t max_batch_events,
                          uint32_t max_batch_hits, velo_scheduler_t** out);
void velo_scheduler_free(velo_scheduler_t* s);

/* End-to-end path over HOST buffers. hits holds HOST pointers (pinned memory makes the copies
 * asynchronous). Events are cut into n_batches contiguous batches at batch_begin[0..n_batches]
 * (event indices, batch_begin[0] = 0, batch_begin[n_batches] = hits->n_events); batch b runs on
 * stream b % n_streams: host->device copy of its slice, velo_reconstruct, device->host copy of
 * exactly the produced tracks into out[b] (HOST pointers, capacities per batch; summary is a
 * HOST u32[VELO_N_SUMMARY]). Offsets in out[b] are batch-local; track_hits are absolute hit indices.
 * Returns after every copy has completed. A batch larger than the scheduler's limits or an
 * output capacity below cap_tracks = n_hits/4 + n_events, cap_track_hits = 2*n_hits of the
 * device buffers is reported per batch through out[b].summary[2]. */
int velo_scheduler_run_host(velo_scheduler_t* s, const velo_params_t* params, const velo_hits_t* hits,
                            const uint32_t* batch_begin, uint32_t n_batches, velo_tracks_t* out);

/* ---- in front of the hot path: SURVEY.md §8(f) f1, packed pixel hits decoded inside S0 -------- */
/* The VELO is a pixel detector read out as raw data (PAPER.md:24 §2, :42 §3); the paper gives no
 * format, so this one is the repository's (DESIGN.md §2 F-1, F-2). One u32 per hit:
 *   bits 0-10 column + 1024, bits 11-21 row + 1024, bit 22 half (1 = the +x half), bits 23-27 module;
 * column and row count pixels of `pitch` from the half's local origin. Decode, in double precision
 * with one final rounding: x = fl32((column + 0.5) * pitch + h * half_shift_x), h = +1 / -1 for the
 * half bit; y = fl32((row + 0.5) * pitch); z = module_z[module]. 4 bytes per hit instead of 13. */
typedef struct {                 /* DEVICE pointers for velo_reconstruct_pixels, HOST for the scheduler call */
  const uint32_t* pixel;         /* n_hits packed addresses, indexed by absolute hit index */
  const uint32_t* event_offsets; /* n_events+1, as in velo_hits_t */
  uint32_t n_events, n_hits;
} velo_pixel_hits_t;
typedef struct { double pitch, half_shift_x; } velo_pixel_format_t;   /* 0.055 mm; 0 closed, 24.5 open */
/* velo_reconstruct with the decode fused into stage 1 (S0): same outputs, same workspace size, same
 * error behaviour (a module id >= n_modules -> VELO_ERR_INPUT). The fp32 coordinates exist only
 * inside the kernels; events that the pipeline defers to the general kernel are decoded into the
 * workspace first. opts may be NULL. */
int velo_reconstruct_pixels(const velo_geometry_t* g, const velo_pixel_hits_t* hits, const velo_pixel_format_t* fmt,
                            const velo_params_t* params, velo_tracks_t* out, void* workspace, size_t workspace_bytes,
                            void* stream, const velo_launch_options_t* opts);
/* velo_scheduler_run_host over packed HOST input: 4 bytes per hit cross the bus instead of 13. */
int velo_scheduler_run_host_pixels(velo_scheduler_t* s, const velo_params_t* params, const velo_pixel_hits_t* hits,
                                   const velo_pixel_format_t* fmt, const uint32_t* batch_begin, uint32_t n_batches,
                                   velo_tracks_t* out);

/* ---- after the hot path: SURVEY.md §8(f) f2 and f3 ------------------------------------------- */
/* f2. Parameterised Kalman filter on the VELO segment of every track (§5: "the Kalman
 * filtering process on track uses a parameterised approach ... only the segment of a track inside
 * the VELO is considered for the filtering process"; the paper gives no formula: readings K-1 ... K-5
 * of DESIGN.md §2). x(z) and y(z) are independent lines; every hit measures both with variance
 * sigma_hit^2; at every measured plane the slopes pick up noise ms_theta2 * (1 + tx^2 + ty^2); the
 * filter starts from the exact two-point state of the two most downstream hits, runs towards the
 * beamline and reports the state at closest approach to the z axis in the 13-word layout of
 * velo_tracks_t.states (chi2 = sum of squared innovations over their variances, ndof = 2 n - 4).
 * hits: the DEVICE planes velo_reconstruct was given (absolute hit index 0 at x[0]); tracks: its
 * DEVICE outputs (track_hit_offsets, track_hits, summary, cap_tracks are read); kalman_states: DEVICE,
 * 13 planes of tracks->cap_tracks words, written for the tracks the batch produced (none if the
 * batch reported an error). Asynchronous on `stream`; returns VELO_ERR_ARG / VELO_ERR_CUDA. */
int velo_kalman_fit(const velo_hits_t* hits, const velo_tracks_t* tracks, float sigma_hit, float ms_theta2,
                    float* kalman_states, void* stream);
/* The same on the packed pixel addresses that velo_reconstruct_pixels was given (decoded per hit as F-2). */
int velo_kalman_fit_pixels(const velo_geometry_t* g, const velo_pixel_hits_t* hits, const velo_pixel_format_t* fmt,
                           const velo_tracks_t* tracks, float sigma_hit, float ms_theta2, float* kalman_states,
                           void* stream);

/* f3. Primary vertices from the beamline states (§5: VELO tracks are straight
 * lines; displaced-vertex lines need primary vertices; the paper gives no algorithm: readings
 * P-1 ... P-6 of DESIGN.md §2). Per event: histogram of the tracks' z at the beamline; seeds = local
 * maxima of the (1, 2, 1)-smoothed counts; every track goes to the seed nearest in z; each seed is
 * fitted as the weighted least-squares point of its tracks' lines, weights 1/cxx times a Tukey
 * factor (1 - chi2/chi2_max)^2, n_iterations times from (0, 0, z_seed); kept with >= min_tracks
 * tracks of non-zero weight. Sums over tracks run as 32 partial sums by track index mod 32,
 * combined by a butterfly (the order is part of the definition: the oracle does the same). */
#define VELO_PV_MAX_PER_EVENT 32u
#define VELO_PV_MAX_BINS 4096u
#define VELO_N_PV_WORDS 5          /* planes of velo_pvs_t.pvs: x, y, z, sum of weights, n_tracks (u32 bits) */
typedef struct {
  float z_min, bin_width;          /* -300 mm, 0.25 mm */
  uint32_t n_bins;                 /* 2400; at most VELO_PV_MAX_BINS */
  uint32_t seed_min_sum;           /* 5 */
  uint32_t seed_half_window;       /* 6 bins */
  float chi2_max;                  /* 16 */
  uint32_t n_iterations;           /* 4 */
  uint32_t min_tracks;             /* 4 */
  uint32_t max_pv_per_event;       /* 32 = VELO_PV_MAX_PER_EVENT (larger values are clamped); lowest z first */
} velo_pv_params_t;
void velo_pv_params_default(velo_pv_params_t* p);
typedef struct {                   /* caller-allocated DEVICE buffers */
  uint32_t* event_pv_offsets;      /* n_events+1: vertices of event e are [off[e], off[e+1]), ascending seed z */
  float* pvs;                      /* VELO_N_PV_WORDS planes x cap_pvs */
  uint32_t cap_pvs;                /* 32 * n_events can never overflow */
  uint32_t* summary;               /* u32[4]: n_pvs (or the required capacity), status, 0, 0 */
} velo_pvs_t;
size_t velo_pv_workspace_bytes(uint32_t n_events, uint32_t cap_tracks);
/* tracks: DEVICE outputs of velo_reconstruct (event_track_offsets, states, summary, cap_tracks are
 * read); workspace: DEVICE, 256-byte aligned, velo_pv_workspace_bytes(n_events, tracks->cap_tracks).
 * Asynchronous on `stream`. More vertices than cap_pvs -> out->summary[1] = VELO_ERR_CAPACITY and
 * summary[0] = the required capacity; a failed velo_reconstruct status is passed on. */
int velo_pv_find(const velo_tracks_t* tracks, uint32_t n_events, const velo_pv_params_t* params, velo_pvs_t* out,
                 void* workspace, size_t workspace_bytes, void* stream);

/* The same operation for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the workspace is a fixed array inside the
 * library (a file-scope `static __device__` array of 4 736 256 bytes, which every GPU that loads the
 * library holds until the process exits), so the call takes no workspace and performs no cudaMalloc,
 * cudaFree or allocating library call. Inputs, outputs, results and error behaviour are those of
 * velo_pv_find, with two fixed limits: n_events <= VELO_PV_STATIC_MAX_EVENTS and tracks->cap_tracks <=
 * VELO_PV_STATIC_MAX_TRACKS; larger sizes return VELO_ERR_STATIC_LIMIT and enqueue nothing.
 * The array is shared by every call on the device and keeps the last call's contents; the kernels
 * write every word of it before they read it, so nothing needs clearing between calls. Calls that
 * overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it: serialise them
 * (one stream, or events), or use velo_pv_find with one workspace per stream. The array's device
 * address is looked up once per device (cudaGetSymbolAddress, with that device current). */
#define VELO_PV_STATIC_MAX_EVENTS 4096u
#define VELO_PV_STATIC_MAX_TRACKS 2097152u
int velo_pv_find_static(const velo_tracks_t* tracks, uint32_t n_events, const velo_pv_params_t* params, velo_pvs_t* out,
                        void* stream);

/* Library version string, e.g. "velo-b200 0.1 (sm_100a)". */
const char* velo_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VELO_H_ */
