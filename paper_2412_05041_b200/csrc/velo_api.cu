// velo_api.cu — the C-ABI of libvelo (include/velo.h): argument checks, workspace carving, kernel
// launches and the event-batch scheduler on streams. No reconstruction arithmetic lives here.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "velo_internal.h"

extern "C" {

const char* velo_version(void) { return "velo-b200 0.1 (sm_100a)"; }

int velo_geometry_load(const velo_geometry_desc_t* desc, velo_geometry_t** out) {
  if (!desc || !out || !desc->module_z) return VELO_ERR_ARG;
  if (desc->n_modules < 3 || desc->n_modules > VELO_MAX_MODULES) return VELO_ERR_GEOMETRY;
  for (uint32_t m = 0; m < desc->n_modules; ++m) {
    if (!isfinite(desc->module_z[m])) return VELO_ERR_GEOMETRY;
    if (m && !(desc->module_z[m] > desc->module_z[m - 1])) return VELO_ERR_GEOMETRY;
  }
  if (!(desc->pitch > 0.0f) || !isfinite(desc->pitch)) return VELO_ERR_GEOMETRY;
  if (desc->module_z_b) {
    if (desc->n_modules > velo::kTwoPlaneMaxModules) return VELO_ERR_GEOMETRY;
    for (uint32_t m = 0; m < desc->n_modules; ++m) {
      const float a = desc->module_z[m], b = desc->module_z_b[m];
      if (!isfinite(b)) return VELO_ERR_GEOMETRY;
      if (m) {
        const float pa = desc->module_z[m - 1], pb = desc->module_z_b[m - 1];
        if (!((a < b ? a : b) > (pa > pb ? pa : pb))) return VELO_ERR_GEOMETRY;
      }
    }
  }
  velo_geometry* g = new (std::nothrow) velo_geometry();
  if (!g) return VELO_ERR_ARG;
  g->n_modules = desc->n_modules;
  memcpy(g->module_z, desc->module_z, sizeof(float) * desc->n_modules);
  g->two_plane = desc->module_z_b ? 1u : 0u;
  if (desc->module_z_b) memcpy(g->module_z_b, desc->module_z_b, sizeof(float) * desc->n_modules);
  g->r_in = desc->r_in; g->r_out = desc->r_out; g->pitch = desc->pitch; g->half_shift_x = desc->half_shift_x;
  *out = g;
  return VELO_OK;
}

void velo_geometry_free(velo_geometry_t* g) { delete g; }

uint32_t velo_geometry_n_modules(const velo_geometry_t* g) { return g ? g->n_modules : 0; }

void velo_params_default(const velo_geometry_t* g, velo_params_t* p) {
  if (!p) return;
  const double pitch = g ? (double)g->pitch : 0.055;
  p->phi_window_seed = 300; p->phi_window_fwd = 300;
  p->max_scatter_seed = 0.1f; p->max_scatter_fwd = 0.1f; p->max_scatter_weak = 0.05f;
  p->max_skipped = 1;
  p->sigma_hit = (float)(pitch / sqrt(12.0));
  p->max_chi2_ndof = 100.0f;
  p->clone_num = 1; p->clone_den = 3;
}

static uint32_t n_slabs_for(const velo_launch_options_t* opts) {
  const uint32_t per_sm = (opts && opts->ctas_per_sm) ? opts->ctas_per_sm : 0;
  return per_sm ? velo::num_sms() * (per_sm > 16 ? 16 : per_sm) : velo::default_n_slabs();
}

size_t velo_workspace_bytes_opts(uint32_t n_events, uint32_t n_hits, uint32_t cap_tracks, uint32_t cap_track_hits,
                                 const velo_launch_options_t* opts) {
  return velo::carve_workspace(nullptr, n_events, n_hits, cap_tracks, cap_track_hits, n_slabs_for(opts)).bytes;
}

size_t velo_workspace_bytes(uint32_t n_events, uint32_t n_hits, uint32_t cap_tracks, uint32_t cap_track_hits) {
  return velo_workspace_bytes_opts(n_events, n_hits, cap_tracks, cap_track_hits, nullptr);
}

}  // extern "C"

namespace velo {

namespace {

// Argument checks and kernel arguments shared by the fp32 and the packed-pixel entry points.
int run_batch(const velo_geometry_t* g, KernelArgs& a, uint32_t n_events, uint32_t n_hits, const velo_params_t* params,
              velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream, const velo_launch_options_t* opts) {
  if (!out->event_track_offsets || !out->track_hit_offsets || !out->summary) return VELO_ERR_ARG;
  if (!out->track_hits || !out->states || out->cap_tracks == 0 || out->cap_track_hits == 0) return VELO_ERR_ARG;
  if (((uintptr_t)workspace & 255u) != 0) return VELO_ERR_ARG;
  if (params->clone_den == 0) return VELO_ERR_ARG;
  const size_t need = velo_workspace_bytes_opts(n_events, n_hits, out->cap_tracks, out->cap_track_hits, opts);
  if (workspace_bytes < need) return VELO_ERR_WORKSPACE;
  a.n_events = n_events; a.n_modules = g->n_modules; a.n_hits = n_hits;
  uint32_t path = opts ? opts->path : 0u;
  a.team_max_hits = kPipeMaxHits;
  for (uint32_t m = 0; m < VELO_MAX_MODULES; ++m) a.module_z[m] = m < g->n_modules ? g->module_z[m] : 0.0f;
  a.two_plane = g->two_plane;
  for (uint32_t m = 0; m < VELO_MAX_MODULES; ++m) a.module_z_b[m] = (g->two_plane && m < g->n_modules) ? g->module_z_b[m] : 0.0f;
  a.P = *params;
  if (a.P.max_skipped > 200u) a.P.max_skipped = 200u;  // more misses than modules is all the same
  // A negative window holds no hit (O-3). The kernels take windows >= 0; the same result follows
  // from a scatter cut that nothing passes (scatter is a sum of squares, never below zero).
  if (a.P.phi_window_seed < 0) { a.P.phi_window_seed = 0; a.P.max_scatter_seed = -1.0f; }
  if (a.P.phi_window_fwd < 0) { a.P.phi_window_fwd = 0; a.P.max_scatter_fwd = -1.0f; }
  // The module loop of the pipeline keeps "scatter <= cut" as "scatter < the next float above the cut", which
  // needs a cut below +inf: any other cut (+inf, NaN) takes the general kernel and its plain comparison.
  if (!(a.P.max_scatter_seed < INFINITY) || !(a.P.max_scatter_fwd < INFINITY)) path = kPathSlabOnly;
  a.event_track_offsets = out->event_track_offsets; a.track_hit_offsets = out->track_hit_offsets;
  a.track_hits = out->track_hits; a.states = out->states;
  a.cap_tracks = out->cap_tracks; a.cap_track_hits = out->cap_track_hits; a.summary = out->summary;
  a.ws = carve_workspace(workspace, n_events, n_hits, out->cap_tracks, out->cap_track_hits, n_slabs_for(opts));
  PipeOpts po{};
  if (opts) { po.track_group = opts->track_group; po.track_teams = opts->track_teams; po.fit_teams = opts->fit_teams;
              po.sort_teams = opts->sort_teams; po.pool_units = opts->pool_units; }
  const int err = launch_reconstruct(a, (cudaStream_t)stream, opts ? opts->stage_events : nullptr, path, po);
  return err == 0 ? VELO_OK : VELO_ERR_CUDA;
}

}  // namespace

int reconstruct_impl(const velo_geometry_t* g, const velo_hits_t* hits, const velo_params_t* params,
                     velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream,
                     const velo_launch_options_t* opts, uint32_t hit_base) {
  if (!g || !hits || !params || !out || !workspace || !hits->event_offsets) return VELO_ERR_ARG;
  if (hits->n_hits && (!hits->x || !hits->y || !hits->z || !hits->module)) return VELO_ERR_ARG;
  KernelArgs a{};
  a.x = hits->x; a.y = hits->y; a.z = hits->z; a.module = hits->module;
  a.event_offsets = hits->event_offsets; a.hit_base = hit_base;
  return run_batch(g, a, hits->n_events, hits->n_hits, params, out, workspace, workspace_bytes, stream, opts);
}

int reconstruct_pixels_impl(const velo_geometry_t* g, const velo_pixel_hits_t* hits, const velo_pixel_format_t* fmt,
                            const velo_params_t* params, velo_tracks_t* out, void* workspace, size_t workspace_bytes,
                            void* stream, const velo_launch_options_t* opts, uint32_t hit_base) {
  if (!g || !hits || !fmt || !params || !out || !workspace || !hits->event_offsets) return VELO_ERR_ARG;
  if (!hits->pixel) return VELO_ERR_ARG;          // also for an empty batch: it marks the packed path
  if (!(fmt->pitch > 0.0)) return VELO_ERR_ARG;
  KernelArgs a{};
  a.pixel = hits->pixel; a.pitch = fmt->pitch; a.half_shift_x = fmt->half_shift_x;
  a.event_offsets = hits->event_offsets; a.hit_base = hit_base;
  return run_batch(g, a, hits->n_events, hits->n_hits, params, out, workspace, workspace_bytes, stream, opts);
}

}  // namespace velo

extern "C" {

int velo_reconstruct_opts(const velo_geometry_t* g, const velo_hits_t* hits, const velo_params_t* params,
                          velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream,
                          const velo_launch_options_t* opts) {
  return velo::reconstruct_impl(g, hits, params, out, workspace, workspace_bytes, stream, opts, 0u);
}

int velo_reconstruct(const velo_geometry_t* g, const velo_hits_t* hits, const velo_params_t* params,
                     velo_tracks_t* out, void* workspace, size_t workspace_bytes, void* stream) {
  return velo_reconstruct_opts(g, hits, params, out, workspace, workspace_bytes, stream, nullptr);
}

int velo_reconstruct_pixels(const velo_geometry_t* g, const velo_pixel_hits_t* hits, const velo_pixel_format_t* fmt,
                            const velo_params_t* params, velo_tracks_t* out, void* workspace, size_t workspace_bytes,
                            void* stream, const velo_launch_options_t* opts) {
  return velo::reconstruct_pixels_impl(g, hits, fmt, params, out, workspace, workspace_bytes, stream, opts, 0u);
}

}  // extern "C"
