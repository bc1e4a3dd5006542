// velo_scheduler.cu — event-batch scheduler on CUDA streams (the 30 MHz event
// stream of PAPER.md:42 §3 arrives as batches). End-to-end path over host buffers: per batch,
// host->device copy of the slice, velo_reconstruct, device->host copy of exactly the produced
// tracks. Batches on different streams overlap copies with kernels.
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "velo_internal.h"

namespace {

struct Lane {                 // one stream with its device buffers
  cudaStream_t stream = nullptr;
  float *x = nullptr, *y = nullptr, *z = nullptr;
  uint8_t* module = nullptr;
  uint32_t* pixel = nullptr;  // packed input (velo_scheduler_run_host_pixels), allocated on first use
  uint32_t* offsets = nullptr;
  velo_tracks_t out{};        // device output buffers
  void* workspace = nullptr;
  size_t workspace_bytes = 0;
  uint32_t* summary_host = nullptr;  // pinned u32[VELO_N_SUMMARY]
  // batch in flight
  bool busy = false;
  uint32_t batch = 0;
};

}  // namespace

struct velo_scheduler {
  const velo_geometry_t* g = nullptr;
  uint32_t max_events = 0, max_hits = 0, cap_tracks = 0, cap_track_hits = 0;
  std::vector<Lane> lanes;
};

namespace {

bool ok(cudaError_t e) { return e == cudaSuccess; }

void free_lane(Lane& l) {
  if (l.stream) cudaStreamDestroy(l.stream);
  cudaFree(l.x); cudaFree(l.y); cudaFree(l.z); cudaFree(l.module); cudaFree(l.pixel); cudaFree(l.offsets);
  cudaFree(l.out.event_track_offsets); cudaFree(l.out.track_hit_offsets); cudaFree(l.out.track_hits);
  cudaFree(l.out.states); cudaFree(l.out.summary); cudaFree(l.workspace);
  if (l.summary_host) cudaFreeHost(l.summary_host);
  l = Lane();
}

// Waits for the lane's batch, then copies exactly the produced tracks to the caller's host buffers.
int finish_lane(Lane& l, velo_tracks_t* outs) {
  if (!l.busy) return VELO_OK;
  l.busy = false;
  velo_tracks_t& o = outs[l.batch];
  if (!ok(cudaStreamSynchronize(l.stream))) return VELO_ERR_CUDA;
  const uint32_t nt = l.summary_host[0], nh = l.summary_host[1];
  int status = (int)l.summary_host[2];
  if (status == VELO_OK && (nt > o.cap_tracks || nh > o.cap_track_hits)) status = VELO_ERR_CAPACITY;
  for (int k = 0; k < VELO_N_SUMMARY; ++k) o.summary[k] = l.summary_host[k];
  o.summary[2] = (uint32_t)status;
  if (status == VELO_ERR_CAPACITY) return VELO_OK;  // reported per batch; nothing valid to copy
  bool good = true;
  if (nt) {
    good &= ok(cudaMemcpyAsync(o.track_hit_offsets, l.out.track_hit_offsets, 4 * ((size_t)nt + 1),
                               cudaMemcpyDeviceToHost, l.stream));
    for (int p = 0; p < VELO_N_STATE; ++p)
      good &= ok(cudaMemcpyAsync(o.states + (size_t)p * o.cap_tracks, l.out.states + (size_t)p * l.out.cap_tracks,
                                 4 * (size_t)nt, cudaMemcpyDeviceToHost, l.stream));
  } else {
    o.track_hit_offsets[0] = 0;
  }
  if (nh) good &= ok(cudaMemcpyAsync(o.track_hits, l.out.track_hits, 4 * (size_t)nh, cudaMemcpyDeviceToHost, l.stream));
  good &= ok(cudaStreamSynchronize(l.stream));
  return good ? VELO_OK : VELO_ERR_CUDA;
}

}  // namespace

extern "C" {

void velo_scheduler_free(velo_scheduler_t* s) {
  if (!s) return;
  for (Lane& l : s->lanes) free_lane(l);
  delete s;
}

int velo_scheduler_create(const velo_geometry_t* g, uint32_t n_streams, uint32_t max_batch_events,
                          uint32_t max_batch_hits, velo_scheduler_t** out) {
  if (!g || !out || n_streams == 0 || n_streams > 64 || max_batch_events == 0) return VELO_ERR_ARG;
  velo_scheduler* s = new (std::nothrow) velo_scheduler();
  if (!s) return VELO_ERR_ARG;
  s->g = g; s->max_events = max_batch_events; s->max_hits = max_batch_hits;
  const uint64_t ct = (uint64_t)max_batch_hits / 4 + max_batch_events, ch = 2ull * max_batch_hits + 1;
  s->cap_tracks = (uint32_t)(ct > 0xffffffffull ? 0xffffffffull : ct);
  s->cap_track_hits = (uint32_t)(ch > 0xffffffffull ? 0xffffffffull : ch);
  s->lanes.resize(n_streams);
  bool good = true;
  const size_t H = (size_t)max_batch_hits + 1;
  for (Lane& l : s->lanes) {
    good &= ok(cudaStreamCreateWithFlags(&l.stream, cudaStreamNonBlocking));
    good &= ok(cudaMalloc(&l.x, 4 * H)) && ok(cudaMalloc(&l.y, 4 * H)) && ok(cudaMalloc(&l.z, 4 * H));
    good &= ok(cudaMalloc(&l.module, H)) && ok(cudaMalloc(&l.offsets, 4 * ((size_t)max_batch_events + 1)));
    l.out.cap_tracks = s->cap_tracks; l.out.cap_track_hits = s->cap_track_hits;
    good &= ok(cudaMalloc(&l.out.event_track_offsets, 4 * ((size_t)max_batch_events + 1)));
    good &= ok(cudaMalloc(&l.out.track_hit_offsets, 4 * ((size_t)s->cap_tracks + 1)));
    good &= ok(cudaMalloc(&l.out.track_hits, 4 * (size_t)s->cap_track_hits));
    good &= ok(cudaMalloc(&l.out.states, 4 * (size_t)VELO_N_STATE * s->cap_tracks));
    good &= ok(cudaMalloc(&l.out.summary, 4 * VELO_N_SUMMARY));
    l.workspace_bytes = velo_workspace_bytes(max_batch_events, max_batch_hits, s->cap_tracks, s->cap_track_hits);
    good &= ok(cudaMalloc(&l.workspace, l.workspace_bytes));
    good &= ok(cudaMallocHost(&l.summary_host, 4 * VELO_N_SUMMARY));
    if (!good) break;
  }
  if (!good) { cudaGetLastError(); velo_scheduler_free(s); return VELO_ERR_CUDA; }
  *out = s;
  return VELO_OK;
}

}  // extern "C"

namespace {

// One pass over the batches: `upload(lane, h0, nh)` copies the batch's hits, `launch(lane, ne, nh, h0)`
// enqueues its reconstruction.
template <class Upload, class Launch>
int run_batches(velo_scheduler_t* s, const uint32_t* event_offsets, uint32_t n_events, const uint32_t* batch_begin,
                uint32_t n_batches, velo_tracks_t* out, Upload&& upload, Launch&& launch) {
  if (batch_begin[0] != 0 || batch_begin[n_batches] != n_events) return VELO_ERR_ARG;
  int rc = VELO_OK;
  for (uint32_t b = 0; b < n_batches && rc == VELO_OK; ++b) {
    Lane& l = s->lanes[b % s->lanes.size()];
    rc = finish_lane(l, out);
    if (rc != VELO_OK) break;
    const uint32_t e0 = batch_begin[b], e1 = batch_begin[b + 1];
    velo_tracks_t& o = out[b];
    if (e1 < e0 || !o.summary || !o.event_track_offsets || !o.track_hit_offsets || !o.track_hits || !o.states) {
      rc = VELO_ERR_ARG; break;
    }
    const uint32_t ne = e1 - e0;
    const uint32_t h0 = event_offsets[e0], h1 = event_offsets[e1];
    if (h1 < h0 || ne > s->max_events || h1 - h0 > s->max_hits) {
      for (int k = 0; k < VELO_N_SUMMARY; ++k) o.summary[k] = 0;
      o.summary[2] = (uint32_t)VELO_ERR_CAPACITY;
      continue;
    }
    const uint32_t nh = h1 - h0;
    bool good = upload(l, h0, nh);
    good &= ok(cudaMemcpyAsync(l.offsets, event_offsets + e0, 4 * ((size_t)ne + 1), cudaMemcpyHostToDevice, l.stream));
    if (!good) { rc = VELO_ERR_CUDA; break; }
    // the device copy holds hits [h0, h1) at index 0; the batch keeps its absolute offsets, so the
    // emitted track_hits stay absolute hit indices
    rc = launch(l, ne, nh, h0);
    if (rc != VELO_OK) break;
    good &= ok(cudaMemcpyAsync(l.summary_host, l.out.summary, 4 * VELO_N_SUMMARY, cudaMemcpyDeviceToHost, l.stream));
    good &= ok(cudaMemcpyAsync(o.event_track_offsets, l.out.event_track_offsets, 4 * ((size_t)ne + 1),
                               cudaMemcpyDeviceToHost, l.stream));
    if (!good) { rc = VELO_ERR_CUDA; break; }
    l.busy = true; l.batch = b;
  }
  for (Lane& l : s->lanes) {
    const int r = finish_lane(l, out);
    if (rc == VELO_OK) rc = r;
  }
  return rc;
}

}  // namespace

extern "C" {

int velo_scheduler_run_host(velo_scheduler_t* s, const velo_params_t* params, const velo_hits_t* hits,
                            const uint32_t* batch_begin, uint32_t n_batches, velo_tracks_t* out) {
  if (!s || !params || !hits || !batch_begin || !out || !hits->event_offsets) return VELO_ERR_ARG;
  return run_batches(
      s, hits->event_offsets, hits->n_events, batch_begin, n_batches, out,
      [&](Lane& l, uint32_t h0, uint32_t nh) {
        bool good = true;
        if (nh) {
          good &= ok(cudaMemcpyAsync(l.x, hits->x + h0, 4 * (size_t)nh, cudaMemcpyHostToDevice, l.stream));
          good &= ok(cudaMemcpyAsync(l.y, hits->y + h0, 4 * (size_t)nh, cudaMemcpyHostToDevice, l.stream));
          good &= ok(cudaMemcpyAsync(l.z, hits->z + h0, 4 * (size_t)nh, cudaMemcpyHostToDevice, l.stream));
          good &= ok(cudaMemcpyAsync(l.module, hits->module + h0, (size_t)nh, cudaMemcpyHostToDevice, l.stream));
        }
        return good;
      },
      [&](Lane& l, uint32_t ne, uint32_t nh, uint32_t h0) {
        velo_hits_t dh{};
        dh.x = l.x; dh.y = l.y; dh.z = l.z; dh.module = l.module;
        dh.event_offsets = l.offsets; dh.n_events = ne; dh.n_hits = nh;
        return velo::reconstruct_impl(s->g, &dh, params, &l.out, l.workspace, l.workspace_bytes, (void*)l.stream, nullptr, h0);
      });
}

int velo_scheduler_run_host_pixels(velo_scheduler_t* s, const velo_params_t* params, const velo_pixel_hits_t* hits,
                                   const velo_pixel_format_t* fmt, const uint32_t* batch_begin, uint32_t n_batches,
                                   velo_tracks_t* out) {
  if (!s || !params || !hits || !fmt || !batch_begin || !out || !hits->event_offsets) return VELO_ERR_ARG;
  if (hits->n_hits && !hits->pixel) return VELO_ERR_ARG;
  for (Lane& l : s->lanes)
    if (!l.pixel && !ok(cudaMalloc(&l.pixel, 4 * ((size_t)s->max_hits + 4)))) { cudaGetLastError(); return VELO_ERR_CUDA; }
  return run_batches(
      s, hits->event_offsets, hits->n_events, batch_begin, n_batches, out,
      [&](Lane& l, uint32_t h0, uint32_t nh) {
        return nh == 0 || ok(cudaMemcpyAsync(l.pixel, hits->pixel + h0, 4 * (size_t)nh, cudaMemcpyHostToDevice, l.stream));
      },
      [&](Lane& l, uint32_t ne, uint32_t nh, uint32_t h0) {
        velo_pixel_hits_t dh{};
        dh.pixel = l.pixel; dh.event_offsets = l.offsets; dh.n_events = ne; dh.n_hits = nh;
        return velo::reconstruct_pixels_impl(s->g, &dh, fmt, params, &l.out, l.workspace, l.workspace_bytes,
                                             (void*)l.stream, nullptr, h0);
      });
}

}  // extern "C"
