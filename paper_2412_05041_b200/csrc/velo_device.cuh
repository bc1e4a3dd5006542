// velo_device.cuh — device-side primitives of libvelo (sm_100a). Internal header of the CUDA
// path; shares nothing with oracle/.
//
// Every floating-point operation that feeds a predicate, a quantised code or the fitted state is
// written with the round-to-nearest intrinsics (__fadd_rn, __fsub_rn, __fmul_rn, __fdiv_rn), which
// nvcc never contracts into FMA: the reading in SURVEY.md §8(c) ("one rounding per written
// operator, no fused multiply-add", O-1, O-4, O-11) is part of the method's definition, because
// phi16 decides the sort, scatter decides the candidate choice and chi2 enters the clone key.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/velo.h"

namespace velo {

// ---- O-1 phi16(x, y): quantised azimuth about the nominal beam axis, int16 in 65536 bins ------
// Degree-5 polynomial in t^2 for atan(t)/t on [0,1], octant folding, floor.
__device__ __forceinline__ int phi16(float x, float y) {
  const float C0 = 0x1.fffd04p-1f, C1 = -0x1.549b14p-2f, C2 = 0x1.8c5ee6p-3f;
  const float C3 = -0x1.dce202p-4f, C4 = 0x1.af4978p-5f, C5 = -0x1.80032cp-7f;
  const float K = 0x1.45f306p+13f;  // 32768/pi
  const float ax = fabsf(x), ay = fabsf(y);
  const bool xbig = ax > ay;
  const float mx = xbig ? ax : ay;
  const float mn = xbig ? ay : ax;
  if (mx == 0.0f) return 0;
  const float t = __fdiv_rn(mn, mx);
  const float s = __fmul_rn(t, t);
  float p = C5;
  p = __fadd_rn(__fmul_rn(p, s), C4);
  p = __fadd_rn(__fmul_rn(p, s), C3);
  p = __fadd_rn(__fmul_rn(p, s), C2);
  p = __fadd_rn(__fmul_rn(p, s), C1);
  p = __fadd_rn(__fmul_rn(p, s), C0);
  float a = __fmul_rn(__fmul_rn(t, p), K);
  if (ay > ax) a = __fsub_rn(16384.0f, a);
  if (x < 0.0f) a = __fsub_rn(32768.0f, a);
  if (y < 0.0f) a = -a;
  const int k = (int)floorf(a);
  return ((k + 32768) & 65535) - 32768;
}

// ---- F-1, F-2 packed pixel address -> module, x, y (include/velo.h velo_pixel_hits_t) ----
// Double precision with one final rounding, as the format defines it.
__device__ __forceinline__ void pixel_decode(uint32_t w, double pitch, double half_shift_x, uint32_t& m, float& x, float& y) {
  const int col = (int)(w & 2047u) - 1024, row = (int)((w >> 11) & 2047u) - 1024;
  const double h = ((w >> 22) & 1u) ? 1.0 : -1.0;
  m = w >> 23;
  x = __double2float_rn(__dadd_rn(__dmul_rn(__dadd_rn((double)col, 0.5), pitch), __dmul_rn(h, half_shift_x)));
  y = __double2float_rn(__dmul_rn(__dadd_rn((double)row, 0.5), pitch));
}

// ---- O-4 scatter: squared miss distance of the line h0->h1 extrapolated to z of h2 ------------
// The part that depends only on (h0, h1) is hoisted by the callers: dx = x1-x0, dy = y1-y0,
// dz10 = z1-z0. Operation order is exactly O-4's.
__device__ __forceinline__ float scatter(float dx, float dy, float dz10, float x1, float y1, float z1,
                                         float x2, float y2, float z2) {
  const float tz = __fdiv_rn(__fsub_rn(z2, z1), dz10);
  const float ex = __fsub_rn(__fadd_rn(x1, __fmul_rn(dx, tz)), x2);
  const float ey = __fsub_rn(__fadd_rn(y1, __fmul_rn(dy, tz)), y2);
  return __fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey));
}

// ---- block-wide exclusive scan of one 64-bit value per thread ---------------------------------
// All threads of the CTA must call it (blockDim.x a multiple of 32, at most 1024). `warp_sums`
// is 33 words of shared memory. Returns the exclusive prefix; *total = sum over the CTA.
__device__ __forceinline__ unsigned long long block_scan_excl(unsigned long long v,
                                                              unsigned long long* warp_sums,
                                                              unsigned long long* total) {
  const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  unsigned long long inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const unsigned long long o = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= (unsigned)d) inc += o;
  }
  __syncthreads();  // protects warp_sums against the previous call's readers
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    unsigned long long w = lane < nw ? warp_sums[lane] : 0ull;
    unsigned long long wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const unsigned long long o = __shfl_up_sync(0xffffffffu, wi, d);
      if (lane >= (unsigned)d) wi += o;
    }
    warp_sums[lane] = wi - w;  // exclusive prefix of the warp sums
    if (lane == 31) warp_sums[32] = wi;
  }
  __syncthreads();
  *total = warp_sums[32];
  return warp_sums[wid] + inc - v;
}

}  // namespace velo
