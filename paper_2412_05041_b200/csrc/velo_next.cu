// velo_next.cu — the two steps that follow the VELO hot path (sm_100a):
//   velo_kalman_fit: a parameterised Kalman filter on the VELO segment of every track (§5,
//     "the Kalman filtering process on track uses a parameterised approach ... only the segment of a
//     track inside the VELO is considered"), readings K-1 ... K-5 of DESIGN.md §2;
//   velo_pv_find: primary vertices from the beamline states (§5: VELO tracks are
//     straight lines; displaced-vertex lines need primary vertices), readings P-1 ... P-6.
// Both consume the device outputs of velo_reconstruct. Every float operation is a round-to-nearest
// intrinsic in the order DESIGN.md §2 fixes (no FMA contraction): the filter's chi2 and the fitted
// vertex decide integers (track weights > 0, vertices kept), so the order is part of the method.
#include <mutex>

#include "velo_device.cuh"
#include "velo_internal.h"

namespace velo {

namespace {

// ---- f2: one thread per track -----------------------------------------------------------------------
// The hits of a track are gathered through track_hits (absolute hit indices, discovery order =
// decreasing z). The next hit's index and coordinates are loaded while the current one is filtered.
// Where the hits come from: fp32 planes, or packed pixel addresses decoded on the fly (F-2).
struct KalmanHits {
  const float *x, *y, *z;
  const uint32_t* pixel;               // or NULL
  double pitch, half_shift_x;
  float module_z[VELO_MAX_MODULES];
  __device__ __forceinline__ void get(uint32_t i, float& hx, float& hy, float& hz) const {
    if (pixel) { uint32_t m; pixel_decode(pixel[i], pitch, half_shift_x, m, hx, hy); hz = module_z[m & (VELO_MAX_MODULES - 1)]; }
    else { hx = x[i]; hy = y[i]; hz = z[i]; }
  }
};

__global__ void __launch_bounds__(256) velo_kalman_kernel(const KalmanHits H, const uint32_t* __restrict__ tho,
                                                          const uint32_t* __restrict__ th, const uint32_t* __restrict__ summary,
                                                          float sigma_hit, float ms_theta2, float* __restrict__ out,
                                                          uint32_t cap_tracks) {
  const uint32_t n_tracks = summary[2] == 0u ? summary[0] : 0u;     // a failed batch has no tracks to fit
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_tracks || t >= cap_tracks) return;
  const uint32_t a = tho[t], n = tho[t + 1] - a;
  const float s2 = __fmul_rn(sigma_hit, sigma_hit);
  uint32_t i0 = th[a], i1 = th[a + 1];
  float x0, y0, z0, x, y, zp;
  H.get(i0, x0, y0, z0);
  H.get(i1, x, y, zp);
  float dz = __fsub_rn(zp, z0);
  float tx = __fdiv_rn(__fsub_rn(x, x0), dz), ty = __fdiv_rn(__fsub_rn(y, y0), dz);
  float cxx = s2, cxtx = __fdiv_rn(s2, dz), ctxtx = __fdiv_rn(__fadd_rn(s2, s2), __fmul_rn(dz, dz));
  float chi2 = 0.0f;
  // software pipeline, two deep: while hit i is processed the coordinates of hit i+1 are in flight (through the
  // index loaded one trip earlier) and so is the index of hit i+2: a trip waits for one load, not for two in a row
  float nx = 0.0f, ny = 0.0f, nz = 0.0f;
  if (n > 2) H.get(th[a + 2], nx, ny, nz);
  uint32_t nidx = n > 3 ? th[a + 3] : 0u;
  for (uint32_t i = 2; i < n; ++i) {
    const float mx = nx, my = ny, mzz = nz;
    if (i + 1 < n) H.get(nidx, nx, ny, nz);
    if (i + 2 < n) nidx = th[a + i + 2];
    const float sl = __fadd_rn(1.0f, __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty)));
    ctxtx = __fadd_rn(ctxtx, __fmul_rn(ms_theta2, sl));
    dz = __fsub_rn(mzz, zp);
    const float xp = __fadd_rn(x, __fmul_rn(tx, dz)), yp = __fadd_rn(y, __fmul_rn(ty, dz));
    const float cxtx_p = __fadd_rn(cxtx, __fmul_rn(dz, ctxtx));
    const float cxx_p = __fadd_rn(__fadd_rn(cxx, __fmul_rn(dz, cxtx)), __fmul_rn(dz, cxtx_p));
    const float S = __fadd_rn(cxx_p, s2);
    const float k0 = __fdiv_rn(cxx_p, S), k1 = __fdiv_rn(cxtx_p, S);
    const float rx = __fsub_rn(mx, xp), ry = __fsub_rn(my, yp);
    x = __fadd_rn(xp, __fmul_rn(k0, rx)); y = __fadd_rn(yp, __fmul_rn(k0, ry));
    tx = __fadd_rn(tx, __fmul_rn(k1, rx)); ty = __fadd_rn(ty, __fmul_rn(k1, ry));
    cxx = __fmul_rn(__fsub_rn(1.0f, k0), cxx_p);
    cxtx = __fmul_rn(__fsub_rn(1.0f, k0), cxtx_p);
    ctxtx = __fsub_rn(ctxtx, __fmul_rn(k1, cxtx_p));
    const float r2 = __fadd_rn(__fmul_rn(rx, rx), __fmul_rn(ry, ry));
    chi2 = __fadd_rn(chi2, __fdiv_rn(r2, S));
    zp = mzz;
  }
  const float ss = __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty));
  ctxtx = __fadd_rn(ctxtx, __fmul_rn(ms_theta2, __fadd_rn(1.0f, ss)));
  float dzb;
  if (ss < 1e-12f) dzb = 0.0f;
  else dzb = -__fdiv_rn(__fadd_rn(__fmul_rn(x, tx), __fmul_rn(y, ty)), ss);
  const float cxtx_b = __fadd_rn(cxtx, __fmul_rn(dzb, ctxtx));
  const float cxx_b = __fadd_rn(__fadd_rn(cxx, __fmul_rn(dzb, cxtx)), __fmul_rn(dzb, cxtx_b));
  const size_t cs = cap_tracks;
  float* o = out + t;
  o[0] = __fadd_rn(x, __fmul_rn(tx, dzb)); o[cs] = __fadd_rn(y, __fmul_rn(ty, dzb));
  o[2 * cs] = tx; o[3 * cs] = ty; o[4 * cs] = __fadd_rn(zp, dzb);
  o[5 * cs] = cxx_b; o[6 * cs] = cxtx_b; o[7 * cs] = ctxtx;
  o[8 * cs] = cxx_b; o[9 * cs] = cxtx_b; o[10 * cs] = ctxtx;
  o[11 * cs] = chi2; o[12 * cs] = __uint_as_float(n);
}

// ---- f3: one warp per event ---------------------------------------------------------------------------
constexpr uint32_t kPvMax = VELO_PV_MAX_PER_EVENT;   // 32: a seed per lane
constexpr uint32_t kPvWarps = 5;                      // events per CTA: 3 CTAs of 74 KB = 15 warps per SM (4: 12 warps, 1.19 -> 1.05 ms)
// Shared memory of a warp: packed histogram, smoothed counts, seed z, one word per block of 32 bins (16-byte multiple).
__host__ __device__ inline uint32_t pv_smem_per_warp(uint32_t n_bins) {
  const uint32_t nbw = (n_bins + 1u) >> 1;
  return (4u * nbw + 4u * n_bins + 4u * kPvMax + 4u * ((n_bins + 31u) >> 5) + 15u) & ~15u;
}

struct PvArgs {
  const uint32_t* eto;        // event_track_offsets[n_events + 1]
  const float* states;        // 13 planes of `stride` words
  const uint32_t* summary;    // velo_reconstruct's summary (status)
  size_t stride;
  uint32_t n_events;
  velo_pv_params_t P;
  float inv_w;                // 1.0f / bin_width, computed once on the host in fp32
  float* tmp_pv;              // n_events * kPvMax * 5
  uint32_t* tmp_cnt;          // n_events
  uint8_t* asg;               // one byte per track (global track index)
};

__device__ __forceinline__ float warp_butterfly(float v) {
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) v = __fadd_rn(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}

__global__ void __launch_bounds__(32 * kPvWarps) velo_pv_kernel(const PvArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  const uint32_t wid = threadIdx.x >> 5, lane = threadIdx.x & 31u;
  const uint32_t nb = a.P.n_bins, nbw = (nb + 1u) >> 1;          // bins; packed-u16 words
  const uint32_t per_warp = pv_smem_per_warp(nb);
  uint32_t* hw = reinterpret_cast<uint32_t*>(smem + (size_t)wid * per_warp);   // P-1 histogram, two u16 counts per word
  uint32_t* s = hw + nbw;                                                       // P-2 smoothed counts
  float* zs = reinterpret_cast<float*>(s + nb);                                 // seed z
  uint32_t* bm = reinterpret_cast<uint32_t*>(zs + kPvMax);                      // per 32 bins: does any reach seed_min_sum?
  const uint32_t nblk = (nb + 31u) >> 5;
  const bool failed = a.summary[2] != 0u;
  const float* X = a.states; const float* Y = X + a.stride; const float* TX = Y + a.stride; const float* TY = TX + a.stride;
  const float* Z = TY + a.stride; const float* CXX = Z + a.stride;
  for (uint32_t e = blockIdx.x * kPvWarps + wid; e < a.n_events; e += gridDim.x * kPvWarps) {
    const uint32_t t0 = failed ? 0u : a.eto[e], nt = failed ? 0u : a.eto[e + 1] - t0;
    // P-1
    for (uint32_t k = lane; 4u * k < nbw; k += 32u) reinterpret_cast<uint4*>(hw)[k] = make_uint4(0u, 0u, 0u, 0u);   // (may run up to three words into s, which is written later)
    __syncwarp();
    for (uint32_t i = lane; i < nt; i += 32u) {
      const float t = __fmul_rn(__fsub_rn(Z[t0 + i], a.P.z_min), a.inv_w);
      if (t >= 0.0f && t < (float)nb) { const uint32_t b = (uint32_t)(int)t; atomicAdd(&hw[b >> 1], 1u << ((b & 1u) * 16u)); }
    }
    __syncwarp();
    // P-2 smoothed counts, then seeds in ascending bin order (ballot keeps the order)
    // A lane takes a packed word (bins 2k, 2k + 1); a ballot notes which blocks of 32 bins hold a count that
    // can seed: an event's 200 tracks touch a handful of the 75 blocks, and the seed scan skips the rest.
    const uint32_t min_sum = a.P.seed_min_sum > 1u ? a.P.seed_min_sum : 1u;
    for (uint32_t k0 = 0; k0 < nbw; k0 += 32u) {
      const uint32_t k = k0 + lane;
      uint32_t c0 = 0u, c1 = 0u;
      if (k < nbw) {
        const uint32_t wm = k > 0u ? hw[k - 1u] : 0u, wc = hw[k], wp = k + 1u < nbw ? hw[k + 1u] : 0u;
        const uint32_t lo = wc & 0xffffu, hi = wc >> 16;
        c0 = 2u * lo + (wm >> 16) + hi;
        s[2u * k] = c0;
        if (2u * k + 1u < nb) { c1 = 2u * hi + lo + (wp & 0xffffu); s[2u * k + 1u] = c1; }
      }
      const uint32_t m = __ballot_sync(0xffffffffu, c0 >= min_sum || c1 >= min_sum);
      if (lane == 0) { bm[k0 >> 4] = m & 0xffffu; if ((k0 >> 4) + 1u < nblk) bm[(k0 >> 4) + 1u] = m >> 16; }
    }
    __syncwarp();
    uint32_t ns = 0;
    const uint32_t cap = a.P.max_pv_per_event < kPvMax ? a.P.max_pv_per_event : kPvMax;
    for (uint32_t b0 = 0; b0 < nb && ns < cap; b0 += 32u) {
      if (bm[b0 >> 5] == 0u) continue;       // no bin of this block reaches seed_min_sum
      const uint32_t b = b0 + lane;
      bool ok = false;
      if (b < nb) {
        const uint32_t c = s[b];
        ok = c >= a.P.seed_min_sum && c > 0u;
        for (uint32_t j = 1; j <= a.P.seed_half_window && ok; ++j) {
          const uint32_t left = b >= j ? s[b - j] : 0u, right = b + j < nb ? s[b + j] : 0u;
          ok = (c > left) && (c >= right);
        }
      }
      const uint32_t m = __ballot_sync(0xffffffffu, ok);
      const uint32_t pos = ns + (uint32_t)__popc(m & ((1u << lane) - 1u));
      if (ok && pos < cap) zs[pos] = __fadd_rn(a.P.z_min, __fmul_rn(__fadd_rn((float)b, 0.5f), a.P.bin_width));
      ns = min(ns + (uint32_t)__popc(m), cap);
    }
    __syncwarp();
    uint32_t nout = 0;
    if (ns > 0) {
      // Once the seeds are known the histogram is dead. Fast path (the usual event): its shared memory
      // takes, per seed, 8 x 32 partial sums (lane l's column is its own: no conflicts) and the vertex
      // table, and the event's tracks (six words and the seed index each). One pass over the tracks
      // per iteration then serves every vertex of the event: a track adds to the sums of its own seed,
      // in the oracle's order (lane = track index mod 32, increasing index), and the fit iterations
      // touch no global memory.
      // With many tracks the sums of only R < ns seeds fit beside them: the seeds then go in rounds of R
      // (they are independent of each other).
      const uint32_t hist_bytes = 4u * nbw + 4u * nb;
      const uint32_t room = hist_bytes > 25u * nt + 512u ? (hist_bytes - 25u * nt - 512u) / 1024u : 0u;
      const uint32_t R = room < ns ? room : ns;                 // seeds per round
      const bool fast = R >= 1u;
      if (fast) {
        float* acc = reinterpret_cast<float*>(hw);            // [seed of the round][sum][lane]
        float* vt = acc + R * 256u;                             // [seed]{x, y, z, alive}
        const uint32_t cap2 = (hist_bytes - R * 1024u - 512u) / 25u;
        float* sx = vt + 128u;
        float* sy = sx + cap2; float* stx = sy + cap2; float* sty = stx + cap2; float* sz = sty + cap2; float* sw0 = sz + cap2;
        uint8_t* sasg = reinterpret_cast<uint8_t*>(sw0 + cap2);
        float zs_mine = lane < ns ? zs[lane] : 0.0f;
        __syncwarp();                                           // zs is read before the table below may overwrite nothing: zs lies beyond the histogram
        for (uint32_t i = lane; i < nt; i += 32u) {             // P-3
          const float z = Z[t0 + i];
          uint32_t best = 0; float bd = fabsf(__fsub_rn(z, zs[0]));
          for (uint32_t v = 1; v < ns; ++v) { const float dd = fabsf(__fsub_rn(z, zs[v])); if (dd < bd) { bd = dd; best = v; } }
          sasg[i] = (uint8_t)best;
          sx[i] = X[t0 + i]; sy[i] = Y[t0 + i]; stx[i] = TX[t0 + i]; sty[i] = TY[t0 + i]; sz[i] = z;
          sw0[i] = __fdiv_rn(1.0f, CXX[t0 + i]);
        }
        if (lane < ns) { vt[4u * lane] = 0.0f; vt[4u * lane + 1u] = 0.0f; vt[4u * lane + 2u] = zs_mine; vt[4u * lane + 3u] = 1.0f; }
        float my_s0 = 0.0f; uint32_t my_n = 0;                  // lane v keeps seed v's last sums
        __syncwarp();
        for (uint32_t v0 = 0; v0 < ns; v0 += R) {
        const uint32_t v1 = min(v0 + R, ns);
        for (uint32_t it = 0; it < a.P.n_iterations; ++it) {
          for (uint32_t j = lane; j < (v1 - v0) * 256u; j += 32u) acc[j] = 0.0f;
          __syncwarp();
          for (uint32_t i = lane; i < nt; i += 32u) {           // P-4 and the sums of P-5
            const uint32_t v = sasg[i];
            if (v < v0 || v >= v1) continue;
            const float4 vx = *reinterpret_cast<const float4*>(vt + 4u * v);
            if (vx.w == 0.0f) continue;
            const float x = sx[i], y = sy[i], tx = stx[i], ty = sty[i], z = sz[i], w0 = sw0[i];
            const float dz = __fsub_rn(vx.z, z);
            const float rx = __fsub_rn(__fadd_rn(x, __fmul_rn(tx, dz)), vx.x);
            const float ry = __fsub_rn(__fadd_rn(y, __fmul_rn(ty, dz)), vx.y);
            const float c = __fmul_rn(w0, __fadd_rn(__fmul_rn(rx, rx), __fmul_rn(ry, ry)));
            float wt = 0.0f;
            if (c < a.P.chi2_max) { const float u = __fsub_rn(1.0f, __fdiv_rn(c, a.P.chi2_max)); wt = __fmul_rn(u, u); }
            const float w = __fmul_rn(w0, wt);
            const float aa = __fsub_rn(x, __fmul_rn(tx, z)), bb = __fsub_rn(y, __fmul_rn(ty, z));
            const float t2 = __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty));
            const float ab = __fadd_rn(__fmul_rn(tx, aa), __fmul_rn(ty, bb));
            float* q = acc + (v - v0) * 256u + lane;
            q[0] = __fadd_rn(q[0], w);
            q[32] = __fadd_rn(q[32], __fmul_rn(w, tx)); q[64] = __fadd_rn(q[64], __fmul_rn(w, ty));
            q[96] = __fadd_rn(q[96], __fmul_rn(w, t2));
            q[128] = __fadd_rn(q[128], __fmul_rn(w, aa)); q[160] = __fadd_rn(q[160], __fmul_rn(w, bb));
            q[192] = __fadd_rn(q[192], __fmul_rn(w, ab));
            if (wt > 0.0f) q[224] = __fadd_rn(q[224], 1.0f);
          }
          __syncwarp();
          // the rest of P-5: the sums vertex by vertex (every lane gets them; lane v keeps vertex v's), then
          // the closed form for all vertices of the round at once, lane v solving vertex v
          float lS0 = 0.0f, lSx = 0.0f, lSy = 0.0f, lSxx = 0.0f, lA = 0.0f, lB = 0.0f, lC = 0.0f;
          bool mine = false;
          for (uint32_t v = v0; v < v1; ++v) {
            if (vt[4u * v + 3u] == 0.0f) continue;
            const float* q = acc + (v - v0) * 256u + lane;
            const float S0 = warp_butterfly(q[0]);
            const float Sx = warp_butterfly(q[32]), Sy = warp_butterfly(q[64]), Sxx = warp_butterfly(q[96]);
            const float A = warp_butterfly(q[128]), B = warp_butterfly(q[160]), C = warp_butterfly(q[192]);
            const uint32_t ntrk = (uint32_t)warp_butterfly(q[224]);
            if (lane == v) { my_s0 = S0; my_n = ntrk; lS0 = S0; lSx = Sx; lSy = Sy; lSxx = Sxx; lA = A; lB = B; lC = C; mine = true; }
          }
          __syncwarp();
          if (mine) {
            bool alive = lS0 > 0.0f;
            float den = 0.0f;
            if (alive) { den = __fsub_rn(lSxx, __fdiv_rn(__fadd_rn(__fmul_rn(lSx, lSx), __fmul_rn(lSy, lSy)), lS0)); alive = den > 0.0f; }
            if (!alive) vt[4u * lane + 3u] = 0.0f;
            else {
              const float zv = __fdiv_rn(__fsub_rn(__fdiv_rn(__fadd_rn(__fmul_rn(lSx, lA), __fmul_rn(lSy, lB)), lS0), lC), den);
              const float xv = __fdiv_rn(__fadd_rn(lA, __fmul_rn(lSx, zv)), lS0);
              const float yv = __fdiv_rn(__fadd_rn(lB, __fmul_rn(lSy, zv)), lS0);
              vt[4u * lane] = xv; vt[4u * lane + 1u] = yv; vt[4u * lane + 2u] = zv;
            }
          }
          __syncwarp();
        }
        }
        for (uint32_t v = 0; v < ns; ++v) {                     // P-6
          const float s0v = __shfl_sync(0xffffffffu, my_s0, v);
          const uint32_t nv = __shfl_sync(0xffffffffu, my_n, v);
          if (vt[4u * v + 3u] != 0.0f && nv >= a.P.min_tracks) {
            if (lane == 0) {
              float* o = a.tmp_pv + ((size_t)e * kPvMax + nout) * 5u;
              o[0] = vt[4u * v]; o[1] = vt[4u * v + 1u]; o[2] = vt[4u * v + 2u]; o[3] = s0v; o[4] = __uint_as_float(nv);
            }
            ++nout;
          }
        }
      } else {
      // Once the seeds are known the histogram is dead: its shared memory takes the event's tracks
        // (six words and the seed index each), so that the fit iterations touch no global memory. An
        // event with more tracks than fit there reads them from global memory instead, in the same order.
        const uint32_t stage_cap = (4u * nbw + 4u * nb) / 25u;
        const bool resident = nt <= stage_cap;
        float* sx = reinterpret_cast<float*>(hw);
        float* sy = sx + stage_cap; float* stx = sy + stage_cap; float* sty = stx + stage_cap;
        float* sz = sty + stage_cap; float* sw0 = sz + stage_cap;
        uint8_t* sasg = reinterpret_cast<uint8_t*>(sw0 + stage_cap);
        // P-3 every track to its nearest seed (ties to the lower seed)
        for (uint32_t i = lane; i < nt; i += 32u) {
          const float z = Z[t0 + i];
          uint32_t best = 0; float bd = fabsf(__fsub_rn(z, zs[0]));
          for (uint32_t v = 1; v < ns; ++v) { const float dd = fabsf(__fsub_rn(z, zs[v])); if (dd < bd) { bd = dd; best = v; } }
          if (resident) {
            sasg[i] = (uint8_t)best;
            sx[i] = X[t0 + i]; sy[i] = Y[t0 + i]; stx[i] = TX[t0 + i]; sty[i] = TY[t0 + i]; sz[i] = z;
            sw0[i] = __fdiv_rn(1.0f, CXX[t0 + i]);
          } else {
            a.asg[t0 + i] = (uint8_t)best;
          }
        }
        __syncwarp();
        const float* PX = resident ? sx : X + t0; const float* PY = resident ? sy : Y + t0;
        const float* PTX = resident ? stx : TX + t0; const float* PTY = resident ? sty : TY + t0;
        const float* PZ = resident ? sz : Z + t0; const float* PW = resident ? sw0 : CXX + t0;
        const uint8_t* PA = resident ? sasg : a.asg + t0;
        // P-4, P-5, P-6: lane l sums the tracks with i mod 32 == l in increasing i, butterfly combine
        for (uint32_t v = 0; v < ns; ++v) {
          float xv = 0.0f, yv = 0.0f, zv = zs[v], S0 = 0.0f;
          uint32_t ntrk = 0; bool alive = true;
          for (uint32_t it = 0; it < a.P.n_iterations && alive; ++it) {
            float l0 = 0.0f, lx = 0.0f, ly = 0.0f, lxx = 0.0f, la = 0.0f, lb = 0.0f, lc = 0.0f, ln = 0.0f;
            for (uint32_t i = lane; i < nt; i += 32u) {
              if (PA[i] != v) continue;
              const float x = PX[i], y = PY[i], tx = PTX[i], ty = PTY[i], z = PZ[i];
              const float w0 = resident ? PW[i] : __fdiv_rn(1.0f, PW[i]);
              const float dz = __fsub_rn(zv, z);
              const float rx = __fsub_rn(__fadd_rn(x, __fmul_rn(tx, dz)), xv);
              const float ry = __fsub_rn(__fadd_rn(y, __fmul_rn(ty, dz)), yv);
              const float c = __fmul_rn(w0, __fadd_rn(__fmul_rn(rx, rx), __fmul_rn(ry, ry)));
              float wt = 0.0f;
              if (c < a.P.chi2_max) { const float u = __fsub_rn(1.0f, __fdiv_rn(c, a.P.chi2_max)); wt = __fmul_rn(u, u); }
              const float w = __fmul_rn(w0, wt);
              const float aa = __fsub_rn(x, __fmul_rn(tx, z)), bb = __fsub_rn(y, __fmul_rn(ty, z));
              const float t2 = __fadd_rn(__fmul_rn(tx, tx), __fmul_rn(ty, ty));
              const float ab = __fadd_rn(__fmul_rn(tx, aa), __fmul_rn(ty, bb));
              l0 = __fadd_rn(l0, w);
              lx = __fadd_rn(lx, __fmul_rn(w, tx)); ly = __fadd_rn(ly, __fmul_rn(w, ty));
              lxx = __fadd_rn(lxx, __fmul_rn(w, t2));
              la = __fadd_rn(la, __fmul_rn(w, aa)); lb = __fadd_rn(lb, __fmul_rn(w, bb));
              lc = __fadd_rn(lc, __fmul_rn(w, ab));
              if (wt > 0.0f) ln = __fadd_rn(ln, 1.0f);
            }
            S0 = warp_butterfly(l0);
            const float Sx = warp_butterfly(lx), Sy = warp_butterfly(ly), Sxx = warp_butterfly(lxx);
            const float A = warp_butterfly(la), B = warp_butterfly(lb), C = warp_butterfly(lc);
            ntrk = (uint32_t)warp_butterfly(ln);
            if (!(S0 > 0.0f)) { alive = false; break; }
            const float den = __fsub_rn(Sxx, __fdiv_rn(__fadd_rn(__fmul_rn(Sx, Sx), __fmul_rn(Sy, Sy)), S0));
            if (!(den > 0.0f)) { alive = false; break; }
            zv = __fdiv_rn(__fsub_rn(__fdiv_rn(__fadd_rn(__fmul_rn(Sx, A), __fmul_rn(Sy, B)), S0), C), den);
            xv = __fdiv_rn(__fadd_rn(A, __fmul_rn(Sx, zv)), S0);
            yv = __fdiv_rn(__fadd_rn(B, __fmul_rn(Sy, zv)), S0);
          }
          if (alive && ntrk >= a.P.min_tracks) {
            if (lane == 0) {
              float* o = a.tmp_pv + ((size_t)e * kPvMax + nout) * 5u;
              o[0] = xv; o[1] = yv; o[2] = zv; o[3] = S0; o[4] = __uint_as_float(ntrk);
            }
            ++nout;
          }
        }
      }
    }
    if (lane == 0) a.tmp_cnt[e] = nout;
    __syncwarp();
  }
}

// counts -> event_pv_offsets (one CTA), then every event's vertices to their place (a thread per slot)
__global__ void __launch_bounds__(1024) velo_pv_offsets_kernel(const PvArgs a, uint32_t* event_pv_offsets, uint32_t cap_pvs,
                                                               uint32_t* pv_summary) {
  __shared__ unsigned long long warp_sums[33];
  const uint32_t tid = threadIdx.x, nthr = blockDim.x, ne = a.n_events;
  const uint32_t per = (ne + nthr - 1) / nthr;
  const uint32_t e0 = min(tid * per, ne), e1 = min(e0 + per, ne);
  unsigned long long sum = 0;
#pragma unroll 8
  for (uint32_t e = e0; e < e1; ++e) sum += a.tmp_cnt[e];
  unsigned long long tot;
  unsigned long long run = block_scan_excl(sum, warp_sums, &tot);
#pragma unroll 8
  for (uint32_t e = e0; e < e1; ++e) { event_pv_offsets[e] = (uint32_t)run; run += a.tmp_cnt[e]; }
  if (tid == 0) {
    event_pv_offsets[ne] = (uint32_t)tot;
    uint32_t status = a.summary[2];
    if (status == 0u && tot > cap_pvs) status = (uint32_t)VELO_ERR_CAPACITY;
    pv_summary[0] = (uint32_t)tot; pv_summary[1] = status; pv_summary[2] = 0u; pv_summary[3] = 0u;
  }
}

__global__ void __launch_bounds__(256) velo_pv_place_kernel(const PvArgs a, const uint32_t* event_pv_offsets, float* pvs,
                                                            uint32_t cap_pvs) {
  if (event_pv_offsets[a.n_events] > cap_pvs) return;      // VELO_ERR_CAPACITY: nothing valid
  const size_t slot = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t e = (uint32_t)(slot / kPvMax), k = (uint32_t)(slot % kPvMax);
  if (e >= a.n_events || k >= a.tmp_cnt[e]) return;
  const float* src = a.tmp_pv + slot * 5u;
  const uint32_t dst = event_pv_offsets[e] + k;
#pragma unroll
  for (uint32_t p = 0; p < 5; ++p) pvs[(size_t)p * cap_pvs + dst] = src[p];
}

struct PvWorkspace { float* tmp_pv; uint32_t* tmp_cnt; uint8_t* asg; size_t bytes; };
PvWorkspace carve_pv(void* base, uint32_t n_events, uint32_t cap_tracks) {
  PvWorkspace w{};
  size_t o = 0;
  unsigned char* b = (unsigned char*)base;
  auto take = [&](size_t bytes) { size_t r = o; o += ((bytes + 255) / 256) * 256; return b + r; };
  w.tmp_pv = (float*)take(sizeof(float) * 5u * kPvMax * ((size_t)n_events + 1));
  w.tmp_cnt = (uint32_t*)take(4 * ((size_t)n_events + 1));
  w.asg = (uint8_t*)take((size_t)cap_tracks + 1);
  w.bytes = o;
  return w;
}

// ---- velo_pv_find_static: the finder's scratch as a fixed array inside the library ------------------
// For callers that cannot allocate (include/velo.h). In HOST code the name g_pv_static is a host-side
// stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, once per
// device, with that device current. Every call on a device shares the array (calls that overlap race).
constexpr size_t r256(size_t b) { return (b + 255) / 256 * 256; }
constexpr size_t kPvStaticBytes = r256(sizeof(float) * 5u * kPvMax * ((size_t)VELO_PV_STATIC_MAX_EVENTS + 1)) +
                                  r256(4 * ((size_t)VELO_PV_STATIC_MAX_EVENTS + 1)) +
                                  r256((size_t)VELO_PV_STATIC_MAX_TRACKS + 1);       // = carve_pv at the two maxima
static_assert(kPvStaticBytes == 4736256, "include/velo.h states this size");
static __device__ __align__(256) unsigned char g_pv_static[kPvStaticBytes];

constexpr int kMaxDevices = 64;
std::mutex g_pv_static_mutex;
void* g_pv_static_ptr[kMaxDevices] = {};     // device address of g_pv_static on device i, once looked up

// Device address of the array on the current device; nullptr if a CUDA call fails.
void* pv_static_address() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
  std::lock_guard<std::mutex> lock(g_pv_static_mutex);
  if (!g_pv_static_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_pv_static) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    g_pv_static_ptr[dev] = p;
  }
  return g_pv_static_ptr[dev];
}

}  // namespace

}  // namespace velo

extern "C" {

static int kalman_launch(const velo::KalmanHits& H, const velo_tracks_t* tracks, float sigma_hit, float ms_theta2,
                         float* kalman_states, void* stream) {
  if (!tracks || !kalman_states) return VELO_ERR_ARG;
  if (!tracks->track_hit_offsets || !tracks->track_hits || !tracks->summary || tracks->cap_tracks == 0) return VELO_ERR_ARG;
  if (!(sigma_hit > 0.0f) || !(ms_theta2 >= 0.0f)) return VELO_ERR_ARG;
  const uint32_t threads = 256, grid = (tracks->cap_tracks + threads - 1) / threads;
  velo::velo_kalman_kernel<<<grid, threads, 0, (cudaStream_t)stream>>>(
      H, tracks->track_hit_offsets, tracks->track_hits, tracks->summary, sigma_hit, ms_theta2, kalman_states, tracks->cap_tracks);
  return cudaGetLastError() == cudaSuccess ? VELO_OK : VELO_ERR_CUDA;
}

int velo_kalman_fit(const velo_hits_t* hits, const velo_tracks_t* tracks, float sigma_hit, float ms_theta2,
                    float* kalman_states, void* stream) {
  if (!hits) return VELO_ERR_ARG;
  if (hits->n_hits && (!hits->x || !hits->y || !hits->z)) return VELO_ERR_ARG;
  velo::KalmanHits H{};
  H.x = hits->x; H.y = hits->y; H.z = hits->z;
  return kalman_launch(H, tracks, sigma_hit, ms_theta2, kalman_states, stream);
}

int velo_kalman_fit_pixels(const velo_geometry_t* g, const velo_pixel_hits_t* hits, const velo_pixel_format_t* fmt,
                           const velo_tracks_t* tracks, float sigma_hit, float ms_theta2, float* kalman_states, void* stream) {
  if (!g || !hits || !fmt || !hits->pixel || !(fmt->pitch > 0.0)) return VELO_ERR_ARG;
  velo::KalmanHits H{};
  H.pixel = hits->pixel; H.pitch = fmt->pitch; H.half_shift_x = fmt->half_shift_x;
  for (uint32_t m = 0; m < VELO_MAX_MODULES; ++m) H.module_z[m] = m < g->n_modules ? g->module_z[m] : 0.0f;
  return kalman_launch(H, tracks, sigma_hit, ms_theta2, kalman_states, stream);
}

void velo_pv_params_default(velo_pv_params_t* p) {
  if (!p) return;
  p->z_min = -300.0f; p->bin_width = 0.25f; p->n_bins = 2400;
  p->seed_min_sum = 5; p->seed_half_window = 6;
  p->chi2_max = 16.0f; p->n_iterations = 4; p->min_tracks = 4; p->max_pv_per_event = VELO_PV_MAX_PER_EVENT;
}

size_t velo_pv_workspace_bytes(uint32_t n_events, uint32_t cap_tracks) {
  return velo::carve_pv(nullptr, n_events, cap_tracks).bytes;
}

int velo_pv_find(const velo_tracks_t* tracks, uint32_t n_events, const velo_pv_params_t* params, velo_pvs_t* out,
                 void* workspace, size_t workspace_bytes, void* stream) {
  using namespace velo;
  if (!tracks || !params || !out || !workspace) return VELO_ERR_ARG;
  if (!tracks->event_track_offsets || !tracks->states || !tracks->summary || tracks->cap_tracks == 0) return VELO_ERR_ARG;
  if (!out->event_pv_offsets || !out->pvs || !out->summary || out->cap_pvs == 0) return VELO_ERR_ARG;
  if (params->n_bins == 0 || params->n_bins > VELO_PV_MAX_BINS || !(params->bin_width > 0.0f) || !(params->chi2_max > 0.0f))
    return VELO_ERR_ARG;
  if (((uintptr_t)workspace & 255u) != 0) return VELO_ERR_ARG;
  const PvWorkspace w = carve_pv(workspace, n_events, tracks->cap_tracks);
  if (workspace_bytes < w.bytes) return VELO_ERR_WORKSPACE;
  PvArgs a{};
  a.eto = tracks->event_track_offsets; a.states = tracks->states; a.summary = tracks->summary;
  a.stride = tracks->cap_tracks; a.n_events = n_events; a.P = *params;
  a.inv_w = 1.0f / params->bin_width;
  a.tmp_pv = w.tmp_pv; a.tmp_cnt = w.tmp_cnt; a.asg = w.asg;
  cudaStream_t st = (cudaStream_t)stream;
  const uint32_t smem = kPvWarps * pv_smem_per_warp(params->n_bins);
  cudaError_t err = cudaFuncSetAttribute(velo_pv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err != cudaSuccess) return VELO_ERR_CUDA;
  if (n_events > 0) {
    uint32_t grid = (n_events + kPvWarps - 1) / kPvWarps;
    const uint32_t most = num_sms() * 8u;
    if (grid > most) grid = most;
    velo_pv_kernel<<<grid, 32 * kPvWarps, smem, st>>>(a);
  }
  velo_pv_offsets_kernel<<<1, 1024, 0, st>>>(a, out->event_pv_offsets, out->cap_pvs, out->summary);
  if (n_events > 0) {
    const size_t slots = (size_t)n_events * kPvMax;
    velo_pv_place_kernel<<<(uint32_t)((slots + 255) / 256), 256, 0, st>>>(a, out->event_pv_offsets, out->pvs, out->cap_pvs);
  }
  return cudaGetLastError() == cudaSuccess ? VELO_OK : VELO_ERR_CUDA;
}

// The same launches as velo_pv_find over the library's own array: no allocation of any kind.
int velo_pv_find_static(const velo_tracks_t* tracks, uint32_t n_events, const velo_pv_params_t* params, velo_pvs_t* out,
                        void* stream) {
  using namespace velo;
  if (!tracks || !params || !out) return VELO_ERR_ARG;
  if (!tracks->event_track_offsets || !tracks->states || !tracks->summary || tracks->cap_tracks == 0) return VELO_ERR_ARG;
  if (!out->event_pv_offsets || !out->pvs || !out->summary || out->cap_pvs == 0) return VELO_ERR_ARG;
  if (params->n_bins == 0 || params->n_bins > VELO_PV_MAX_BINS || !(params->bin_width > 0.0f) || !(params->chi2_max > 0.0f))
    return VELO_ERR_ARG;
  if (n_events > VELO_PV_STATIC_MAX_EVENTS || tracks->cap_tracks > VELO_PV_STATIC_MAX_TRACKS) return VELO_ERR_STATIC_LIMIT;
  void* base = pv_static_address();
  if (!base) return VELO_ERR_CUDA;
  const PvWorkspace w = carve_pv(base, n_events, tracks->cap_tracks);
  if (w.bytes > kPvStaticBytes) return VELO_ERR_STATIC_LIMIT;      // cannot happen below the two maxima
  PvArgs a{};
  a.eto = tracks->event_track_offsets; a.states = tracks->states; a.summary = tracks->summary;
  a.stride = tracks->cap_tracks; a.n_events = n_events; a.P = *params;
  a.inv_w = 1.0f / params->bin_width;
  a.tmp_pv = w.tmp_pv; a.tmp_cnt = w.tmp_cnt; a.asg = w.asg;
  cudaStream_t st = (cudaStream_t)stream;
  const uint32_t smem = kPvWarps * pv_smem_per_warp(params->n_bins);
  if (cudaFuncSetAttribute(velo_pv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return VELO_ERR_CUDA;
  if (n_events > 0) {
    uint32_t grid = (n_events + kPvWarps - 1) / kPvWarps;
    const uint32_t most = num_sms() * 8u;
    if (grid > most) grid = most;
    velo_pv_kernel<<<grid, 32 * kPvWarps, smem, st>>>(a);
  }
  velo_pv_offsets_kernel<<<1, 1024, 0, st>>>(a, out->event_pv_offsets, out->cap_pvs, out->summary);
  if (n_events > 0) {
    const size_t slots = (size_t)n_events * kPvMax;
    velo_pv_place_kernel<<<(uint32_t)((slots + 255) / 256), 256, 0, st>>>(a, out->event_pv_offsets, out->pvs, out->cap_pvs);
  }
  return cudaGetLastError() == cudaSuccess ? VELO_OK : VELO_ERR_CUDA;
}

}  // extern "C"
