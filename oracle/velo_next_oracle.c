/* velo_next_oracle.c — plain, slow, single-threaded CPU oracle for the steps around the VELO hot path
 * in SURVEY.md §8(f): f1, the decode of packed pixel hits in front of it; f2, a parameterised Kalman
 * filter on the VELO segment of every track, and f3, primary-vertex finding from the beamline states.
 *
 * TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may build,
 * load or call it. It shares no code, header, table or helper with paper_2412_05041_b200/csrc.
 *
 * What the paper says: "the Kalman filtering process on track uses a parameterised approach ...
 * only the segment of a track inside the VELO is considered for the filtering process"
 * (§5); displaced-vertex lines such as TwoTrackKs (§5) need primary
 * vertices, and VELO tracks are straight lines (§5). It gives no formula, constant or
 * worked example for either step, so every step below is the reading fixed in DESIGN.md §2
 * (K-1 ... K-5 for the filter, P-1 ... P-6 for the vertices), written out in that order.
 *
 * Arithmetic: IEEE-754 binary32, round-to-nearest-even, one rounding per written operator, no
 * fused multiply-add. Build with: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math.
 *
 * Sums over the tracks of an event (P-5) are DEFINED as: 32 partial sums, track i of the event
 * (i = 0, 1, ... in output order) added to partial i mod 32 in increasing i, then the 32 partials
 * combined by a butterfly (partner l xor 16, then 8, 4, 2, 1). The order is part of the method's
 * definition here because the fitted vertex decides which tracks keep a non-zero weight.
 *
 * Parity status versus the paper: UNPINNED (no number or worked example in the paper). Pins:
 * tests/test_oracle_next.py — closed forms (zero-noise filter == least-squares line, two-point
 * start, one-scatterer hand case, tracks from one point give that point), brute-force
 * restatements of the seed search, a double-precision weighted least-squares solve, and the
 * generator's vertex and track truth (efficiency, resolution, pulls).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ================================ f1: packed pixel hits ======================================== */
/* The paper says only that the VELO is a pixel detector read out as raw data (PAPER.md:24 §2, :42 §3);
 * the format is this repository's (DESIGN.md §2 F-1, F-2):
 * F-1 one u32 per hit: bits 0-10 column + 1024, bits 11-21 row + 1024, bit 22 half (1 = the +x half),
 *     bits 23-27 module; column and row count pixels of `pitch` from the half's local origin.
 * F-2 decode: x = fl32(((double)column + 0.5) * pitch + h * half_shift_x), y = fl32(((double)row + 0.5) * pitch)
 *     with h = +1 / -1 for the half bit, in double precision with one final rounding; z = module_z[module].
 * Returns 0, or -1 if a module id is out of range (nothing else can be wrong in a 28-bit address). */
int vn_pixel_decode(uint32_t n, const uint32_t* pixel, double pitch, double half_shift_x, const float* module_z,
                    uint32_t n_modules, float* x, float* y, float* z, uint8_t* module) {
  for (uint32_t i = 0; i < n; ++i) {
    const uint32_t w = pixel[i];
    const int32_t col = (int32_t)(w & 2047u) - 1024, row = (int32_t)((w >> 11) & 2047u) - 1024;
    const double h = ((w >> 22) & 1u) ? 1.0 : -1.0;
    const uint32_t m = w >> 23;
    if (m >= n_modules) return -1;
    x[i] = (float)(((double)col + 0.5) * pitch + h * half_shift_x);
    y[i] = (float)(((double)row + 0.5) * pitch);
    z[i] = module_z[m];
    module[i] = (uint8_t)m;
  }
  return 0;
}

/* ================================ f2: Kalman filter on the VELO segment ======================= */
/* K-1 model: x(z) and y(z) are independent straight lines with state (x, tx), (y, ty); z is exact;
 *     every hit measures x and y with variance sigma_hit^2 (the same for both, so the two filters
 *     share one 2x2 covariance); at every measured plane the slopes pick up multiple-scattering
 *     noise of variance theta2 = ms_theta2 * (1 + tx^2 + ty^2)  ("parameterised": one constant,
 *     scaled by the path length through the plane; default ms_theta2 = (0.3 mrad)^2 = 9e-8).
 * K-2 direction: hits in discovery order (decreasing z): the filter runs from the most downstream
 *     hit towards the beamline, where the state is wanted.
 * K-3 start: exact two-point state at the second hit: tx = (x1-x0)/(z1-z0), x = x1,
 *     cxx = s2, cxtx = s2/dz, ctxtx = (s2+s2)/(dz*dz)   with s2 = sigma_hit^2, dz = z1-z0; chi2 = 0.
 * K-4 step to hit i >= 2: noise at the plane just left (ctxtx += theta2 with the current slopes),
 *     transport by dz = z_i - z_(i-1), update with (x_i, y_i), chi2 += (rx^2 + ry^2) / S.
 * K-5 output: the slopes pick up the noise of the last plane too (the particle came through it on its
 *     way from the beamline), then the state at the last (most upstream) hit is moved to the point of
 *     closest approach to the z axis exactly as O-11 does for the least-squares line; 13 words in the O-11 layout
 *     (x, y, tx, ty, z, cxx, cxtx, ctxtx, cyy = cxx, cyty = cxtx, ctyty = ctxtx, chi2, n bits);
 *     ndof = 2n - 4. */
void vn_kalman(uint32_t n, const float* hx, const float* hy, const float* hz, float sigma_hit, float ms_theta2,
               float* out13) {
  const float s2 = sigma_hit * sigma_hit;
  float dz = hz[1] - hz[0];
  float tx = (hx[1] - hx[0]) / dz;
  float ty = (hy[1] - hy[0]) / dz;
  float x = hx[1], y = hy[1];
  float cxx = s2;
  float cxtx = s2 / dz;
  float ctxtx = (s2 + s2) / (dz * dz);
  float chi2 = 0.0f;
  for (uint32_t i = 2; i < n; ++i) {
    /* K-4: scattering in the plane of hit i-1 */
    float sl = tx * tx;
    sl = sl + ty * ty;
    sl = 1.0f + sl;
    ctxtx = ctxtx + ms_theta2 * sl;
    /* transport to the plane of hit i */
    dz = hz[i] - hz[i - 1];
    float xp = x + tx * dz;
    float yp = y + ty * dz;
    float cxtx_p = cxtx + dz * ctxtx;
    float cxx_p = cxx + dz * cxtx;
    cxx_p = cxx_p + dz * cxtx_p;          /* cxx + 2 dz cxtx + dz^2 ctxtx, as (cxx + dz cxtx) + dz (cxtx + dz ctxtx) */
    /* update */
    float S = cxx_p + s2;
    float k0 = cxx_p / S;
    float k1 = cxtx_p / S;
    float rx = hx[i] - xp;
    float ry = hy[i] - yp;
    x = xp + k0 * rx;
    y = yp + k0 * ry;
    tx = tx + k1 * rx;
    ty = ty + k1 * ry;
    cxx = (1.0f - k0) * cxx_p;
    cxtx = (1.0f - k0) * cxtx_p;
    ctxtx = ctxtx - k1 * cxtx_p;
    float r2 = rx * rx;
    r2 = r2 + ry * ry;
    chi2 = chi2 + r2 / S;
  }
  /* K-5: scattering in the plane of the last hit, then to the point of closest approach to the z axis */
  float ss = tx * tx;
  ss = ss + ty * ty;
  ctxtx = ctxtx + ms_theta2 * (1.0f + ss);
  float dzb;
  if (ss < 1e-12f) dzb = 0.0f;
  else {
    float num = x * tx;
    num = num + y * ty;
    dzb = -(num / ss);
  }
  float cxtx_b = cxtx + dzb * ctxtx;
  float cxx_b = cxx + dzb * cxtx;
  cxx_b = cxx_b + dzb * cxtx_b;
  out13[0] = x + tx * dzb;
  out13[1] = y + ty * dzb;
  out13[2] = tx;
  out13[3] = ty;
  out13[4] = hz[n - 1] + dzb;
  out13[5] = cxx_b; out13[6] = cxtx_b; out13[7] = ctxtx;
  out13[8] = cxx_b; out13[9] = cxtx_b; out13[10] = ctxtx;
  out13[11] = chi2;
  uint32_t nn = n;
  memcpy(&out13[12], &nn, 4);
}

/* Every track of a batch: hits gathered through track_hits (global original hit indices, discovery
 * order). states_out: 13 planes of n_tracks words. */
void vn_kalman_tracks(uint32_t n_tracks, const uint32_t* track_hit_offsets, const uint32_t* track_hits, const float* x,
                      const float* y, const float* z, float sigma_hit, float ms_theta2, float* states_out) {
  float hx[64], hy[64], hz[64], s[13];
  for (uint32_t t = 0; t < n_tracks; ++t) {
    const uint32_t a = track_hit_offsets[t], n = track_hit_offsets[t + 1] - a;
    for (uint32_t i = 0; i < n && i < 64; ++i) {
      hx[i] = x[track_hits[a + i]]; hy[i] = y[track_hits[a + i]]; hz[i] = z[track_hits[a + i]];
    }
    vn_kalman(n, hx, hy, hz, sigma_hit, ms_theta2, s);
    for (int k = 0; k < 13; ++k) states_out[(size_t)k * n_tracks + t] = s[k];
  }
}

/* ================================ f3: primary vertices from the beamline states =============== */
typedef struct {
  float z_min, bin_width;      /* P-1 histogram of the tracks' z at the beamline: -300 mm, 0.25 mm */
  uint32_t n_bins;             /* 2400 */
  uint32_t seed_min_sum;       /* P-2: smoothed count a seed needs: 5 */
  uint32_t seed_half_window;   /* P-2: a seed is the maximum within +- this many bins: 6 */
  float chi2_max;              /* P-4: Tukey cut on a track's chi2 to the vertex: 16 */
  uint32_t n_iterations;       /* P-5: 4 */
  uint32_t min_tracks;         /* P-6: 4 */
  uint32_t max_pv_per_event;   /* P-2: at most 32 seeds per event, lowest z first */
} vn_pv_params_t;

#define VN_MAX_PV 32

/* P-1 bin of a track; -1 if outside the histogram. inv_w = 1.0f / bin_width (one fp32 division). */
int32_t vn_pv_bin(float z, float z_min, float inv_w, uint32_t n_bins) {
  float t = (z - z_min) * inv_w;
  if (!(t >= 0.0f) || !(t < (float)n_bins)) return -1;
  return (int32_t)t;
}

/* P-2 seeds of one histogram: s[b] = h[b-1] + 2 h[b] + h[b+1] (0 outside); b is a seed iff
 * s[b] >= seed_min_sum, s[b] > s[b-j] and s[b] >= s[b+j] for j = 1 .. seed_half_window (values
 * outside the histogram count as 0). Ascending b, at most max_pv. Returns the number of seeds. */
uint32_t vn_pv_seeds(const uint32_t* h, uint32_t n_bins, const vn_pv_params_t* P, uint32_t* seed_bins) {
  uint32_t ns = 0;
  uint32_t* s = (uint32_t*)calloc(n_bins ? n_bins : 1, sizeof(uint32_t));
  for (uint32_t b = 0; b < n_bins; ++b) {
    uint32_t v = 2u * h[b];
    if (b > 0) v += h[b - 1];
    if (b + 1 < n_bins) v += h[b + 1];
    s[b] = v;
  }
  const uint32_t cap = P->max_pv_per_event < VN_MAX_PV ? P->max_pv_per_event : VN_MAX_PV;
  for (uint32_t b = 0; b < n_bins && ns < cap; ++b) {
    if (s[b] < P->seed_min_sum || s[b] == 0) continue;
    int ok = 1;
    for (uint32_t j = 1; j <= P->seed_half_window && ok; ++j) {
      uint32_t left = b >= j ? s[b - j] : 0u;
      uint32_t right = b + j < n_bins ? s[b + j] : 0u;
      if (!(s[b] > left) || !(s[b] >= right)) ok = 0;
    }
    if (ok) seed_bins[ns++] = b;
  }
  free(s);
  return ns;
}

/* P-5 sum: 32 partials by track index mod 32, butterfly combine. */
static float vn_butterfly(float* lane) {
  for (int d = 16; d >= 1; d >>= 1) {
    float t[32];
    for (int l = 0; l < 32; ++l) t[l] = lane[l] + lane[l ^ d];
    for (int l = 0; l < 32; ++l) lane[l] = t[l];
  }
  return lane[0];
}

/* One event. st: 13 planes with stride `stride`, tracks t0 .. t0+nt-1. out: up to VN_MAX_PV vertices
 * of 5 words (x, y, z, sum of weights, n_tracks as u32 bits). Returns the number of vertices kept.
 * P-3 assignment: every track goes to the seed nearest in z (|z_i - z_seed|, ties to the lower
 *     seed), once, before the fits; z_seed = z_min + ((float)b + 0.5f) * bin_width.
 * P-4 weight of track i for vertex (xv, yv, zv): dz = zv - z_i; rx = (x_i + tx_i*dz) - xv;
 *     ry likewise; c = w0_i * (rx*rx + ry*ry) with w0_i = 1.0f / cxx_i; wt = (1 - c/chi2_max)^2 if
 *     c < chi2_max, else 0; w = w0_i * wt.
 * P-5 fit: xv = yv = 0, zv = z_seed; n_iterations times: with a_i = x_i - tx_i*z_i, b_i = y_i - ty_i*z_i
 *     S0 = sum w, Sx = sum w tx, Sy = sum w ty, Sxx = sum w (tx*tx + ty*ty), A = sum w a, B = sum w b,
 *     C = sum w (tx*a + ty*b), n = number of tracks with wt > 0 (sums as defined in the header);
 *     if not S0 > 0, or den = Sxx - (Sx*Sx + Sy*Sy)/S0 is not > 0: the vertex is dropped;
 *     zv = ((Sx*A + Sy*B)/S0 - C)/den; xv = (A + Sx*zv)/S0; yv = (B + Sy*zv)/S0
 *     (the weighted least-squares point of the tracks' straight lines).
 * P-6 a vertex is kept iff n >= min_tracks in the last iteration; output in seed order. */
uint32_t vn_pv_event(const float* st, size_t stride, uint32_t t0, uint32_t nt, const vn_pv_params_t* P, float* out) {
  const uint32_t nb = P->n_bins;
  const float inv_w = 1.0f / P->bin_width;
  uint32_t* h = (uint32_t*)calloc(nb ? nb : 1, sizeof(uint32_t));
  const float* X = st + 0 * stride + t0; const float* Y = st + 1 * stride + t0;
  const float* TX = st + 2 * stride + t0; const float* TY = st + 3 * stride + t0;
  const float* Z = st + 4 * stride + t0; const float* CXX = st + 5 * stride + t0;
  for (uint32_t i = 0; i < nt; ++i) {
    int32_t b = vn_pv_bin(Z[i], P->z_min, inv_w, nb);
    if (b >= 0) h[b] += 1u;
  }
  uint32_t seed_bins[VN_MAX_PV];
  const uint32_t ns = vn_pv_seeds(h, nb, P, seed_bins);
  free(h);
  if (ns == 0) return 0;
  float zs[VN_MAX_PV];
  for (uint32_t v = 0; v < ns; ++v) {
    float c = (float)seed_bins[v] + 0.5f;
    zs[v] = P->z_min + c * P->bin_width;
  }
  uint8_t* asg = (uint8_t*)malloc(nt ? nt : 1);
  for (uint32_t i = 0; i < nt; ++i) {
    uint32_t best = 0; float bd = fabsf(Z[i] - zs[0]);
    for (uint32_t v = 1; v < ns; ++v) {
      float dd = fabsf(Z[i] - zs[v]);
      if (dd < bd) { bd = dd; best = v; }
    }
    asg[i] = (uint8_t)best;
  }
  uint32_t nout = 0;
  for (uint32_t v = 0; v < ns; ++v) {
    float xv = 0.0f, yv = 0.0f, zv = zs[v], S0 = 0.0f;
    uint32_t ntrk = 0; int alive = 1;
    for (uint32_t it = 0; it < P->n_iterations && alive; ++it) {
      float l0[32], lx[32], ly[32], lxx[32], la[32], lb[32], lc[32], ln[32];
      for (int l = 0; l < 32; ++l) l0[l] = lx[l] = ly[l] = lxx[l] = la[l] = lb[l] = lc[l] = ln[l] = 0.0f;
      for (uint32_t i = 0; i < nt; ++i) {
        if (asg[i] != v) continue;
        const int l = (int)(i & 31u);
        float dz = zv - Z[i];
        float rx = (X[i] + TX[i] * dz) - xv;
        float ry = (Y[i] + TY[i] * dz) - yv;
        float w0 = 1.0f / CXX[i];
        float r2 = rx * rx;
        r2 = r2 + ry * ry;
        float c = w0 * r2;
        float wt = 0.0f;
        if (c < P->chi2_max) { float u = 1.0f - c / P->chi2_max; wt = u * u; }
        float w = w0 * wt;
        float a = X[i] - TX[i] * Z[i];
        float b = Y[i] - TY[i] * Z[i];
        float t2 = TX[i] * TX[i];
        t2 = t2 + TY[i] * TY[i];
        float ab = TX[i] * a;
        ab = ab + TY[i] * b;
        l0[l] = l0[l] + w;
        lx[l] = lx[l] + w * TX[i];
        ly[l] = ly[l] + w * TY[i];
        lxx[l] = lxx[l] + w * t2;
        la[l] = la[l] + w * a;
        lb[l] = lb[l] + w * b;
        lc[l] = lc[l] + w * ab;
        if (wt > 0.0f) ln[l] = ln[l] + 1.0f;
      }
      S0 = vn_butterfly(l0);
      const float Sx = vn_butterfly(lx), Sy = vn_butterfly(ly), Sxx = vn_butterfly(lxx);
      const float A = vn_butterfly(la), B = vn_butterfly(lb), C = vn_butterfly(lc);
      ntrk = (uint32_t)vn_butterfly(ln);           /* counts below 2^24 are exact in fp32 */
      if (!(S0 > 0.0f)) { alive = 0; break; }
      float q = Sx * Sx;
      q = q + Sy * Sy;
      float den = Sxx - q / S0;
      if (!(den > 0.0f)) { alive = 0; break; }
      float num = Sx * A;
      num = num + Sy * B;
      zv = (num / S0 - C) / den;
      xv = (A + Sx * zv) / S0;
      yv = (B + Sy * zv) / S0;
    }
    if (alive && ntrk >= P->min_tracks) {
      float* o = out + 5 * (size_t)nout;
      o[0] = xv; o[1] = yv; o[2] = zv; o[3] = S0;
      memcpy(&o[4], &ntrk, 4);
      ++nout;
    }
  }
  free(asg);
  return nout;
}

/* A batch: event_pv_offsets[n_events+1]; pvs = 5 planes of cap_pvs words. Returns the total number of
 * vertices (they are written only while they fit cap_pvs). */
uint32_t vn_pv_find(uint32_t n_events, const uint32_t* event_track_offsets, const float* states, size_t stride,
                    const vn_pv_params_t* P, uint32_t* event_pv_offsets, float* pvs, uint32_t cap_pvs) {
  uint32_t tot = 0;
  float tmp[5 * VN_MAX_PV];
  event_pv_offsets[0] = 0;
  for (uint32_t e = 0; e < n_events; ++e) {
    const uint32_t t0 = event_track_offsets[e], nt = event_track_offsets[e + 1] - t0;
    const uint32_t n = vn_pv_event(states, stride, t0, nt, P, tmp);
    for (uint32_t k = 0; k < n; ++k) {
      if (tot + k < cap_pvs)
        for (int p = 0; p < 5; ++p) pvs[(size_t)p * cap_pvs + tot + k] = tmp[5 * k + p];
    }
    tot += n;
    event_pv_offsets[e + 1] = tot;
  }
  return tot;
}
