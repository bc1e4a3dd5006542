/* velo_oracle.c — plain, slow, single-threaded CPU oracle for VELO track reconstruction.
 *
 * TEST INFRASTRUCTURE ONLY. This file is the parity oracle for the CUDA path: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call it. It shares no code, header, table or helper with paper_2412_05041_b200/csrc.
 *
 * What it computes: the data-parallel VELO hot path named by BASELINE.json:north_star —
 * per-module phi sort, search-by-triplet seeding, forwarding, ghost/clone filtering and a
 * straight-line least-squares fit to the state at closest approach to the beamline. The paper
 * names VELO tracks only as an input of forward tracking (§5) and says
 * HLT1 uses "a more simplified pattern recognition algorithm" and "simplified track fitting"
 * (§5); it gives no step, constant or formula. Every step below therefore follows
 * the reading fixed in SURVEY.md §8(c) (items O-1 ... O-17, ambiguity log A1 ... A23), restated
 * in DESIGN.md §2. The method is a heuristic, so the oracle IS the algorithm, written step by
 * step in that order and notation: no blocking, no fusion, windows by linear scan.
 *
 * Arithmetic: IEEE-754 binary32, round-to-nearest-even, one rounding per written operator, no
 * fused multiply-add. Build with: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math.
 *
 * Parity status versus the paper: UNPINNED (the paper prints no worked example or number for
 * this path). Pins are the SURVEY.md §8(c) vectors/checksum for phi16, closed forms, brute force
 * and invariants in tests/test_oracle_*.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define VO_MAX_MODULES 32

typedef struct {
  int32_t phi_window_seed, phi_window_fwd; /* phi16 units */
  float max_scatter_seed, max_scatter_fwd, max_scatter_weak; /* mm^2 */
  uint32_t max_skipped;
  float sigma_hit;
  float max_chi2_ndof;
  uint32_t clone_num, clone_den;
} vo_params_t;

/* ---- O-1: phi16(x, y) -> int16 --------------------------------------- */
int16_t vo_phi16(float x, float y) {
  const float C0 = 0x1.fffd04p-1f, C1 = -0x1.549b14p-2f, C2 = 0x1.8c5ee6p-3f;
  const float C3 = -0x1.dce202p-4f, C4 = 0x1.af4978p-5f, C5 = -0x1.80032cp-7f;
  const float K = 0x1.45f306p+13f;
  float ax = fabsf(x), ay = fabsf(y);
  float mx = ax > ay ? ax : ay;
  float mn = ax > ay ? ay : ax;
  if (mx == 0.0f) return 0;
  float t = mn / mx;
  float s = t * t;
  float p = C5;
  p = p * s; p = p + C4;
  p = p * s; p = p + C3;
  p = p * s; p = p + C2;
  p = p * s; p = p + C1;
  p = p * s; p = p + C0;
  float a = t * p;
  a = a * K;
  if (ay > ax) a = 16384.0f - a;
  if (x < 0.0f) a = 32768.0f - a;
  if (y < 0.0f) a = -a;
  int k = (int)floorf(a);
  return (int16_t)(((k + 32768) & 65535) - 32768);
}

/* ---- O-4: scatter(h0, h1, h2) ---------------------------------------- */
float vo_scatter(float x0, float y0, float z0, float x1, float y1, float z1, float x2, float y2,
                 float z2) {
  float tz = (z2 - z1) / (z1 - z0);
  float dx = x1 - x0;
  float dy = y1 - y0;
  float px = dx * tz;
  float py = dy * tz;
  float ex = (x1 + px) - x2;
  float ey = (y1 + py) - y2;
  float ex2 = ex * ex;
  float ey2 = ey * ey;
  return ex2 + ey2;
}

/* ---- O-3: modular phi window predicate ------------------------------- */
int vo_in_window(int16_t phi, int16_t c, int32_t W) {
  if (2 * (int64_t)W + 1 >= 65536) return 1;
  int d = (int)(int16_t)(uint16_t)((uint16_t)phi - (uint16_t)c);
  int ad = d < 0 ? -d : d;
  return ad <= W;
}

/* ---- O-2: per-event sort by (module, phi16, original index) -------------------------------- */
typedef struct { uint32_t module; int32_t phi; uint32_t idx; } vo_key_t;
static int vo_key_cmp(const void* a, const void* b) {
  const vo_key_t* p = (const vo_key_t*)a; const vo_key_t* q = (const vo_key_t*)b;
  if (p->module != q->module) return p->module < q->module ? -1 : 1;
  if (p->phi != q->phi) return p->phi < q->phi ? -1 : 1;
  if (p->idx != q->idx) return p->idx < q->idx ? -1 : 1;
  return 0;
}

/* perm[k] = original local index of the k-th sorted hit; phi[k] its phi16; mod_off[m] = first
 * sorted index of module m, mod_off[n_modules] = n. Returns 0, or -1 on a module id out of
 * range. */
int vo_sort_event(uint32_t n, const float* x, const float* y, const uint8_t* module,
                  uint32_t n_modules, uint32_t* perm, int16_t* phi, uint32_t* mod_off) {
  vo_key_t* k = (vo_key_t*)malloc(sizeof(vo_key_t) * (n ? n : 1));
  for (uint32_t i = 0; i < n; ++i) {
    if (module[i] >= n_modules) { free(k); return -1; }
    k[i].module = module[i]; k[i].phi = vo_phi16(x[i], y[i]); k[i].idx = i;
  }
  qsort(k, n, sizeof(vo_key_t), vo_key_cmp);
  for (uint32_t i = 0; i < n; ++i) { perm[i] = k[i].idx; phi[i] = (int16_t)k[i].phi; }
  /* mod_off[m] = number of hits in modules < m */
  for (uint32_t m = 0; m <= n_modules; ++m) {
    uint32_t c = 0;
    for (uint32_t i = 0; i < n; ++i) if (module[i] < m) ++c;
    mod_off[m] = c;
  }
  free(k);
  return 0;
}

/* ---- O-11: straight-line least-squares fit -------------------------- */
/* out[13]: x, y, tx, ty, z, cxx, cxtx, ctxtx, cyy, cyty, ctyty, chi2, n (as float bits of u32) */
void vo_fit(uint32_t n, const float* hx, const float* hy, const float* hz, float sigma_hit,
            float* out) {
  float sz = 0.0f, sx = 0.0f, sy = 0.0f;
  for (uint32_t i = 0; i < n; ++i) { sz = sz + hz[i]; sx = sx + hx[i]; sy = sy + hy[i]; }
  float nf = (float)n;
  float zb = sz / nf, xb = sx / nf, yb = sy / nf;
  float sdd = 0.0f, sdx = 0.0f, sdy = 0.0f;
  for (uint32_t i = 0; i < n; ++i) {
    float d = hz[i] - zb;
    float dd = d * d; sdd = sdd + dd;
    float ux = hx[i] - xb; float dx = d * ux; sdx = sdx + dx;
    float uy = hy[i] - yb; float dy = d * uy; sdy = sdy + dy;
  }
  float tx = sdx / sdd, ty = sdy / sdd;
  float c = 0.0f;
  for (uint32_t i = 0; i < n; ++i) {
    float d = hz[i] - zb;
    float ux = hx[i] - xb; float txd = tx * d; float rx = ux - txd;
    float uy = hy[i] - yb; float tyd = ty * d; float ry = uy - tyd;
    float rx2 = rx * rx; c = c + rx2;
    float ry2 = ry * ry; c = c + ry2;
  }
  float sig2 = sigma_hit * sigma_hit;
  float inv_s2 = 1.0f / sig2;
  float chi2 = c * inv_s2;
  float txx = tx * tx, tyy = ty * ty;
  float s2 = txx + tyy;
  float dzb;
  if (s2 < 1e-12f) {
    dzb = 0.0f;
  } else {
    float a = xb * tx, b = yb * ty;
    float num = a + b;
    dzb = -(num / s2);
  }
  float z = zb + dzb;
  float txdz = tx * dzb, tydz = ty * dzb;
  float x = xb + txdz, y = yb + tydz;
  float vt = sig2 / sdd;
  float cxtx = dzb * vt;
  float v0 = sig2 / nf;
  float dz2 = dzb * dzb;
  float v1 = dz2 * vt;
  float cxx = v0 + v1;
  out[0] = x; out[1] = y; out[2] = tx; out[3] = ty; out[4] = z;
  out[5] = cxx; out[6] = cxtx; out[7] = vt;
  out[8] = cxx; out[9] = cxtx; out[10] = vt;
  out[11] = chi2;
  uint32_t nn = n; memcpy(&out[12], &nn, 4);
}

/* ---- O-5 ... O-14: one event --------------------------------------------------------------- */
typedef struct {
  uint32_t hits[VO_MAX_MODULES]; /* sorted indices, discovery order (decreasing module) */
  uint32_t n, n_missed, active;
  float seed_scatter;
  uint32_t centre; /* sorted index of the seed's h1 */
  /* filled after the module loop */
  uint32_t pass;   /* survived O-10 and O-12 */
  float state[13];
  uint64_t key;    /* O-13 */
  uint32_t lost, survive;
} vo_cand_t;

typedef struct {
  uint32_t n;                /* hits in the event */
  uint32_t* perm; int16_t* phi; float *sx, *sy, *sz; uint8_t* flag;
  uint32_t mod_off[VO_MAX_MODULES + 1];
  vo_cand_t* cand; uint32_t n_cand, cap_cand;
} vo_event_t;

static void vo_event_free(vo_event_t* ev) {
  free(ev->perm); free(ev->phi); free(ev->sx); free(ev->sy); free(ev->sz); free(ev->flag);
  free(ev->cand);
}

static vo_cand_t* vo_new_cand(vo_event_t* ev) {
  if (ev->n_cand == ev->cap_cand) {
    ev->cap_cand = ev->cap_cand ? 2 * ev->cap_cand : 64;
    ev->cand = (vo_cand_t*)realloc(ev->cand, sizeof(vo_cand_t) * ev->cap_cand);
  }
  vo_cand_t* c = &ev->cand[ev->n_cand++];
  memset(c, 0, sizeof(*c));
  return c;
}

static float vo_scatter_idx(const vo_event_t* ev, uint32_t a, uint32_t b, uint32_t c) {
  return vo_scatter(ev->sx[a], ev->sy[a], ev->sz[a], ev->sx[b], ev->sy[b], ev->sz[b], ev->sx[c],
                    ev->sy[c], ev->sz[c]);
}

/* Runs O-2 and O-5 ... O-13 on one event. Returns 0 or -1 (module id out of range). */
static int vo_run_event(vo_event_t* ev, uint32_t n, const float* x, const float* y, const float* z,
                        const uint8_t* module, uint32_t M, const vo_params_t* P) {
  memset(ev, 0, sizeof(*ev));
  ev->n = n;
  uint32_t na = n ? n : 1;
  ev->perm = (uint32_t*)malloc(4 * na); ev->phi = (int16_t*)malloc(2 * na);
  ev->sx = (float*)malloc(4 * na); ev->sy = (float*)malloc(4 * na); ev->sz = (float*)malloc(4 * na);
  ev->flag = (uint8_t*)calloc(na, 1);
  if (vo_sort_event(n, x, y, module, M, ev->perm, ev->phi, ev->mod_off) != 0) return -1;
  for (uint32_t k = 0; k < n; ++k) {
    ev->sx[k] = x[ev->perm[k]]; ev->sy[k] = y[ev->perm[k]]; ev->sz[k] = z[ev->perm[k]];
  }
  uint8_t* mark = (uint8_t*)calloc(na, 1);

  /* O-6: module loop, s = M-2 down to 1 */
  for (uint32_t s = M - 2; s >= 1; --s) {
    /* (A) forwarding into module u = s-1, for all tracks active at the start of the step (O-7) */
    const uint32_t u = s - 1;
    const uint32_t n_start = ev->n_cand;
    for (uint32_t t = 0; t < n_start; ++t) {
      vo_cand_t* T = &ev->cand[t];
      if (!T->active) continue;
      const uint32_t ha = T->hits[T->n - 2], hb = T->hits[T->n - 1];
      int found = 0; uint32_t best = 0; float best_sc = 0.0f;
      for (uint32_t c = ev->mod_off[u]; c < ev->mod_off[u + 1]; ++c) { /* sorted-index order */
        if (!vo_in_window(ev->phi[c], ev->phi[hb], P->phi_window_fwd)) continue; /* flags ignored */
        float sc = vo_scatter_idx(ev, ha, hb, c);
        if (!(sc <= P->max_scatter_fwd)) continue;
        if (!found || sc < best_sc) { found = 1; best = c; best_sc = sc; } /* tie -> lowest index */
      }
      if (found) {
        T->hits[T->n++] = best; T->n_missed = 0;
        if (T->n >= 4) for (uint32_t i = 0; i < T->n; ++i) mark[T->hits[i]] = 1;
      } else {
        T->n_missed += 1;
        if (T->n_missed > P->max_skipped) T->active = 0;
      }
    }
    /* (B) apply the flags produced in (A) */
    for (uint32_t k = 0; k < n; ++k) if (mark[k]) ev->flag[k] = 1;
    /* (C) seeding with centre module s (O-8); sets no flags */
    for (uint32_t h1 = ev->mod_off[s]; h1 < ev->mod_off[s + 1]; ++h1) {
      if (ev->flag[h1]) continue;
      int found = 0; uint32_t b0 = 0, b2 = 0; float best_sc = 0.0f;
      for (uint32_t h0 = ev->mod_off[s + 1]; h0 < ev->mod_off[s + 2]; ++h0) {
        if (ev->flag[h0] || !vo_in_window(ev->phi[h0], ev->phi[h1], P->phi_window_seed)) continue;
        for (uint32_t h2 = ev->mod_off[s - 1]; h2 < ev->mod_off[s]; ++h2) {
          if (ev->flag[h2] || !vo_in_window(ev->phi[h2], ev->phi[h1], P->phi_window_seed)) continue;
          float sc = vo_scatter_idx(ev, h0, h1, h2);
          if (!(sc <= P->max_scatter_seed)) continue;
          /* minimum under (sc, h0, h2); loops ascend in h0 then h2, so strict < keeps the first */
          if (!found || sc < best_sc) { found = 1; b0 = h0; b2 = h2; best_sc = sc; }
        }
      }
      if (found) {
        vo_cand_t* T = vo_new_cand(ev);
        T->hits[0] = b0; T->hits[1] = h1; T->hits[2] = b2; T->n = 3; T->n_missed = 0;
        T->active = 1; T->seed_scatter = best_sc; T->centre = h1;
      }
    }
  }
  free(mark);
  /* O-9 */
  for (uint32_t t = 0; t < ev->n_cand; ++t) ev->cand[t].active = 0;

  /* O-10, O-11, O-12 */
  for (uint32_t t = 0; t < ev->n_cand; ++t) {
    vo_cand_t* T = &ev->cand[t];
    T->pass = 1;
    if (T->n == 3) {
      if (ev->flag[T->hits[0]] || ev->flag[T->hits[1]] || ev->flag[T->hits[2]]) T->pass = 0;
      if (!(T->seed_scatter <= P->max_scatter_weak)) T->pass = 0;
    }
    if (!T->pass) continue;
    float hx[VO_MAX_MODULES], hy[VO_MAX_MODULES], hz[VO_MAX_MODULES];
    for (uint32_t i = 0; i < T->n; ++i) {
      hx[i] = ev->sx[T->hits[i]]; hy[i] = ev->sy[T->hits[i]]; hz[i] = ev->sz[T->hits[i]];
    }
    vo_fit(T->n, hx, hy, hz, P->sigma_hit, T->state);
    float ndof = (float)(2 * (int)T->n - 4);
    float lim = P->max_chi2_ndof * ndof;
    if (T->state[11] > lim) T->pass = 0; /* O-12 */
  }

  /* O-13 clone filter */
  uint64_t* owner = (uint64_t*)malloc(8 * na);
  for (uint32_t k = 0; k < n; ++k) owner[k] = ~(uint64_t)0;
  for (uint32_t t = 0; t < ev->n_cand; ++t) {
    vo_cand_t* T = &ev->cand[t];
    if (!T->pass) continue;
    uint32_t bits; memcpy(&bits, &T->state[11], 4);
    T->key = ((uint64_t)(255u - T->n) << 56) | ((uint64_t)bits << 24) | (uint64_t)T->centre;
    for (uint32_t i = 0; i < T->n; ++i)
      if (T->key < owner[T->hits[i]]) owner[T->hits[i]] = T->key;
  }
  for (uint32_t t = 0; t < ev->n_cand; ++t) {
    vo_cand_t* T = &ev->cand[t];
    T->survive = 0; T->lost = 0;
    if (!T->pass) continue;
    for (uint32_t i = 0; i < T->n; ++i) if (owner[T->hits[i]] != T->key) T->lost += 1;
    T->survive = !((uint64_t)T->lost * P->clone_den > (uint64_t)T->n * P->clone_num);
  }
  free(owner);
  return 0;
}

/* ---- whole batch (O-14) -------------------------------------------------------------------- */
typedef struct {
  uint32_t n_events, n_tracks, n_track_hits, n_candidates;
  uint32_t* event_track_offsets; /* n_events+1 */
  uint32_t* track_hit_offsets;   /* n_tracks+1 */
  uint32_t* track_hits;          /* n_track_hits, GLOBAL original hit indices */
  float* states;                 /* 13 planes x n_tracks */
  int status;
} vo_result_t;

void vo_result_free(vo_result_t* r) {
  if (!r) return;
  free(r->event_track_offsets); free(r->track_hit_offsets); free(r->track_hits); free(r->states);
  free(r);
}

/* Reconstruct events [0, n_events). All pointers are HOST pointers. Tracks of an event are
 * emitted in candidate-creation order (step descending, then sorted index of the centre hit).
 * status: 0 ok, -6 bad input (module id >= n_modules, non-monotone offsets, event too large). */
vo_result_t* vo_reconstruct(uint32_t n_modules, const float* x, const float* y, const float* z,
                            const uint8_t* module, const uint32_t* event_offsets, uint32_t n_events,
                            const vo_params_t* P) {
  vo_result_t* r = (vo_result_t*)calloc(1, sizeof(vo_result_t));
  r->n_events = n_events;
  r->event_track_offsets = (uint32_t*)calloc((size_t)n_events + 1, 4);
  size_t cap_t = 1024, cap_h = 8192;
  uint32_t* tho = (uint32_t*)malloc(4 * (cap_t + 1));
  uint32_t* th = (uint32_t*)malloc(4 * cap_h);
  float* st = (float*)malloc(4 * 13 * cap_t); /* [track][13] while growing */
  tho[0] = 0;
  if (n_modules < 3 || n_modules > VO_MAX_MODULES) r->status = -2;
  for (uint32_t e = 0; e < n_events && r->status == 0; ++e) {
    uint32_t o0 = event_offsets[e], o1 = event_offsets[e + 1];
    if (o1 < o0 || (o1 - o0) >= (1u << 24)) { r->status = -6; break; }
    vo_event_t ev;
    if (vo_run_event(&ev, o1 - o0, x + o0, y + o0, z + o0, module + o0, n_modules, P) != 0) {
      r->status = -6; vo_event_free(&ev); break;
    }
    r->n_candidates += ev.n_cand;
    for (uint32_t t = 0; t < ev.n_cand; ++t) {
      const vo_cand_t* T = &ev.cand[t];
      if (!T->survive) continue;
      if (r->n_tracks + 1 > cap_t) {
        cap_t *= 2; tho = (uint32_t*)realloc(tho, 4 * (cap_t + 1)); st = (float*)realloc(st, 4 * 13 * cap_t);
      }
      if (r->n_track_hits + T->n > cap_h) { cap_h *= 2; th = (uint32_t*)realloc(th, 4 * cap_h); }
      for (uint32_t i = 0; i < T->n; ++i) th[r->n_track_hits + i] = o0 + ev.perm[T->hits[i]];
      memcpy(st + 13 * (size_t)r->n_tracks, T->state, 13 * 4);
      r->n_track_hits += T->n;
      r->n_tracks += 1;
      tho[r->n_tracks] = r->n_track_hits;
    }
    r->event_track_offsets[e + 1] = r->n_tracks;
    vo_event_free(&ev);
  }
  r->track_hit_offsets = tho; r->track_hits = th;
  r->states = (float*)malloc(4 * 13 * (size_t)(r->n_tracks ? r->n_tracks : 1));
  for (uint32_t t = 0; t < r->n_tracks; ++t)
    for (int k = 0; k < 13; ++k) r->states[(size_t)k * r->n_tracks + t] = st[13 * (size_t)t + k];
  free(st);
  return r;
}

/* accessors for ctypes */
void vo_result_sizes(const vo_result_t* r, uint32_t* out4) {
  out4[0] = r->n_tracks; out4[1] = r->n_track_hits; out4[2] = (uint32_t)r->status; out4[3] = r->n_candidates;
}
void vo_result_copy(const vo_result_t* r, uint32_t* eto, uint32_t* tho, uint32_t* th, float* states) {
  memcpy(eto, r->event_track_offsets, 4 * ((size_t)r->n_events + 1));
  memcpy(tho, r->track_hit_offsets, 4 * ((size_t)r->n_tracks + 1));
  memcpy(th, r->track_hits, 4 * (size_t)r->n_track_hits);
  memcpy(states, r->states, 4 * 13 * (size_t)r->n_tracks);
}

/* ---- single-event candidate dump, for the brute-force pins in tests/ ----------------------- */
/* Writes up to cap candidates: hits (cap x 32 sorted indices), meta (cap x 8 u32: n, centre, pass,
 * survive, lost, key_lo, key_hi, bits(seed_scatter)), states (cap x 13), plus the sort (perm, phi,
 * mod_off[n_modules+1]) and final flags. Returns the number of candidates, or -1. */
int vo_event_candidates(uint32_t n, const float* x, const float* y, const float* z, const uint8_t* module,
                        uint32_t n_modules, const vo_params_t* P, uint32_t cap, uint32_t* hits,
                        uint32_t* meta, float* states, uint32_t* perm, int16_t* phi, uint32_t* mod_off,
                        uint8_t* flags) {
  vo_event_t ev;
  if (n_modules < 3 || n_modules > VO_MAX_MODULES) return -1;
  if (vo_run_event(&ev, n, x, y, z, module, n_modules, P) != 0) { vo_event_free(&ev); return -1; }
  for (uint32_t t = 0; t < ev.n_cand && t < cap; ++t) {
    const vo_cand_t* T = &ev.cand[t];
    memcpy(hits + 32 * (size_t)t, T->hits, 32 * 4);
    uint32_t* m = meta + 8 * (size_t)t;
    m[0] = T->n; m[1] = T->centre; m[2] = T->pass; m[3] = T->survive; m[4] = T->lost;
    m[5] = (uint32_t)(T->key & 0xffffffffu); m[6] = (uint32_t)(T->key >> 32);
    memcpy(&m[7], &T->seed_scatter, 4);
    memcpy(states + 13 * (size_t)t, T->state, 13 * 4);
  }
  memcpy(perm, ev.perm, 4 * (size_t)n); memcpy(phi, ev.phi, 2 * (size_t)n);
  memcpy(mod_off, ev.mod_off, 4 * ((size_t)n_modules + 1)); memcpy(flags, ev.flag, n);
  int nc = (int)ev.n_cand;
  vo_event_free(&ev);
  return nc;
}
