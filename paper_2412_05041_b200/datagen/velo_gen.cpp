// Synthetic VELO event generator (host, multi-threaded over events).
//
// Stands in for the LHCb collision data the paper's plots use, which are not
// available. Recipe: BASELINE.json:configs[0..4], restated in SURVEY.md §8(d) and DESIGN.md §4.
// This module holds NONE of the reconstruction method's arithmetic (no phi16, no scatter, no
// fit): it only writes the input arrays (x, y, z fp32 planes, module u8, event offsets u32)
// that both the CPU oracle and the CUDA path consume, plus generator truth for sanity tests.
//
// Event e's random stream depends only on (seed, e): never on n_events, batch boundaries or the
// thread count, so configs[0] is the first 100 events of configs[1].
//
// Coordinate system: origin at the nominal interaction point, z along the beam, y up
// (§2). Acceptance 2 < eta < 5 (§2). Pile-up mu = 5 (§1).
// Open geometry: halves displaced by +-24.5 mm in x = 49 mm opening (§2).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <unordered_set>
#include <vector>

extern "C" {

typedef struct {
  uint64_t seed;
  uint32_t n_modules;     // <= 32
  int32_t ion_mode;       // 0: Poisson(mu) vertices x Poisson(trk_mean) tracks; 1: one vertex,
                          //    multiplicity floor(exp(U(ln mult_lo, ln mult_hi)))
  double r_in, r_out, pitch, half_shift_x;
  double mu, trk_mean, mult_lo, mult_hi;
  double eta_lo, eta_hi;
  double sigma_vxy, sigma_vz;
  double hit_eff, noise_frac, ms_sigma;
  int32_t quantise;       // 1: snap to pixel centres and merge same-pixel hits (A19)
  int32_t shuffle;        // 1: Fisher-Yates shuffle of the event's hits (A16)
  double backward_frac;   // fraction of tracks that leave the vertex towards -z (eta -> -eta; A23); 0 in BASELINE's configs
  double stagger_z;       // 52-sensor layout: the -x sensor of a station sits at z - stagger_z/2, the +x one at z + stagger_z/2
  double overlap_x;       // ... and both reach this far over the x = 0 line (a track in the strip crosses both); 0, 0 in BASELINE's configs
} velogen_config_t;

}  // extern "C"

namespace {

struct Rng {
  uint64_t s;
  bool has_spare = false;
  double spare = 0.0;
  static uint64_t mix(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
  }
  Rng(uint64_t seed, uint64_t event) {
    s = mix(seed + 0x9E3779B97F4A7C15ULL) ^ mix(event * 0xD1342543DE82EF95ULL + 0x632BE59BD9B4E019ULL);
  }
  uint64_t next() {
    s += 0x9E3779B97F4A7C15ULL;
    return mix(s);
  }
  double uniform() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }  // [0,1)
  double normal() {  // Box-Muller, pairs cached
    if (has_spare) { has_spare = false; return spare; }
    double u1 = 1.0 - uniform();  // (0,1]
    double u2 = uniform();
    double r = std::sqrt(-2.0 * std::log(u1));
    double a = 6.283185307179586476925 * u2;
    spare = r * std::sin(a);
    has_spare = true;
    return r * std::cos(a);
  }
  uint32_t poisson(double lam) {  // CDF inversion; lam <= ~100
    if (lam <= 0.0) return 0;
    double p = std::exp(-lam), c = p, u = uniform();
    uint32_t k = 0;
    while (u > c && k < 100000u) { ++k; p *= lam / (double)k; c += p; if (p < 1e-300) break; }
    return k;
  }
  uint32_t below(uint32_t n) { return (uint32_t)(uniform() * (double)n); }  // [0,n)
};

struct Hit { float x, y, z; uint8_t module; int32_t track; uint32_t pixel; };
struct Trk { double xv, yv, zv, tx, ty; };

struct EventBuf {
  std::vector<Hit> hits;
  std::vector<Trk> trks;
  std::unordered_set<uint64_t> pixels;
};

inline uint64_t pixel_key(uint32_t m, int h, long ix, long iy) {
  return ((uint64_t)m << 58) | ((uint64_t)(h > 0) << 57) | ((uint64_t)((ix + (1L << 27)) & 0xFFFFFFF) << 28) |
         (uint64_t)((iy + (1L << 27)) & 0xFFFFFFF);
}

// Record one crossing (local coordinates xl, y in half h of module m). Returns true if a new
// hit was stored (false: pixel already hit, A19).
bool record(const velogen_config_t& c, const double* mz, EventBuf& b, uint32_t m, int h, double xl, double y,
            int32_t track, double z_sensor = 1e300) {
  double xo = xl, yo = y;
  if (c.quantise) {
    long ix = (long)std::floor(xl / c.pitch), iy = (long)std::floor(y / c.pitch);
    if (!b.pixels.insert(pixel_key(m, h, ix, iy)).second) return false;
    xo = ((double)ix + 0.5) * c.pitch;
    yo = ((double)iy + 0.5) * c.pitch;
  }
  Hit hit;
  hit.pixel = 0xffffffffu;
  if (c.quantise) {
    // the detector's packed pixel address (include/velo.h, velo_pixel_hits_t): column and row biased
    // by 1024, half bit, module
    long ix = (long)std::floor(xl / c.pitch), iy = (long)std::floor(y / c.pitch);
    if (ix >= -1024 && ix < 1024 && iy >= -1024 && iy < 1024)
      hit.pixel = (uint32_t)(ix + 1024) | ((uint32_t)(iy + 1024) << 11) | ((uint32_t)(h > 0) << 22) | (m << 23);
  }
  hit.x = (float)(xo + (double)h * c.half_shift_x);
  hit.y = (float)yo;
  hit.z = (float)(z_sensor < 1e299 ? z_sensor : mz[m]);
  hit.module = (uint8_t)m;
  hit.track = track;
  b.hits.push_back(hit);
  return true;
}

void gen_event(const velogen_config_t& c, const double* mz, uint64_t e, EventBuf& b) {
  b.hits.clear(); b.trks.clear(); b.pixels.clear();
  Rng rng(c.seed, e);
  const uint32_t M = c.n_modules;
  uint32_t n_pv = c.ion_mode ? 1u : rng.poisson(c.mu);
  uint32_t signal_on_module[32];
  for (uint32_t m = 0; m < 32; ++m) signal_on_module[m] = 0;
  for (uint32_t v = 0; v < n_pv; ++v) {
    double xv = c.sigma_vxy * rng.normal();
    double yv = c.sigma_vxy * rng.normal();
    double zv = c.sigma_vz * rng.normal();
    uint32_t n_trk;
    if (c.ion_mode) {
      double lu = std::log(c.mult_lo) + rng.uniform() * (std::log(c.mult_hi) - std::log(c.mult_lo));
      n_trk = (uint32_t)std::floor(std::exp(lu));
    } else {
      n_trk = rng.poisson(c.trk_mean);
    }
    for (uint32_t t = 0; t < n_trk; ++t) {
      double eta = c.eta_lo + rng.uniform() * (c.eta_hi - c.eta_lo);
      double phi = 6.283185307179586476925 * rng.uniform();
      double theta = 2.0 * std::atan(std::exp(-eta));
      double tt = std::tan(theta);
      double tx = tt * std::cos(phi), ty = tt * std::sin(phi);
      int32_t tid = (int32_t)b.trks.size();
      b.trks.push_back(Trk{xv, yv, zv, tx, ty});
      double x = xv, y = yv, zp = zv;
      // a backward track crosses the modules below the vertex, nearest first (no extra random number
      // is drawn when backward_frac is 0, so BASELINE's configs are unchanged)
      const bool back = c.backward_frac > 0.0 && rng.uniform() < c.backward_frac;
      const bool sensors52 = c.stagger_z != 0.0 || c.overlap_x != 0.0;
      for (uint32_t mm = 0; sensors52 && mm < M; ++mm) {
        // 52-sensor layout: the two sensors of a station are planes of their own, crossed in z order;
        // a track inside the overlap strip leaves a hit on both
        const uint32_t m = back ? M - 1 - mm : mm;
        for (int hh = 0; hh < 2; ++hh) {
          const int h = (back ? (hh == 0) : (hh != 0)) ? 1 : -1;       // forward: -x sensor (lower z) first
          const double zs = mz[m] + 0.5 * (double)h * c.stagger_z;
          if (back ? !(zs < zv) : !(zs > zv)) continue;
          x += tx * (zs - zp);
          y += ty * (zs - zp);
          zp = zs;
          const double xl = x - (double)h * c.half_shift_x;
          const bool in_half = (h < 0) ? (xl < c.overlap_x) : (xl >= -c.overlap_x);
          if (!in_half) continue;
          const double r = std::sqrt(xl * xl + y * y);
          if (r < c.r_in || r > c.r_out) continue;
          if (rng.uniform() < c.hit_eff) {
            if (record(c, mz, b, m, h, xl, y, tid, zs)) signal_on_module[m]++;
          }
          if (c.ms_sigma > 0.0) {
            tx += c.ms_sigma * rng.normal();
            ty += c.ms_sigma * rng.normal();
          }
        }
      }
      for (uint32_t mm = 0; !sensors52 && mm < M; ++mm) {
        const uint32_t m = back ? M - 1 - mm : mm;
        if (back ? !(mz[m] < zv) : !(mz[m] > zv)) continue;
        x += tx * (mz[m] - zp);
        y += ty * (mz[m] - zp);
        zp = mz[m];
        for (int h = -1; h <= 1; h += 2) {
          double xl = x - (double)h * c.half_shift_x;
          bool in_half = (h < 0) ? (xl < 0.0) : (xl >= 0.0);
          if (!in_half) continue;
          double r = std::sqrt(xl * xl + y * y);
          if (r < c.r_in || r > c.r_out) continue;
          if (rng.uniform() < c.hit_eff) {
            if (record(c, mz, b, m, h, xl, y, tid)) signal_on_module[m]++;
          }
          if (c.ms_sigma > 0.0) {  // A18: kick after every crossed active area, recorded or not
            tx += c.ms_sigma * rng.normal();
            ty += c.ms_sigma * rng.normal();
          }
          break;
        }
      }
    }
  }
  if (c.noise_frac > 0.0) {  // A17: Poisson(noise_frac x signal hits on that module), uniform in area
    for (uint32_t m = 0; m < M; ++m) {
      uint32_t nn = rng.poisson(c.noise_frac * (double)signal_on_module[m]);
      for (uint32_t k = 0; k < nn; ++k) {
        double r = std::sqrt(c.r_in * c.r_in + rng.uniform() * (c.r_out * c.r_out - c.r_in * c.r_in));
        double a = 6.283185307179586476925 * rng.uniform();
        double xl = r * std::cos(a), y = r * std::sin(a);
        int h = (xl < 0.0) ? -1 : 1;
        record(c, mz, b, m, h, xl, y, -1, (c.stagger_z != 0.0) ? mz[m] + 0.5 * (double)h * c.stagger_z : 1e300);
      }
    }
  }
  if (c.shuffle) {
    for (uint32_t i = (uint32_t)b.hits.size(); i > 1; --i) {
      uint32_t j = rng.below(i);
      std::swap(b.hits[i - 1], b.hits[j]);
    }
  }
}

template <class F>
void parallel_events(uint32_t n, int nthreads, F f) {
  if (nthreads < 1) nthreads = 1;
  if ((uint32_t)nthreads > n) nthreads = n ? (int)n : 1;
  std::vector<std::thread> th;
  const uint32_t chunk = 64;
  // static interleaved chunks: deterministic output regardless of scheduling (each event
  // writes only its own slots)
  for (int t = 0; t < nthreads; ++t) {
    th.emplace_back([=]() {
      EventBuf buf;
      for (uint32_t c0 = (uint32_t)t * chunk; c0 < n; c0 += (uint32_t)nthreads * chunk)
        for (uint32_t i = c0; i < std::min(n, c0 + chunk); ++i) f(i, buf);
    });
  }
  for (auto& x : th) x.join();
}

}  // namespace

extern "C" {

// Pass 1: per-event hit and generated-track counts for events [e0, e0+n).
int velogen_count(const velogen_config_t* cfg, const double* module_z, uint64_t e0, uint32_t n,
                  uint32_t* n_hits, uint32_t* n_trks, int nthreads) {
  if (!cfg || !module_z || cfg->n_modules < 1 || cfg->n_modules > 32) return -1;
  velogen_config_t c = *cfg;
  parallel_events(n, nthreads, [&, c](uint32_t i, EventBuf& b) {
    gen_event(c, module_z, e0 + i, b);
    n_hits[i] = (uint32_t)b.hits.size();
    n_trks[i] = (uint32_t)b.trks.size();
  });
  return 0;
}

// Pass 2: regenerate and write into caller arrays at the given exclusive-scan offsets.
// hit_track: index into this call's truth-track table (trk_off[i] + local id) or -1 for noise.
// trk_truth: 5 doubles per generated track (xv, yv, zv, tx, ty at the vertex).
int velogen_fill(const velogen_config_t* cfg, const double* module_z, uint64_t e0, uint32_t n,
                 const uint32_t* hit_off, const uint32_t* trk_off, float* x, float* y, float* z,
                 uint8_t* module, int32_t* hit_track, double* trk_truth, int nthreads) {
  if (!cfg || !module_z || cfg->n_modules < 1 || cfg->n_modules > 32) return -1;
  velogen_config_t c = *cfg;
  std::vector<int> bad((size_t)std::max(nthreads, 1) + 1, 0);
  int* badp = bad.data();
  parallel_events(n, nthreads, [&, c, badp](uint32_t i, EventBuf& b) {
    gen_event(c, module_z, e0 + i, b);
    if (b.hits.size() != (size_t)(hit_off[i + 1] - hit_off[i]) ||
        b.trks.size() != (size_t)(trk_off[i + 1] - trk_off[i])) { badp[0] = 1; return; }
    uint32_t o = hit_off[i];
    for (size_t k = 0; k < b.hits.size(); ++k) {
      x[o + k] = b.hits[k].x; y[o + k] = b.hits[k].y; z[o + k] = b.hits[k].z;
      module[o + k] = b.hits[k].module;
      if (hit_track) hit_track[o + k] = b.hits[k].track < 0 ? -1 : (int32_t)(trk_off[i] + (uint32_t)b.hits[k].track);
    }
    if (trk_truth) {
      double* t = trk_truth + 5 * (size_t)trk_off[i];
      for (size_t k = 0; k < b.trks.size(); ++k) {
        t[5 * k + 0] = b.trks[k].xv; t[5 * k + 1] = b.trks[k].yv; t[5 * k + 2] = b.trks[k].zv;
        t[5 * k + 3] = b.trks[k].tx; t[5 * k + 4] = b.trks[k].ty;
      }
    }
  });
  return bad[0] ? -2 : 0;
}

// The same events as packed pixel addresses (one u32 per hit, same order as velogen_fill's arrays).
// Needs cfg->quantise; returns -3 if a hit has no pixel address.
int velogen_pixels(const velogen_config_t* cfg, const double* module_z, uint64_t e0, uint32_t n,
                   const uint32_t* hit_off, uint32_t* pixel, int nthreads) {
  if (!cfg || !module_z || cfg->n_modules < 1 || cfg->n_modules > 32) return -1;
  velogen_config_t c = *cfg;
  std::vector<int> bad(2, 0);
  int* badp = bad.data();
  parallel_events(n, nthreads, [&, c, badp](uint32_t i, EventBuf& b) {
    gen_event(c, module_z, e0 + i, b);
    if (b.hits.size() != (size_t)(hit_off[i + 1] - hit_off[i])) { badp[0] = 1; return; }
    const uint32_t o = hit_off[i];
    for (size_t k = 0; k < b.hits.size(); ++k) {
      pixel[o + k] = b.hits[k].pixel;
      if (b.hits[k].pixel == 0xffffffffu) badp[1] = 1;
    }
  });
  return bad[0] ? -2 : (bad[1] ? -3 : 0);
}

}  // extern "C"
