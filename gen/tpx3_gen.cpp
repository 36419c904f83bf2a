// Seeded synthetic TimePix3 workload generator (BASELINE.json configs 0-4).
//
// This module is shared by the oracle, the tests and the CUDA path. It holds NONE of the
// method's arithmetic (no sorting by (shot, ToA) for the method, no linking, no centroid):
// it only draws pixel events (x, y, ToA, ToT) with the shapes, sizes and value
// distributions of the paper's workloads (PAPER.md:38 "up to 50 particles/shot", :42 the
// four event fields, :68 the 100 us ToF cut, :150 ToT quantum of 25 ns).
//
// RNG: stateless 64-bit mixing hash of (seed, shot, particle, pixel, field); uniforms from
// the top 53 bits; normals by Box-Muller in fp64. The data are generated ONCE on the host
// and the same arrays feed both sides, so libm differences never matter.
//
// Recipe per particle:
//   centre c (fp64), size k, width sigma, amplitude a, arrival tick t0
//   footprint = the k integer pixels nearest c, ordered by (r^2, y, x)
//   ToT = clip(floor(a*exp(-r^2/(2 sigma^2)) + 5*N(0,1) + 0.5), 1, 1023)        [25 ns units]
//   ToA = shot*P + t0 + U{0..30}                                             [1.5625 ns ticks]
// Each shot is delivered stably sorted by ToA (configs 0-3, 5) or locally shuffled
// (config 4: stable sort on pos + U{0..2047}).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr uint64_t kShotPeriod = 640000;  // ticks, 1 kHz at 1.5625 ns
constexpr double kTwoPi = 6.283185307179586476925286766559;

inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// Field ids (per particle unless noted).
enum Field : uint64_t {
  F_K = 1, F_CX, F_CY, F_CN1, F_CN2, F_AMP, F_ARR, F_ARR2, F_PEAK, F_PAIR, F_PAIR_D, F_PAIR_TH,
  F_PAIR_DT, F_NOISE_X, F_NOISE_Y, F_NOISE_T, F_NOISE_TOT, F_SHUF,
  F_PIX_TW = 64, F_PIX_N1, F_PIX_N2
};

struct Rng {
  uint64_t hs;  // hash of (seed, shot)
  Rng(uint64_t seed, uint64_t shot) { hs = mix64(mix64(seed) ^ (shot * 0xD1342543DE82EF95ull)); }
  inline uint64_t raw(uint64_t particle, uint64_t pixel, uint64_t field, uint64_t attempt = 0) const {
    uint64_t h = mix64(hs ^ ((particle + 1) * 0xA24BAED4963EE407ull));
    h = mix64(h ^ ((pixel + 1) * 0x9FB21C651E98DF25ull));
    return mix64(h ^ (field + (attempt << 16)));
  }
  inline double u01(uint64_t p, uint64_t px, uint64_t f, uint64_t a = 0) const {  // [0,1)
    return (double)(raw(p, px, f, a) >> 11) * (1.0 / 9007199254740992.0);
  }
  inline double u01_open(uint64_t p, uint64_t px, uint64_t f, uint64_t a = 0) const {  // (0,1]
    return (double)((raw(p, px, f, a) >> 11) + 1) * (1.0 / 9007199254740992.0);
  }
  inline uint64_t uint_below(uint64_t p, uint64_t px, uint64_t f, uint64_t n, uint64_t a = 0) const {
    return (uint64_t)(u01(p, px, f, a) * (double)n);  // n << 2^53, bias negligible
  }
  inline double normal(uint64_t p, uint64_t px, uint64_t f1, uint64_t f2, uint64_t a = 0) const {
    double u1 = u01_open(p, px, f1, a), u2 = u01(p, px, f2, a);
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(kTwoPi * u2);
  }
};

struct Cfg {
  int id;
  int64_t shots;
  int particles;
  int kmin, kmax;
  double sigma;
  double amp_lo, amp_hi;  // amplitude U[lo,hi) (lo==hi: fixed)
  int centre_mode;        // 0 uniform [8,248)^2, 1 ring, 2 gaussian sigma 40, 3 separated >= 12 px
  int arrival_mode;       // 0 U{0..63}, 1 five TOF peaks
  bool pairs;             // 20 % of ions as close pairs
  bool noise;             // + floor(5 % of the shot's hits) single-pixel noise hits
  bool shuffle;           // local shuffle, displacement < 2048
};

Cfg make_cfg(int id, int64_t shots) {
  switch (id) {
    case 0: return {0, shots > 0 ? shots : 1000, 10, 3, 12, 1.0, 400, 400, 0, 0, false, false, false};
    case 1: return {1, shots > 0 ? shots : 100000, 30, 4, 20, 1.2, 400, 400, 1, 0, false, false, false};
    case 2: return {2, shots > 0 ? shots : 200000, 50, 6, 30, 1.5, 200, 900, 0, 1, true, false, false};
    case 3: return {3, shots > 0 ? shots : 50000, 200, 4, 16, 1.2, 400, 400, 2, 0, false, true, false};
    case 4: return {4, shots > 0 ? shots : 1111112, 50, 6, 30, 1.5, 200, 900, 0, 1, true, false, true};
    default: return {5, shots > 0 ? shots : 1000, 10, 3, 12, 1.0, 400, 400, 3, 0, false, false, false};
  }
}

struct Particle {
  double cx, cy, amp;
  int k;
  int64_t t0;
};

struct Hit {
  uint64_t toa;
  uint16_t x, y, tot;
};

inline bool inside(double cx, double cy) { return cx >= 8.0 && cx < 248.0 && cy >= 8.0 && cy < 248.0; }

const int64_t kPeakTicks[5] = {1280, 2560, 4480, 7040, 10240};  // 2,4,7,11,16 us

void draw_particles(const Cfg& c, const Rng& r, std::vector<Particle>& ps) {
  ps.resize(c.particles);
  for (int j = 0; j < c.particles; ++j) {
    Particle& p = ps[j];
    p.k = c.kmin + (int)r.uint_below(j, 0, F_K, (uint64_t)(c.kmax - c.kmin + 1));
    p.amp = c.amp_lo + (c.amp_hi - c.amp_lo) * r.u01(j, 0, F_AMP);
    bool second_of_pair = false;
    if (c.pairs && (j & 1) && r.u01(j - 1, 0, F_PAIR) < 0.2) second_of_pair = true;
    if (second_of_pair) {
      const Particle& q = ps[j - 1];
      uint64_t a = 0;
      for (;; ++a) {
        double d = 2.0 + 4.0 * r.u01(j, 0, F_PAIR_D, a);
        double th = kTwoPi * r.u01(j, 0, F_PAIR_TH, a);
        p.cx = q.cx + d * std::cos(th);
        p.cy = q.cy + d * std::sin(th);
        if (inside(p.cx, p.cy) || a >= 63) break;
      }
      if (!inside(p.cx, p.cy)) { p.cx = q.cx; p.cy = q.cy; }
      int64_t dt = (int64_t)r.uint_below(j, 0, F_PAIR_DT, 13) - 6;
      p.t0 = std::max<int64_t>(0, q.t0 + dt);
      continue;
    }
    for (uint64_t a = 0;; ++a) {
      if (c.centre_mode == 0) {
        p.cx = 8.0 + 240.0 * r.u01(j, 0, F_CX, a);
        p.cy = 8.0 + 240.0 * r.u01(j, 0, F_CY, a);
      } else if (c.centre_mode == 1) {
        double rad = 90.0 + 15.0 * r.normal(j, 0, F_CN1, F_CN2, a);
        double th = kTwoPi * r.u01(j, 0, F_CX, a);
        p.cx = 128.0 + rad * std::cos(th);
        p.cy = 128.0 + rad * std::sin(th);
      } else if (c.centre_mode == 2) {
        p.cx = 128.0 + 40.0 * r.normal(j, 0, F_CN1, F_CN2, a);
        p.cy = 128.0 + 40.0 * r.normal(j, 0, F_CX, F_CY, a);
      } else {
        p.cx = 8.0 + 240.0 * r.u01(j, 0, F_CX, a);
        p.cy = 8.0 + 240.0 * r.u01(j, 0, F_CY, a);
        bool ok = true;
        for (int i = 0; i < j; ++i) {
          double dx = ps[i].cx - p.cx, dy = ps[i].cy - p.cy;
          if (dx * dx + dy * dy < 144.0) { ok = false; break; }
        }
        if (!ok && a < 4095) continue;
      }
      if (inside(p.cx, p.cy)) break;
    }
    if (c.arrival_mode == 0) {
      p.t0 = (int64_t)r.uint_below(j, 0, F_ARR, 64);
    } else {
      int m = (int)r.uint_below(j, 0, F_PEAK, 5);
      double t = (double)kPeakTicks[m] + 12.8 * r.normal(j, 0, F_ARR, F_ARR2);
      p.t0 = std::max<int64_t>(0, (int64_t)std::llround(t));
    }
  }
}

inline int64_t shot_particle_hits(const std::vector<Particle>& ps) {
  int64_t s = 0;
  for (const Particle& p : ps) s += p.k;
  return s;
}

void fill_shot(const Cfg& c, const Rng& r, uint64_t shot, const std::vector<Particle>& ps, std::vector<Hit>& hits) {
  hits.clear();
  struct Cand { double r2; int y, x; };
  Cand cand[121];
  const double inv2s2 = 1.0 / (2.0 * c.sigma * c.sigma);
  for (int j = 0; j < (int)ps.size(); ++j) {
    const Particle& p = ps[j];
    int ix = (int)std::llround(p.cx), iy = (int)std::llround(p.cy);
    int nc = 0;
    for (int dy = -5; dy <= 5; ++dy)
      for (int dx = -5; dx <= 5; ++dx) {
        int px = ix + dx, py = iy + dy;
        if (px < 0 || px > 255 || py < 0 || py > 255) continue;
        double ddx = (double)px - p.cx, ddy = (double)py - p.cy;
        cand[nc++] = {ddx * ddx + ddy * ddy, py, px};
      }
    std::partial_sort(cand, cand + p.k, cand + nc, [](const Cand& a, const Cand& b) {
      if (a.r2 != b.r2) return a.r2 < b.r2;
      if (a.y != b.y) return a.y < b.y;
      return a.x < b.x;
    });
    for (int q = 0; q < p.k; ++q) {
      double v = p.amp * std::exp(-cand[q].r2 * inv2s2) + 5.0 * r.normal(j, q, F_PIX_N1, F_PIX_N2) + 0.5;
      double f = std::floor(v);
      int tot = f < 1.0 ? 1 : (f > 1023.0 ? 1023 : (int)f);
      uint64_t tw = r.uint_below(j, q, F_PIX_TW, 31);
      hits.push_back({shot * kShotPeriod + (uint64_t)p.t0 + tw, (uint16_t)cand[q].x, (uint16_t)cand[q].y, (uint16_t)tot});
    }
  }
  if (c.noise) {
    int64_t nn = (int64_t)hits.size() / 20;  // floor(5 %)
    const uint64_t NP = 0x40000000ull;       // pseudo-particle id space for noise hits
    for (int64_t q = 0; q < nn; ++q) {
      uint16_t x = (uint16_t)r.uint_below(NP, q, F_NOISE_X, 256);
      uint16_t y = (uint16_t)r.uint_below(NP, q, F_NOISE_Y, 256);
      uint64_t t = r.uint_below(NP, q, F_NOISE_T, 64000);
      uint16_t tot = (uint16_t)(1 + r.uint_below(NP, q, F_NOISE_TOT, 30));
      hits.push_back({shot * kShotPeriod + t, x, y, tot});
    }
  }
  std::stable_sort(hits.begin(), hits.end(), [](const Hit& a, const Hit& b) { return a.toa < b.toa; });
  if (c.shuffle) {
    const uint64_t SP = 0x50000000ull;
    std::vector<std::pair<uint64_t, Hit>> tmp(hits.size());
    for (size_t q = 0; q < hits.size(); ++q) tmp[q] = {q + r.uint_below(SP, q, F_SHUF, 2048), hits[q]};
    std::stable_sort(tmp.begin(), tmp.end(),
                     [](const std::pair<uint64_t, Hit>& a, const std::pair<uint64_t, Hit>& b) { return a.first < b.first; });
    for (size_t q = 0; q < hits.size(); ++q) hits[q] = tmp[q].second;
  }
}

}  // namespace

extern "C" {

// Default number of shots of a config (config 4: enough whole shots for >= 1e9 hits).
int64_t tpx3gen_default_shots(int cfg_id) { return make_cfg(cfg_id, 0).shots; }
int32_t tpx3gen_particles_per_shot(int cfg_id) { return make_cfg(cfg_id, 0).particles; }

// hits_per_shot[s - shot_begin] = number of pixel hits generated for shot s. Returns the total.
int64_t tpx3gen_count(int cfg_id, uint64_t seed, int64_t shot_begin, int64_t shot_end, int64_t* hits_per_shot,
                      int threads) {
  Cfg c = make_cfg(cfg_id, shot_end);
  int64_t total = 0;
#ifdef _OPENMP
  if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel
  {
    std::vector<Particle> ps;
#pragma omp for schedule(static) reduction(+ : total)
    for (int64_t s = shot_begin; s < shot_end; ++s) {
      Rng r(seed, (uint64_t)s);
      draw_particles(c, r, ps);
      int64_t h = shot_particle_hits(ps);
      if (c.noise) h += h / 20;
      hits_per_shot[s - shot_begin] = h;
      total += h;
    }
  }
  return total;
}

// Fill the SoA arrays. offsets[s - shot_begin] = exclusive prefix sum of hits_per_shot.
// Optional truth arrays (may be null), one entry per particle, shot-major:
//   truth_cx, truth_cy (fp64 centre), truth_k (pixels), truth_t0 (arrival tick within the shot).
void tpx3gen_fill(int cfg_id, uint64_t seed, int64_t shot_begin, int64_t shot_end, const int64_t* offsets,
                  uint16_t* x, uint16_t* y, uint64_t* toa, uint16_t* tot, double* truth_cx, double* truth_cy,
                  int32_t* truth_k, int64_t* truth_t0, int threads) {
  Cfg c = make_cfg(cfg_id, shot_end);
#ifdef _OPENMP
  if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel
  {
    std::vector<Particle> ps;
    std::vector<Hit> hits;
#pragma omp for schedule(dynamic, 64)
    for (int64_t s = shot_begin; s < shot_end; ++s) {
      Rng r(seed, (uint64_t)s);
      draw_particles(c, r, ps);
      fill_shot(c, r, (uint64_t)s, ps, hits);
      int64_t o = offsets[s - shot_begin];
      for (size_t q = 0; q < hits.size(); ++q) {
        x[o + q] = hits[q].x;
        y[o + q] = hits[q].y;
        toa[o + q] = hits[q].toa;
        tot[o + q] = hits[q].tot;
      }
      if (truth_cx) {
        int64_t b = (s - shot_begin) * c.particles;
        for (int j = 0; j < c.particles; ++j) {
          truth_cx[b + j] = ps[j].cx;
          truth_cy[b + j] = ps[j].cy;
          truth_k[b + j] = ps[j].k;
          truth_t0[b + j] = ps[j].t0;
        }
      }
    }
  }
}

}  // extern "C"
