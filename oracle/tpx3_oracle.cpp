// ORACLE — TEST INFRASTRUCTURE ONLY. Plain, slow, obviously-correct CPU definition of what
// the hot path computes. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call it. It shares no code with the CUDA path
// (paper_2603_04942_b200/csrc): different algorithm (per-shot BFS over a cell -> hits map,
// std::stable_sort), different language unit, no common headers.
//
// What it computes (north_star's clustering; the relation is the paper's Eq. 5):
//   1. shot_i = toa_i div P            (P = 0: one shot)        PAPER.md:68 "most recent laser
//      trigger"; BASELINE.json configs: shot_start = shot * P   (reading R6)
//   2. perm = stable sort of hit indices by (shot, toa); everything below is indexed by
//      sorted position k                                          (north_star; PAPER.md:96
//      "essentially unsorted order")
//   3. neighbours: i != j, same shot, |x_i-x_j| <= 1, |y_i-y_j| <= 1, |toa_i-toa_j| <= W,
//      all three inclusive — A = A^X (.) A^Y (.) A^ToF, PAPER.md:117 ("|D| <= 5" inclusive),
//      :122-126 (Eq. 5) with w_x = w_y = 1, w_t = W. A hit (particle hit) is a connected
//      component of that relation; label[k] = smallest sorted index in k's component
//      (per-shot BFS started from hits in ascending order).
//   4. per component: size, sum tot, sum tot*x, sum tot*y (int64), peak = member maximising
//      (tot, sorted index) lexicographically — PAPER.md:134 (ToT as brightness), :150 (ties:
//      the later pixel in the stream wins) — toa_peak = toa[peak], shot.
//   5. centroid cx = (float)sum(tot*x) / (float)sum(tot), cy likewise — PAPER.md:156 (Eq. 8),
//      :162 (Eq. 9) with A_ij restricted to the component; fp32 IEEE divide of the two
//      int64 sums each rounded to fp32 (reading R12). Clusters are listed in
//      ascending label order.
//   6. time-of-flight centroid: "this procedure is identical for X, Y and
//      ToF", ToF = ToA - laser trigger = toa - shot*P (R6; P = 0:
//      ToF = ToA): sum_tot_tof = sum(tot*tof) in int64, ctof = (float)sum_tot_tof / (float)sum(tot)
//      in ticks (R20).
//
// Pins (tests/test_oracle_pins.py): the paper's worked example (Eq. 2-7, :106-148), brute
// force O(n^2) adjacency + closure on tiny inputs (oracle/bruteforce.py, written directly
// from Eq. 3-5), invariants, closed forms for 1- and 2-pixel clusters, generated truth.
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <numeric>
#include <unordered_map>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct ShotRange { uint64_t a, b; };

// BFS over one shot's hits [a, b) (sorted positions). cells: cell id -> sorted positions.
void label_shot(uint64_t a, uint64_t b, const uint32_t* perm, const uint16_t* x, const uint16_t* y,
                const uint64_t* toa, uint64_t W, uint32_t* label) {
  std::unordered_map<uint64_t, std::vector<uint32_t>> cells;
  cells.reserve((size_t)(b - a) * 2);
  auto cell_of = [](int64_t cx, int64_t cy) { return ((uint64_t)(uint32_t)cy << 32) | (uint64_t)(uint32_t)cx; };
  for (uint64_t k = a; k < b; ++k) cells[cell_of(x[perm[k]], y[perm[k]])].push_back((uint32_t)k);
  const uint32_t UNSET = 0xFFFFFFFFu;
  for (uint64_t k = a; k < b; ++k) label[k] = UNSET;
  std::vector<uint32_t> queue;
  for (uint64_t k = a; k < b; ++k) {
    if (label[k] != UNSET) continue;
    label[k] = (uint32_t)k;
    queue.clear();
    queue.push_back((uint32_t)k);
    for (size_t qi = 0; qi < queue.size(); ++qi) {
      uint32_t u = queue[qi];
      int64_t ux = x[perm[u]], uy = y[perm[u]];
      uint64_t ut = toa[perm[u]];
      for (int64_t dy = -1; dy <= 1; ++dy)
        for (int64_t dx = -1; dx <= 1; ++dx) {
          int64_t vx = ux + dx, vy = uy + dy;
          if (vx < 0 || vy < 0) continue;  // no wrap-around at the sensor edge
          auto it = cells.find(cell_of(vx, vy));
          if (it == cells.end()) continue;
          for (uint32_t v : it->second) {
            if (v == u || label[v] != UNSET) continue;
            uint64_t vt = toa[perm[v]];
            uint64_t d = ut > vt ? ut - vt : vt - ut;
            if (d <= W) {
              label[v] = (uint32_t)k;
              queue.push_back(v);
            }
          }
        }
    }
  }
}

}  // namespace

extern "C" {

// Returns 0 on success. All arrays are caller-owned host memory.
//   perm[n], label[n] (indexed by sorted position), *n_clusters
//   cluster arrays have capacity n: c_label, c_size, c_shot (uint32; shot truncated to 32 bits),
//   c_sum_tot, c_sum_tot_x, c_sum_tot_y (int64), c_toa_peak (uint64), c_cx, c_cy (float),
//   c_sum_tot_tof (int64), c_ctof (float)
//   any cluster array pointer may be null (skipped).
int tpx3_oracle_run(uint64_t n, const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                    uint64_t W, uint64_t P, int threads, uint32_t* perm, uint32_t* label, uint64_t* n_clusters,
                    uint32_t* c_label, uint32_t* c_size, uint32_t* c_shot, int64_t* c_sum_tot, int64_t* c_sum_tot_x,
                    int64_t* c_sum_tot_y, uint64_t* c_toa_peak, float* c_cx, float* c_cy, int64_t* c_sum_tot_tof,
                    float* c_ctof) {
  if (n >= 0xFFFFFFFFull) return -1;
#ifdef _OPENMP
  if (threads > 0) omp_set_num_threads(threads);
#endif
  // 1-2. shot and stable sort by (shot, toa)
  std::iota(perm, perm + n, 0u);
  auto shot_of = [&](uint32_t i) -> uint64_t { return P ? toa[i] / P : 0; };
  std::stable_sort(perm, perm + n, [&](uint32_t i, uint32_t j) {
    uint64_t si = shot_of(i), sj = shot_of(j);
    if (si != sj) return si < sj;
    return toa[i] < toa[j];
  });
  // shot ranges in sorted order
  std::vector<ShotRange> shots;
  for (uint64_t k = 0; k < n;) {
    uint64_t s = shot_of(perm[k]), e = k + 1;
    while (e < n && shot_of(perm[e]) == s) ++e;
    shots.push_back({k, e});
    k = e;
  }
  // 3. connected components per shot
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t si = 0; si < (int64_t)shots.size(); ++si)
    label_shot(shots[si].a, shots[si].b, perm, x, y, toa, W, label);
  // 4-5. per-component sums, peak, centroid; clusters in ascending label order
  std::vector<uint32_t> slot(n);
  uint64_t nc = 0;
  for (uint64_t k = 0; k < n; ++k)
    if (label[k] == k) slot[k] = (uint32_t)nc++;
  *n_clusters = nc;
  std::vector<int64_t> st(nc, 0), sx(nc, 0), sy(nc, 0), sf(nc, 0);
  std::vector<uint32_t> sz(nc, 0), peak(nc, 0), ptot(nc, 0);
  for (uint64_t k = 0; k < n; ++k) {
    uint32_t c = slot[label[k]];
    uint32_t i = perm[k];
    int64_t t = tot[i];
    sz[c] += 1;
    st[c] += t;
    sx[c] += t * (int64_t)x[i];
    sy[c] += t * (int64_t)y[i];
    sf[c] += t * (int64_t)(P ? toa[i] % P : toa[i]);  // ToF = ToA - shot*P
    if (sz[c] == 1 || tot[i] >= ptot[c]) {  // k ascending: '>=' makes the later pixel win ties
      ptot[c] = tot[i];
      peak[c] = (uint32_t)k;
    }
  }
  uint64_t c = 0;
  for (uint64_t k = 0; k < n; ++k) {
    if (label[k] != k) continue;
    if (c_label) c_label[c] = (uint32_t)k;
    if (c_size) c_size[c] = sz[c];
    if (c_shot) c_shot[c] = (uint32_t)shot_of(perm[k]);
    if (c_sum_tot) c_sum_tot[c] = st[c];
    if (c_sum_tot_x) c_sum_tot_x[c] = sx[c];
    if (c_sum_tot_y) c_sum_tot_y[c] = sy[c];
    if (c_toa_peak) c_toa_peak[c] = toa[perm[peak[c]]];
    if (c_cx) c_cx[c] = (float)sx[c] / (float)st[c];
    if (c_cy) c_cy[c] = (float)sy[c] / (float)st[c];
    if (c_sum_tot_tof) c_sum_tot_tof[c] = sf[c];
    if (c_ctof) c_ctof[c] = (float)sf[c] / (float)st[c];
    ++c;
  }
  return 0;
}


// Paper-literal mode — the paper's own definition of a hit, §V:
//   neighbourhood  A_ij = [|X_i-X_j| <= wx] [|Y_i-Y_j| <= wy] [|ToF_i-ToF_j| <= wt], same laser shot,
//                  A_ii = 1                                   Eq. 3-5, PAPER.md:109-126 (inclusive, :117)
//   hit            a pixel i with no neighbour of greater ToT (Eq. 6-7, :134-148); equal ToT: the pixel
//                  later in the (sorted) stream wins (:150) — taken as the lexicographic order on
//                  (ToT, sorted index), reading R7
//   centroid       sum_j V_j A_ij ToT_j / sum_j ToT_j A_ij over ROW i of A (the box about the local
//                  maximum), V = X, Y and ToF alike          Eq. 8-9
// Plain definition: after the stable (shot, ToA) sort every pair of a shot is tested, O(m^2) per shot.
// Outputs as tpx3_oracle_run, one row per hit in ascending sorted index: c_label = the sorted index of
// the local-maximum pixel, c_size = sum_j A_ij, c_toa_peak = its ToA; lmax[k] = k for a hit, 0xFFFFFFFF else.
int tpx3_oracle_localmax(uint64_t n, const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                         uint64_t wx, uint64_t wy, uint64_t wt, uint64_t P, int threads, uint32_t* perm,
                         uint32_t* lmax, uint64_t* n_hits, uint32_t* c_label, uint32_t* c_size, uint32_t* c_shot,
                         int64_t* c_sum_tot, int64_t* c_sum_tot_x, int64_t* c_sum_tot_y, uint64_t* c_toa_peak,
                         float* c_cx, float* c_cy, int64_t* c_sum_tot_tof, float* c_ctof) {
  if (n >= 0xFFFFFFFFull) return -1;
#ifdef _OPENMP
  if (threads > 0) omp_set_num_threads(threads);
#endif
  std::iota(perm, perm + n, 0u);
  auto shot_of = [&](uint32_t i) -> uint64_t { return P ? toa[i] / P : 0; };
  std::stable_sort(perm, perm + n, [&](uint32_t i, uint32_t j) {
    uint64_t si = shot_of(i), sj = shot_of(j);
    if (si != sj) return si < sj;
    return toa[i] < toa[j];
  });
  std::vector<ShotRange> shots;
  for (uint64_t k = 0; k < n;) {
    uint64_t s = shot_of(perm[k]), e = k + 1;
    while (e < n && shot_of(perm[e]) == s) ++e;
    shots.push_back({k, e});
    k = e;
  }
  auto adjacent = [&](uint64_t i, uint64_t j) -> bool {  // i, j sorted positions of one shot
    uint32_t a = perm[i], b = perm[j];
    uint64_t dx = x[a] > x[b] ? x[a] - x[b] : x[b] - x[a];
    uint64_t dy = y[a] > y[b] ? y[a] - y[b] : y[b] - y[a];
    uint64_t dt = toa[a] > toa[b] ? toa[a] - toa[b] : toa[b] - toa[a];  // same shot: dToF = dToA
    return dx <= wx && dy <= wy && dt <= wt;
  };
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t si = 0; si < (int64_t)shots.size(); ++si) {
    for (uint64_t i = shots[si].a; i < shots[si].b; ++i) {
      bool is_max = true;
      for (uint64_t j = shots[si].a; j < shots[si].b && is_max; ++j) {
        if (j == i || !adjacent(i, j)) continue;
        uint16_t ti = tot[perm[i]], tj = tot[perm[j]];
        if (tj > ti || (tj == ti && j > i)) is_max = false;
      }
      lmax[i] = is_max ? (uint32_t)i : 0xFFFFFFFFu;
    }
  }
  uint64_t c = 0;
  for (size_t si = 0; si < shots.size(); ++si) {
    for (uint64_t i = shots[si].a; i < shots[si].b; ++i) {
      if (lmax[i] != i) continue;
      int64_t st = 0, sx = 0, sy = 0, sf = 0;
      uint32_t sz = 0;
      for (uint64_t j = shots[si].a; j < shots[si].b; ++j) {
        if (!adjacent(i, j)) continue;  // j == i included: A_ii = 1
        uint32_t b = perm[j];
        int64_t t = tot[b];
        ++sz;
        st += t;
        sx += t * (int64_t)x[b];
        sy += t * (int64_t)y[b];
        sf += t * (int64_t)(P ? toa[b] % P : toa[b]);
      }
      if (c_label) c_label[c] = (uint32_t)i;
      if (c_size) c_size[c] = sz;
      if (c_shot) c_shot[c] = (uint32_t)shot_of(perm[i]);
      if (c_sum_tot) c_sum_tot[c] = st;
      if (c_sum_tot_x) c_sum_tot_x[c] = sx;
      if (c_sum_tot_y) c_sum_tot_y[c] = sy;
      if (c_toa_peak) c_toa_peak[c] = toa[perm[i]];
      if (c_cx) c_cx[c] = (float)sx / (float)st;
      if (c_cy) c_cy[c] = (float)sy / (float)st;
      if (c_sum_tot_tof) c_sum_tot_tof[c] = sf;
      if (c_ctof) c_ctof[c] = (float)sf / (float)st;
      ++c;
    }
  }
  *n_hits = c;
  return 0;
}

}  // extern "C"
