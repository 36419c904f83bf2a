// Paper-literal mode: the paper's own definition of a hit, §V.
//
//   neighbourhood  A_ij = [|X_i-X_j| <= wx] [|Y_i-Y_j| <= wy] [|ToF_i-ToF_j| <= wt], same laser shot,
//                  A_ii = 1                                   Eq. 3-5, PAPER.md:109-126 (inclusive, :117)
//   hit            a pixel i with no neighbour of greater ToT (Eq. 6-7, :134-148); equal ToT: the pixel
//                  later in the sorted stream wins (:150) = lexicographic (ToT, sorted index), R7
//   centroid       sum_j V_j A_ij ToT_j / sum_j ToT_j A_ij over row i of A, V = X, Y, ToF
//                                                             Eq. 8-9
//
// The paper forms A as a dense N x N array per shot (its stated memory limit). Here the
// rows of A are never stored: after the stable (shot, ToA) sort (general path, tpx3_sort.cuh) the events
// that can be neighbours of i in time — same shot, |dToA| <= wt — are one contiguous window of the
// sorted stream around i, and a thread walks that window testing the two spatial inequalities.
//   k_lm_gather  sorted records: ToA (u64) and x | y << 8 | tot << 16 (u32)
//   k_lm_flag    lmax[k] = k if k is a local maximum, 0xFFFFFFFF otherwise (stops at the first brighter neighbour)
//   k_root_*     (tpx3_centroid.cuh) ordinals of the hits in ascending k, hit count
//   k_lm_emit    one thread per hit walks the window again: exact integer row sums of Eq. 9, fp32 divides
#pragma once
#include "tpx3_common.cuh"

namespace tpx3 {

__global__ void __launch_bounds__(256) k_lm_gather(uint64_t n, const uint32_t* __restrict__ perm,
                                                 const uint16_t* __restrict__ x, const uint16_t* __restrict__ y,
                                                 const uint64_t* __restrict__ toa, const uint16_t* __restrict__ tot,
                                                 uint64_t* __restrict__ toa_s, uint32_t* __restrict__ rec) {
  for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t i = perm[k];
    toa_s[k] = toa[i];
    rec[k] = ((uint32_t)x[i] & 0xFFu) | (((uint32_t)y[i] & 0xFFu) << 8) | ((uint32_t)tot[i] << 16);
  }
}

// The ToA interval that holds every possible time neighbour of an event at ToA t: same shot
// (R6) and |dToA| <= wt (inside a shot dToF = dToA, R5).
__device__ __forceinline__ void lm_window(uint64_t t, uint64_t P, uint64_t wt, uint64_t& lo, uint64_t& hi) {
  lo = t >= wt ? t - wt : 0ull;
  hi = t + wt >= t ? t + wt : ~0ull;
  if (P) {
    const uint64_t s0 = t - t % P;               // start of the shot
    const uint64_t s1 = s0 + (P - 1ull);         // its last tick
    if (lo < s0) lo = s0;
    if (s1 >= s0 && hi > s1) hi = s1;
  }
}

__device__ __forceinline__ bool lm_near(uint32_t ra, uint32_t rb, uint32_t wx, uint32_t wy) {
  const uint32_t xa = ra & 0xFFu, xb = rb & 0xFFu, ya = (ra >> 8) & 0xFFu, yb = (rb >> 8) & 0xFFu;
  const uint32_t dx = xa > xb ? xa - xb : xb - xa, dy = ya > yb ? ya - yb : yb - ya;
  return dx <= wx && dy <= wy;
}

__global__ void __launch_bounds__(256) k_lm_flag(uint64_t n, uint64_t P, uint32_t wx, uint32_t wy, uint64_t wt,
                                               const uint64_t* __restrict__ toa_s, const uint32_t* __restrict__ rec,
                                               uint32_t* __restrict__ lmax) {
  for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t t = toa_s[k];
    const uint32_t r = rec[k], ti = r >> 16;
    uint64_t lo, hi;
    lm_window(t, P, wt, lo, hi);
    bool is_max = true;
    // earlier pixels: a strictly greater ToT beats k (an equal one loses to k, the later pixel)
    for (uint64_t j = k; is_max && j-- > 0;) {
      if (toa_s[j] < lo) break;
      const uint32_t rj = rec[j];
      if ((rj >> 16) > ti && lm_near(r, rj, wx, wy)) is_max = false;
    }
    // later pixels: greater or equal ToT beats k
    for (uint64_t j = k + 1; is_max && j < n; ++j) {
      if (toa_s[j] > hi) break;
      const uint32_t rj = rec[j];
      if ((rj >> 16) >= ti && lm_near(r, rj, wx, wy)) is_max = false;
    }
    lmax[k] = is_max ? (uint32_t)k : 0xFFFFFFFFu;
  }
}

// One thread per hit c (out.label[c] = sorted position of the local maximum, written by k_root_slots).
__global__ void __launch_bounds__(128) k_lm_emit(Ctrl* c, uint64_t n, uint64_t P, uint32_t wx, uint32_t wy, uint64_t wt,
                                               const uint64_t* __restrict__ toa_s, const uint32_t* __restrict__ rec,
                                               const uint32_t* n_hits, uint64_t max_clusters, tpx3_clusters_t out) {
  uint64_t nc = *n_hits;
  if (nc > max_clusters) nc = max_clusters;
  if (blockIdx.x == 0 && threadIdx.x == 0) { c->status.path = 3; }
  for (uint64_t h = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; h < nc; h += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t k = out.label[h];
    const uint64_t t = toa_s[k];
    const uint32_t r = rec[k];
    uint64_t lo, hi;
    lm_window(t, P, wt, lo, hi);
    const uint64_t s0 = P ? t - t % P : 0ull;   // ToF = ToA - shot * P (P = 0: ToF = ToA)
    unsigned long long st = 0, sx = 0, sy = 0, sf = 0;
    uint32_t size = 0;
    auto add = [&](uint64_t j) {
      const uint32_t rj = rec[j];
      if (lm_near(r, rj, wx, wy)) {
        const unsigned long long w = rj >> 16;
        ++size;
        st += w;
        sx += w * (rj & 0xFFu);
        sy += w * ((rj >> 8) & 0xFFu);
        sf += w * (toa_s[j] - s0);
      }
    };
    add(k);                                       // A_ii = 1 (Eq. 4 diagonal)
    for (uint64_t j = k; j-- > 0;) {
      if (toa_s[j] < lo) break;
      add(j);
    }
    for (uint64_t j = k + 1; j < n; ++j) {
      if (toa_s[j] > hi) break;
      add(j);
    }
    out.size[h] = size;
    out.shot[h] = (uint32_t)(P ? t / P : 0ull);
    out.sum_tot[h] = (long long)st;
    out.sum_tot_x[h] = (long long)sx;
    out.sum_tot_y[h] = (long long)sy;
    out.sum_tot_tof[h] = (long long)sf;
    out.toa_peak[h] = t;
    const float fst = __ll2float_rn((long long)st);
    out.cx[h] = __fdiv_rn(__ll2float_rn((long long)sx), fst);
    out.cy[h] = __fdiv_rn(__ll2float_rn((long long)sy), fst);
    out.ctof[h] = __fdiv_rn(__ll2float_rn((long long)sf), fst);
  }
}

}  // namespace tpx3
