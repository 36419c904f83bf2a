// General path, S2/S3: space-time neighbour linking and label compression on the sorted
// stream, for inputs of any shape (one giant shot, shots interleaved in the stream, ...).
//
// Relation (Eq. 4-5 with w_x = w_y = 1, w_t = W, inclusive; same shot only):
//   i ~ j  <=>  shot_i == shot_j, |x_i - x_j| <= 1, |y_i - y_j| <= 1, |toa_i - toa_j| <= W.
// The dense N x N adjacency of the paper (the O(N^2) memory it names as its limit,
// PAPER.md:181) is never formed. Instead time inside a shot is cut into slabs of W+1 ticks:
//   * two events of the same (slab, pixel) are always related (same cell, |dt| <= W);
//   * an event in slab s can only be related to events of slabs s-1, s, s+1;
//   * for a (slab s-1, cell c) it suffices to test the LATEST event of that slab-cell: if any
//     event of it is within W of k, the latest one is, and it is related to all the others.
// So a hash table keyed by (slab, cell) holding the largest sorted index of each slab-cell,
// probed at 5 cells of the own slab (own + 4 "forward" neighbours; the relation is symmetric)
// and 9 cells of the previous slab, yields a set of links whose transitive closure equals the
// closure of the full relation. Links are applied to a lock-free union-find in global memory
// that always hooks the larger root under the smaller, so the root of a component is its
// smallest sorted index — the canonical label of S3 — without renumbering.
#pragma once
#include "tpx3_common.cuh"

namespace tpx3 {

struct SortedView {       // the sorted stream as the general path stores it
  const uint64_t* key;    // ToA - toa_min, ascending
  uint32_t* xy;           // x | y << 16
  uint16_t* tot;
  uint64_t* slab;         // global slab number (see k_gather)
};

__device__ __forceinline__ uint32_t slab_hash(uint64_t slab, uint32_t xy, uint32_t mask) {
  uint64_t h = (slab * 0x9E3779B97F4A7C15ull) ^ ((uint64_t)xy * 0xC2B2AE3D27D4EB4Full);
  h ^= h >> 29;
  h *= 0xBF58476D1CE4E5B9ull;
  return (uint32_t)(h >> 32) & mask;
}

// Gather the sorted records and number the slabs:
//   slab = shot * (SPS + 1) + tof div (W+1) + 1,  SPS = ceil(P / (W+1))
// so that (slab - 1) of the first slab of a shot is a number no event carries: a probe of the
// "previous slab" can never cross into the previous shot. P == 0: slab = toa div (W+1) + 1.
__global__ void __launch_bounds__(256) k_gather(Ctrl* c, Params p, const uint64_t* __restrict__ keyA,
                                              const uint64_t* __restrict__ keyB, const uint32_t* __restrict__ perm,
                                              const uint16_t* __restrict__ x, const uint16_t* __restrict__ y,
                                              const uint16_t* __restrict__ tot, uint32_t* __restrict__ s_xy,
                                              uint16_t* __restrict__ s_tot, uint64_t* __restrict__ s_slab,
                                              uint32_t* __restrict__ parent) {
  if (c->fused_state == 1) return;
  const uint64_t* key = ((c->npass - 1) & 1) ? keyB : keyA;
  const uint64_t tmin = c->toa_min;
  for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < p.n; k += (uint64_t)gridDim.x * blockDim.x) {
    uint32_t i = perm[k];
    uint32_t xx = x[i], yy = y[i], tt = tot[i];
    if ((p.flags & TPX3_FLAG_VALIDATE_INPUT) && (xx >= p.sensor_w || yy >= p.sensor_h || tt == 0))
      set_error(c, TPX3_ERR_OUT_OF_RANGE);
    s_xy[k] = xx | (yy << 16);
    s_tot[k] = (uint16_t)tt;
    uint64_t t = key[k] + tmin;
    uint64_t slab;
    if (p.P) {
      uint64_t shot = t / p.P, tof = t - shot * p.P;
      slab = shot * p.slabs_per_shot_p1 + tof / (p.W + 1ull) + 1ull;
    } else {
      slab = t / (p.W + 1ull) + 1ull;
    }
    s_slab[k] = slab;
    parent[k] = (uint32_t)k;
  }
}

__global__ void __launch_bounds__(256) k_hash_insert(Ctrl* c, uint64_t n, const uint32_t* __restrict__ s_xy,
                                                   const uint64_t* __restrict__ s_slab, uint32_t* table,
                                                   uint32_t mask) {
  if (c->fused_state == 1) return;
  for (uint64_t kk = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; kk < n; kk += (uint64_t)gridDim.x * blockDim.x) {
    uint32_t k = (uint32_t)kk, xy = s_xy[k];
    uint64_t slab = s_slab[k];
    uint32_t h = slab_hash(slab, xy, mask);
    for (;;) {
      uint32_t cur = table[h];
      if (cur == kEmpty) {
        cur = atomicCAS(&table[h], kEmpty, k);
        if (cur == kEmpty) break;
      }
      if (s_slab[cur] == slab && s_xy[cur] == xy) {  // same slab-cell: keep the latest event
        atomicMax(&table[h], k);
        break;
      }
      h = (h + 1) & mask;
    }
  }
}

__device__ __forceinline__ uint32_t hash_lookup(const uint32_t* table, uint32_t mask, const uint32_t* s_xy,
                                                const uint64_t* s_slab, uint64_t slab, uint32_t xy) {
  uint32_t h = slab_hash(slab, xy, mask);
  for (;;) {
    uint32_t cur = table[h];
    if (cur == kEmpty) return kEmpty;
    if (s_slab[cur] == slab && s_xy[cur] == xy) return cur;
    h = (h + 1) & mask;
  }
}

__device__ __forceinline__ uint32_t uf_find(uint32_t* parent, uint32_t a) {
  uint32_t p = parent[a];
  while (p != a) {
    uint32_t g = parent[p];
    if (g != p) parent[a] = g;  // path halving (benign race: only ever lowers towards the root)
    a = p;
    p = g;
  }
  return a;
}

// Lock-free union: hook the larger root under the smaller one.
__device__ __forceinline__ void uf_union(uint32_t* parent, uint32_t a, uint32_t b) {
  for (;;) {
    a = uf_find(parent, a);
    b = uf_find(parent, b);
    if (a == b) return;
    if (a < b) { uint32_t t = a; a = b; b = t; }  // a > b
    uint32_t old = atomicMin(&parent[a], b);
    if (old == a) return;  // a was still a root: hooked
    a = old;               // someone hooked a elsewhere in the meantime: continue from there
  }
}

__global__ void __launch_bounds__(256) k_link(Ctrl* c, Params p, const uint64_t* __restrict__ keyA,
                                            const uint64_t* __restrict__ keyB, const uint32_t* __restrict__ s_xy,
                                            const uint64_t* __restrict__ s_slab, const uint32_t* __restrict__ table,
                                            uint32_t mask, uint32_t* parent) {
  if (c->fused_state == 1) return;
  const uint64_t* key = ((c->npass - 1) & 1) ? keyB : keyA;
  for (uint64_t kk = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; kk < p.n; kk += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t k = (uint32_t)kk, xy = s_xy[k];
    const int x = (int)(xy & 0xFFFF), y = (int)(xy >> 16);
    const uint64_t slab = s_slab[k], t = key[k];
    // own slab: own cell + 4 forward neighbours (E, SW, S, SE)
    const int fdx[5] = {0, 1, -1, 0, 1}, fdy[5] = {0, 0, 1, 1, 1};
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      int nx = x + fdx[q], ny = y + fdy[q];
      if (nx < 0 || ny < 0 || nx >= (int)p.sensor_w || ny >= (int)p.sensor_h) continue;
      uint32_t j = hash_lookup(table, mask, s_xy, s_slab, slab, (uint32_t)nx | ((uint32_t)ny << 16));
      if (j != kEmpty && j != k) uf_union(parent, k, j);
    }
    // previous slab: all 9 cells, latest event of each, explicit time test
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        int nx = x + dx, ny = y + dy;
        if (nx < 0 || ny < 0 || nx >= (int)p.sensor_w || ny >= (int)p.sensor_h) continue;
        uint32_t j = hash_lookup(table, mask, s_xy, s_slab, slab - 1, (uint32_t)nx | ((uint32_t)ny << 16));
        if (j != kEmpty && t - key[j] <= (uint64_t)p.W) uf_union(parent, k, j);
      }
  }
}

// S3: label[k] = root of k (the smallest sorted index of the component); count the roots.
__global__ void __launch_bounds__(256) k_compress(Ctrl* c, uint64_t n, uint32_t* parent, uint32_t* n_clusters) {
  if (c->fused_state == 1) return;
  uint32_t roots = 0;
  for (uint64_t kk = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; kk < n; kk += (uint64_t)gridDim.x * blockDim.x) {
    uint32_t k = (uint32_t)kk, r = k, q = parent[r];
    while (q != r) { r = q; q = parent[r]; }
    // Writing the root into parent[k] while others traverse is safe: every value ever stored
    // at parent[k] is an ancestor of k, and the root never changes in this kernel.
    parent[k] = r;
    roots += (r == k);
  }
  for (int o = 16; o; o >>= 1) roots += __shfl_xor_sync(0xffffffffu, roots, o);
  if ((threadIdx.x & 31) == 0 && roots) {
    atomicAdd(n_clusters, roots);
    atomicAdd(&c->status.n_clusters, roots);
  }
}

}  // namespace tpx3
