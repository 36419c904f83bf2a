// S4/S5 as a standalone step: per-hit integer sums, brightest pixel and ToT-weighted centroid
// (Eq. 8-9 with A_ij restricted to the connected component) from ANY valid
// (perm, label) pair. Used by tpx3_centroid and by the general path of tpx3_cluster_centroid;
// the fused path computes the same quantities inside its tile kernel.
//
//   k_root_count / k_root_scan / k_root_slots : ordinal of each root in ascending label order
//   k_accumulate : exact integer atomics into the output arrays (order-independent)
//   k_finalize   : peak ToA, shot, fp32 divide (IEEE RN; no fast-math)
#pragma once
#include "tpx3_common.cuh"

namespace tpx3 {

constexpr int kCentThreads = 256;
constexpr int kCentItems = 16;
constexpr int kCentTile = kCentThreads * kCentItems;  // 4096 sorted positions per block

__device__ __forceinline__ uint32_t block_exclusive_scan_256(uint32_t v, uint32_t* smem33, uint32_t* total) {
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t inc = v;
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (uint32_t)o) inc += t;
  }
  if (lane == 31) smem33[w] = inc;
  __syncthreads();
  if (w == 0) {
    uint32_t ws = lane < (blockDim.x >> 5) ? smem33[lane] : 0, x = ws;
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= (uint32_t)o) x += t;
    }
    if (lane < (blockDim.x >> 5)) smem33[lane] = x - ws;
    if (lane == 31) smem33[32] = x;
  }
  __syncthreads();
  uint32_t r = smem33[w] + inc - v;
  if (total) *total = smem33[32];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(kCentThreads) k_root_count(Ctrl* c, int general_only, uint64_t n,
                                                           const uint32_t* __restrict__ label, uint32_t* blk_cnt) {
  if (general_only && c->fused_state == 1) return;
  __shared__ uint32_t sm[33];
  uint64_t base = (uint64_t)blockIdx.x * kCentTile;
  uint32_t cnt = 0;
#pragma unroll
  for (int i = 0; i < kCentItems; ++i) {
    uint64_t k = base + (uint64_t)i * kCentThreads + threadIdx.x;
    if (k < n) cnt += (label[k] == (uint32_t)k);
  }
  uint32_t total;
  block_exclusive_scan_256(cnt, sm, &total);
  if (threadIdx.x == 0) blk_cnt[blockIdx.x] = total;
}

// Exclusive scan of blk_cnt[nblk] in place (single block); writes the hit count.
__global__ void __launch_bounds__(1024) k_root_scan(Ctrl* c, int general_only, uint32_t* blk_cnt, uint32_t nblk,
                                                  uint64_t max_clusters, uint32_t* n_clusters) {
  if (general_only && c->fused_state == 1) return;
  const uint32_t x = scan_inplace_1024(blk_cnt, nblk);
  if (threadIdx.x == 0) {
    *n_clusters = x;
    c->status.n_clusters = x;
    if ((uint64_t)x > max_clusters) set_error(c, TPX3_ERR_CAPACITY);
  }
}

// slot[k] = ordinal of root k (only written for roots); the root initialises its cluster row.
__global__ void __launch_bounds__(kCentThreads) k_root_slots(Ctrl* c, int general_only, uint64_t n,
                                                           const uint32_t* __restrict__ label,
                                                           const uint32_t* __restrict__ blk_cnt, uint32_t* slot,
                                                           uint64_t max_clusters, tpx3_clusters_t out,
                                                           unsigned long long* peak) {
  if (general_only && c->fused_state == 1) return;
  __shared__ uint32_t sm[33];
  // blocked arrangement so that the in-block order is ascending k
  uint64_t base = (uint64_t)blockIdx.x * kCentTile + (uint64_t)threadIdx.x * kCentItems;
  uint32_t flags = 0, cnt = 0;
#pragma unroll
  for (int i = 0; i < kCentItems; ++i) {
    uint64_t k = base + i;
    if (k < n && label[k] == (uint32_t)k) { flags |= 1u << i; ++cnt; }
  }
  uint32_t off = block_exclusive_scan_256(cnt, sm, nullptr) + blk_cnt[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kCentItems; ++i) {
    if (flags & (1u << i)) {
      uint64_t k = base + i;
      slot[k] = off;
      if ((uint64_t)off < max_clusters) {
        out.label[off] = (uint32_t)k;
        out.size[off] = 0;
        out.sum_tot[off] = 0;
        out.sum_tot_x[off] = 0;
        out.sum_tot_y[off] = 0;
        out.sum_tot_tof[off] = 0;
        peak[off] = 0ull;
      }
      ++off;
    }
  }
}

__global__ void __launch_bounds__(256) k_accumulate(Ctrl* c, int general_only, uint64_t n,
                                                  const uint16_t* __restrict__ x, const uint16_t* __restrict__ y,
                                                  const uint16_t* __restrict__ tot, const uint64_t* __restrict__ toa,
                                                  uint64_t P, const uint32_t* __restrict__ perm,
                                                  const uint32_t* __restrict__ label, const uint32_t* __restrict__ slot,
                                                  uint64_t max_clusters, tpx3_clusters_t out, unsigned long long* peak) {
  if (general_only && c->fused_state == 1) return;
  for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (uint64_t)gridDim.x * blockDim.x) {
    uint32_t i = perm[k], s = slot[label[k]];
    if ((uint64_t)s >= max_clusters) continue;
    unsigned long long t = tot[i];
    atomicAdd(&out.size[s], 1u);
    atomicAdd((unsigned long long*)&out.sum_tot[s], t);
    atomicAdd((unsigned long long*)&out.sum_tot_x[s], t * (unsigned long long)x[i]);
    atomicAdd((unsigned long long*)&out.sum_tot_y[s], t * (unsigned long long)y[i]);
    // time of flight = ToA - shot * P (P = 0: one shot triggered at tick 0)
    const unsigned long long tof = P ? toa[i] % P : toa[i];
    atomicAdd((unsigned long long*)&out.sum_tot_tof[s], t * tof);
    // brightest pixel: max over (ToT, sorted position) — the later pixel wins ties
    atomicMax(&peak[s], (t << 32) | (unsigned long long)k);
  }
}

__global__ void __launch_bounds__(256) k_finalize(Ctrl* c, int general_only, Params p,
                                                const uint64_t* __restrict__ toa, const uint32_t* __restrict__ perm,
                                                const uint32_t* n_clusters, uint64_t max_clusters, tpx3_clusters_t out,
                                                const unsigned long long* __restrict__ peak,
                                                const uint64_t* __restrict__ label_base) {
  if (general_only && c->fused_state == 1) return;
  uint64_t nc = *n_clusters;
  if (nc > max_clusters) nc = max_clusters;
  const uint32_t lbase = label_base ? (uint32_t)*label_base : 0u;   // stream pushes: labels continue the batch numbering
  for (uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; s < nc; s += (uint64_t)gridDim.x * blockDim.x) {
    uint32_t kpeak = (uint32_t)(peak[s] & 0xFFFFFFFFull);
    out.toa_peak[s] = toa[perm[kpeak]];
    uint64_t t0 = toa[perm[out.label[s]]];
    out.shot[s] = (uint32_t)(p.P ? t0 / p.P : 0ull);
    long long st = out.sum_tot[s], sx = out.sum_tot_x[s], sy = out.sum_tot_y[s];
    float fst = __ll2float_rn(st);
    out.cx[s] = __fdiv_rn(__ll2float_rn(sx), fst);
    out.cy[s] = __fdiv_rn(__ll2float_rn(sy), fst);
    out.ctof[s] = __fdiv_rn(__ll2float_rn(out.sum_tot_tof[s]), fst);
    if (lbase) out.label[s] += lbase;     // after the reads of out.label above
  }
}

}  // namespace tpx3
