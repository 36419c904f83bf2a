// Preprocessing (section IV.B-C, :66-76), event by event in the paper's order:
//   shot    the most recent laser trigger: the largest s with trig[s] <= ToA; an event
//           before the first trigger has none and is dropped
//   cut     ToF = ToA - trig[s]; kept "only ... if its ToF does not exceed 100 us" (:68): ToF <= cut
//   walk    ToF' = ToF - dToF(ToT), dToF = Eq. 1 (:74) as a calibrated integer table in ticks (a ToT beyond
//           the table uses its last entry), clamped to [0, P - 1] (R23)
//   rebase  ToA' = (shot_base + s) * P + ToF': downstream `shot = ToA' div P` is the trigger index (R6)
// Kept events stay in stream order (an order-preserving stream compaction):
//   k_pre_mark     ToA' or "dropped" per event (binary search in the trigger list, L2-resident), kept per block
//   k_pre_scan     exclusive scan of the block counts (one block); total -> n_out
//   k_pre_scatter  in-block ranks in stream order, coalesced copies of x, y, ToT, ToA' and the input index
#pragma once
#include "tpx3_centroid.cuh"
#include "tpx3_common.cuh"

namespace tpx3 {

constexpr int kPreThreads = 256;
constexpr int kPreItems = 16;
constexpr int kPreTile = kPreThreads * kPreItems;   // 4096 events per block
constexpr uint64_t kPreDropped = ~0ull;

struct PreArgs {
  uint64_t n;
  const uint16_t *x, *y, *tot;
  const uint64_t* toa;
  uint64_t n_trig;
  const uint64_t* trig;
  uint64_t cut, P, shot_base;
  const int32_t* table;
  uint32_t table_len;
  uint16_t *x_out, *y_out, *tot_out;
  uint64_t* toa_out;
  uint32_t* index_out;   // may be null
  uint32_t* n_out;
  uint64_t* tmp;         // ToA' or kPreDropped per event
  uint32_t* blk;
  uint32_t nblk;
};

__device__ __forceinline__ uint64_t pre_event(const PreArgs& a, uint64_t k) {
  const uint64_t t = a.toa[k];
  uint64_t lo = 0, hi = a.n_trig;       // first trigger later than t
  while (lo < hi) {
    const uint64_t mid = (lo + hi) >> 1;
    if (a.trig[mid] <= t) lo = mid + 1; else hi = mid;
  }
  if (lo == 0) return kPreDropped;
  const uint64_t s = lo - 1;
  const uint64_t tof = t - a.trig[s];
  if (tof > a.cut) return kPreDropped;
  long long corr = 0;
  if (a.table_len) {
    const uint32_t tt = a.tot[k];
    corr = a.table[tt < a.table_len ? tt : a.table_len - 1u];
  }
  long long tc = (long long)tof - corr;   // tof <= cut < 2^63
  if (tc < 0) tc = 0;
  if ((uint64_t)tc > a.P - 1ull) tc = (long long)(a.P - 1ull);
  return (a.shot_base + s) * a.P + (uint64_t)tc;
}

__global__ void __launch_bounds__(kPreThreads) k_pre_mark(PreArgs a) {
  __shared__ uint32_t sm[33];
  const uint64_t base = (uint64_t)blockIdx.x * kPreTile;
  uint32_t cnt = 0;
#pragma unroll 2
  for (int i = 0; i < kPreItems; ++i) {
    const uint64_t k = base + (uint64_t)i * kPreThreads + threadIdx.x;
    if (k < a.n) {
      const uint64_t v = pre_event(a, k);
      a.tmp[k] = v;
      cnt += v != kPreDropped;
    }
  }
  uint32_t total;
  block_exclusive_scan_256(cnt, sm, &total);
  if (threadIdx.x == 0) a.blk[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) k_pre_scan(PreArgs a) {
  const uint32_t x = scan_inplace_1024(a.blk, a.nblk);
  if (threadIdx.x == 0) *a.n_out = x;
}

__global__ void __launch_bounds__(kPreThreads) k_pre_scatter(PreArgs a) {
  __shared__ uint32_t sm[33];
  // blocked arrangement: a thread owns 16 consecutive events, so ranks follow the stream order
  const uint64_t base = (uint64_t)blockIdx.x * kPreTile + (uint64_t)threadIdx.x * kPreItems;
  uint64_t v[kPreItems];
  uint32_t cnt = 0;
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {
    const uint64_t k = base + i;
    v[i] = k < a.n ? a.tmp[k] : kPreDropped;
    cnt += v[i] != kPreDropped;
  }
  uint32_t off = block_exclusive_scan_256(cnt, sm, nullptr) + a.blk[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {
    if (v[i] != kPreDropped) {
      const uint64_t k = base + i;
      a.x_out[off] = a.x[k];
      a.y_out[off] = a.y[k];
      a.tot_out[off] = a.tot[k];
      a.toa_out[off] = v[i];
      if (a.index_out) a.index_out[off] = (uint32_t)k;
      ++off;
    }
  }
}

}  // namespace tpx3
