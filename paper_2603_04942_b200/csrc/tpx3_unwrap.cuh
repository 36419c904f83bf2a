// ToA counter unwrapping (section IV.A, :58-62).
//
// The TimePix3 ToA is a counter of 42 bits (pixels) or 44 bits (TDC triggers) that wraps every 26.8 s /
// 107.4 s. The paper's rule, a sequential scan: "Each time the ToA of the next pixel or TDC
// is more than 20 seconds less than the previous one, the global counter of time wrappings is incremented
// by one and the appropriate integer multiple ... is added to all subsequent data" (:60); and for pixels
// reported out of order across a wrap: "both large negative and large positive jumps are tracked ... and
// the appropriate time unwrapping adjustment is applied in each case" (:62) — a jump UP by more than the
// threshold takes the counter back down by one (R22).
//
// The counter after event i is therefore wraps_in + sum_{k <= i} d_k with d_k in {+1, 0, -1} decided by the
// ADJACENT difference raw[k] - raw[k-1] alone: a prefix sum, not a sequential dependence.
//   k_unwrap_count   d_k summed per block of 4096 events
//   k_unwrap_scan    exclusive scan of the block sums (one block); total -> wraps_out
//   k_unwrap_apply   in-block scan (ballots per 32-event row), toa[i] = raw[i] + wraps_i * modulus
#pragma once
#include "tpx3_centroid.cuh"
#include "tpx3_common.cuh"

namespace tpx3 {

constexpr int kUnwrapThreads = 512;
constexpr int kUnwrapItems = 8;
constexpr int kUnwrapTile = kUnwrapThreads * kUnwrapItems;   // 4096 events per block

struct UnwrapArgs {
  uint64_t n;
  const uint64_t* raw;
  uint64_t modulus, jump;
  long long wraps_in;
  int has_prev;
  uint64_t prev_raw;
  uint64_t* out;
  long long* wraps_out;
  uint32_t* blk;       // block sums (two's complement)
  uint32_t nblk;
};

// +1: the counter wrapped between p and v; -1: v is a pre-wrap value reported after the wrap (or the way back)
__device__ __forceinline__ int unwrap_delta(uint64_t p, uint64_t v, uint64_t jump) {
  if (p > v) return p - v > jump ? 1 : 0;
  return v - p > jump ? -1 : 0;
}

__device__ __forceinline__ int unwrap_delta_at(const UnwrapArgs& a, uint64_t i) {
  if (i == 0) return a.has_prev ? unwrap_delta(a.prev_raw, a.raw[0], a.jump) : 0;
  return unwrap_delta(a.raw[i - 1], a.raw[i], a.jump);
}

__global__ void __launch_bounds__(kUnwrapThreads) k_unwrap_count(UnwrapArgs a) {
  __shared__ uint32_t sm[33];
  const uint64_t base = (uint64_t)blockIdx.x * kUnwrapTile;
  int s = 0;
  uint64_t v[kUnwrapItems];
#pragma unroll
  for (int i = 0; i < kUnwrapItems; ++i) {      // all loads first
    const uint64_t k = base + (uint64_t)i * kUnwrapThreads + threadIdx.x;
    v[i] = k < a.n ? a.raw[k] : 0ull;
  }
#pragma unroll
  for (int i = 0; i < kUnwrapItems; ++i) {
    const uint64_t k = base + (uint64_t)i * kUnwrapThreads + threadIdx.x;
    // the predecessor is the neighbouring lane's value; lane 0 reads it (the previous warp's line, an L1 / L2 hit)
    uint64_t p = __shfl_up_sync(0xffffffffu, v[i], 1);
    if (k < a.n) {
      if ((threadIdx.x & 31) == 0) s += unwrap_delta_at(a, k);
      else s += unwrap_delta(p, v[i], a.jump);
    }
  }
  uint32_t total;
  block_exclusive_scan_256((uint32_t)s, sm, &total);
  if (threadIdx.x == 0) a.blk[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) k_unwrap_scan(UnwrapArgs a) {
  const uint32_t x = scan_inplace_1024(a.blk, a.nblk);
  if (threadIdx.x == 0) *a.wraps_out = a.wraps_in + (long long)(int)x;
}

// A warp owns 256 consecutive events and walks them in 8 rows of 32 (coalesced 256-byte rows). Within a row
// the running count is two ballots (+1 lanes, -1 lanes) and two popcounts; the row total carries to the next.
__global__ void __launch_bounds__(kUnwrapThreads, 3) k_unwrap_apply(UnwrapArgs a) {
  __shared__ int s_warp[kUnwrapThreads / 32];
  const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
  const uint64_t base = (uint64_t)blockIdx.x * kUnwrapTile + (uint64_t)wid * (32 * kUnwrapItems);
  const uint32_t le = 0xFFFFFFFFu >> (31u - lane);   // lanes <= this one
  uint64_t v[kUnwrapItems];
  int pre[kUnwrapItems];
  int run = 0;
  // all loads first (independent, coalesced); the predecessor of an event comes from the neighbouring lane
#pragma unroll
  for (int i = 0; i < kUnwrapItems; ++i) {
    const uint64_t k = base + (uint64_t)i * 32 + lane;
    v[i] = k < a.n ? a.raw[k] : 0ull;
  }
  uint64_t before = a.prev_raw;          // predecessor of the warp's first event
  bool have_before = a.has_prev != 0;
  if (base > 0 && base < a.n) { before = a.raw[base - 1]; have_before = true; }
#pragma unroll
  for (int i = 0; i < kUnwrapItems; ++i) {
    const uint64_t k = base + (uint64_t)i * 32 + lane;
    uint64_t p = __shfl_up_sync(0xffffffffu, v[i], 1);
    bool havep = true;
    if (lane == 0) { p = before; havep = have_before; }
    before = __shfl_sync(0xffffffffu, v[i], 31);
    have_before = true;
    const int d = (k < a.n && havep) ? unwrap_delta(p, v[i], a.jump) : 0;
    const uint32_t up = __ballot_sync(0xffffffffu, d > 0), dn = __ballot_sync(0xffffffffu, d < 0);
    pre[i] = run + __popc(up & le) - __popc(dn & le);
    run += __popc(up) - __popc(dn);
  }
  if (lane == 0) s_warp[wid] = run;
  __syncthreads();
  int off = (int)a.blk[blockIdx.x];
  for (uint32_t w2 = 0; w2 < wid; ++w2) off += s_warp[w2];
#pragma unroll
  for (int i = 0; i < kUnwrapItems; ++i) {
    const uint64_t k = base + (uint64_t)i * 32 + lane;
    if (k < a.n) {
      const long long wraps = a.wraps_in + (long long)(off + pre[i]);
      a.out[k] = v[i] + (uint64_t)wraps * a.modulus;   // two's complement: a negative count subtracts
    }
  }
}

}  // namespace tpx3
