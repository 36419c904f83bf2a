// Internal definitions shared by the kernels of libtpx3 (sm_100a). Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpx3.h"

namespace tpx3 {

constexpr int kNumSMs = 148;               // B200; sizes compile-time tables only (the plan reads the device's count)
constexpr uint32_t kEmpty = 0xFFFFFFFFu;   // empty hash slot / "no hit"
constexpr uint64_t kMaxHits = 1ull << 28;  // sorted index fits 28 bits

// Device-resident control block at the start of the workspace.
struct Ctrl {
  tpx3_status_t status;          // error, path, n_clusters, sort_passes, n
  unsigned long long toa_min;    // general path: min / max ToA of the call
  unsigned long long toa_max;
  uint32_t npass;                // general path: radix passes to run (>= 1)
  uint32_t fused_state;          // 0 = not attempted, 1 = succeeded, 2 = failed (general path must run)
  uint32_t tile_ticket;          // fused path: dynamic tile counter
  uint32_t n_roots;              // scratch root counter
  uint32_t tiles_done;           // fused path: tiles finished
  uint32_t fused_fail;           // fused path: some tile could not be handled
  uint32_t tight_tiles;          // fused path: tiles of this call whose time clusters were all tight
  uint32_t tiles_run;            // fused path: tiles of this call that owned events
  // Kept ACROSS calls on the same workspace (never reset; any garbage is a legal value: it only steers which of
  // two exact code paths a tile takes). A stream keeps its character from chunk to chunk: when hardly any tile
  // of a call had tight time clusters, the tiles of the next calls skip the check (and retry every 16th call).
  uint32_t scan_hint;            // kScanSkip: the last call found the time-cluster check not worth its cost
  uint32_t calls;                // fused calls served on this workspace
  uint32_t sort_packed;          // general sort of this call: key and index travel in one 64-bit word (tpx3_sort.cuh)
};
constexpr uint32_t kScanSkip = 0x5C1Fu;
static_assert(sizeof(Ctrl) <= 256, "Ctrl must fit the 256-byte workspace header");

// Parameters every kernel needs (passed by value).
struct Params {
  uint64_t n;
  uint64_t P;        // shot period (0 = one shot)
  uint32_t W;        // ToA window, inclusive
  uint32_t sensor_w, sensor_h;
  uint32_t flags;
  uint64_t slabs_per_shot_p1;  // ceil(P / (W+1)) + 1 (general path slab numbering), 0 if P == 0
};

__device__ __forceinline__ void set_error(Ctrl* c, int err) {
  atomicCAS(&c->status.error, 0u, (uint32_t)(-err));
}

__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// 64-bit unsigned atomic min / max on global memory.
__device__ __forceinline__ void atomic_min_u64(unsigned long long* p, unsigned long long v) { atomicMin(p, v); }
__device__ __forceinline__ void atomic_max_u64(unsigned long long* p, unsigned long long v) { atomicMax(p, v); }

// Exclusive prefix sum of v[0..n) in place by ONE block of 1024 threads (each thread owns a contiguous
// run). Returns the total, the same value in every thread. Sums are taken modulo 2^32, so two's-complement
// signed counts scan correctly too.
__device__ __forceinline__ uint32_t scan_inplace_1024(uint32_t* v, uint32_t n) {
  __shared__ uint32_t s_warp[33];
  const uint32_t per = (n + 1023u) / 1024u;
  uint32_t beg = threadIdx.x * per, end = beg + per;
  if (beg > n) beg = n;
  if (end > n) end = n;
  uint32_t s = 0;
  for (uint32_t i = beg; i < end; ++i) s += v[i];
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  uint32_t inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= (uint32_t)o) inc += t;
  }
  if (lane == 31u) s_warp[w] = inc;
  __syncthreads();
  if (w == 0) {
    const uint32_t ws = s_warp[lane];
    uint32_t x = ws;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= (uint32_t)o) x += t;
    }
    s_warp[lane] = x - ws;
    if (lane == 31u) s_warp[32] = x;
  }
  __syncthreads();
  uint32_t run = s_warp[w] + inc - s;
  for (uint32_t i = beg; i < end; ++i) {
    const uint32_t t = v[i];
    v[i] = run;
    run += t;
  }
  return s_warp[32];
}

// Fill `n` 32-bit words (general_only: skipped when the fused path already succeeded).
__global__ void __launch_bounds__(256) k_fill_u32(Ctrl* c, int general_only, uint32_t* p, uint64_t n, uint32_t v) {
  if (general_only && c->fused_state == 1) return;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
    p[i] = v;
}

}  // namespace tpx3
