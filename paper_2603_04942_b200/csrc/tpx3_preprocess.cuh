// Preprocessing (section IV.B-C, :66-76), event by event in the paper's order:
//   shot    the most recent laser trigger: the largest s with trig[s] <= ToA; an event
//           before the first trigger has none and is dropped
//   cut     ToF = ToA - trig[s]; kept "only ... if its ToF does not exceed 100 us" (:68): ToF <= cut
//   walk    ToF' = ToF - dToF(ToT), dToF = Eq. 1 (:74) as a calibrated integer table in ticks (a ToT beyond
//           the table uses its last entry), clamped to [0, P - 1] (R23)
//   rebase  ToA' = (shot_base + s) * P + ToF': downstream `shot = ToA' div P` is the trigger index (R6)
// Kept events stay in stream order (an order-preserving stream compaction):
//   k_pre_mark     kept / dropped per event (trigger lookup: 64 triggers around the block's first event in
//                  shared memory, binary search in the L2-resident list otherwise), kept per block; reads ToA only
//   k_pre_scan     exclusive scan of the block counts (one block); total -> n_out
//   k_pre_scatter  ToA' again (striped, coalesced), in-block ranks in stream order through shared memory,
//                  striped coalesced copies of x, y, ToT, ToA' and the input index
#pragma once
#include "tpx3_centroid.cuh"
#include "tpx3_common.cuh"

namespace tpx3 {

constexpr int kPreThreads = 512;
constexpr int kPreItems = 8;
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
  uint32_t* blk;
  uint32_t nblk;
};

constexpr int kPreWin = 64;   // triggers of the block's neighbourhood held in shared memory

// The block's window of the trigger list: trig[h0 .. h0 + valid), h0 a few triggers before the most recent
// trigger of the block's first event (the stream is close to time order, so nearly every event of the block
// finds its trigger inside the window; the rest take the binary search in global memory).
struct PreWindow {
  uint64_t trig[kPreWin];
  uint64_t h0;
  uint32_t valid;
};

__device__ __forceinline__ uint64_t pre_search(const PreArgs& a, uint64_t t) {   // first trigger later than t
  uint64_t lo = 0, hi = a.n_trig;
  while (lo < hi) {
    const uint64_t mid = (lo + hi) >> 1;
    if (a.trig[mid] <= t) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// Every thread of the block must call this. The position of the block's first event in the trigger list is
// found by the whole block in two rounds of loads (every stride-th trigger, then the stride that holds it)
// instead of 17 dependent steps of one thread; a list too long for that (more than blockDim^2 triggers)
// finishes the second round with a binary search.
__device__ __forceinline__ void pre_window_fill(const PreArgs& a, uint64_t k_first, PreWindow* w) {
  const uint64_t nt = a.n_trig;
  uint64_t lo = 0;                                   // first trigger later than the block's first event
  if (k_first < a.n && nt) {                         // block-uniform
    const uint64_t t0 = a.toa[k_first];
    const uint64_t stride = (nt + blockDim.x - 1) / blockDim.x;
    const uint64_t p1 = (uint64_t)threadIdx.x * stride;
    const int c1 = __syncthreads_count(p1 < nt && a.trig[p1] <= t0);      // trig ascending: a prefix of the threads
    if (c1) {
      const uint64_t seg = (uint64_t)(c1 - 1) * stride;
      if (stride <= blockDim.x) {
        const uint64_t p2 = seg + threadIdx.x;
        const int c2 = __syncthreads_count(threadIdx.x < stride && p2 < nt && a.trig[p2] <= t0);
        lo = seg + (uint64_t)c2;
      } else {
        uint64_t l = seg, h = seg + stride < nt ? seg + stride : nt;
        while (l < h) {
          const uint64_t mid = (l + h) >> 1;
          if (a.trig[mid] <= t0) l = mid + 1; else h = mid;
        }
        lo = l;
      }
    }
  }
  if (threadIdx.x == 0) {
    const uint64_t h0 = lo > 9 ? lo - 9 : 0ull;
    w->h0 = h0;
    w->valid = (uint32_t)(nt - h0 < (uint64_t)kPreWin ? nt - h0 : (uint64_t)kPreWin);
  }
  __syncthreads();
  if (threadIdx.x < kPreWin) w->trig[threadIdx.x] = threadIdx.x < w->valid ? a.trig[w->h0 + threadIdx.x] : ~0ull;
  __syncthreads();
}

// Index of the most recent trigger (largest s with trig[s] <= t), or false if there is none. Exact for any
// input: the window only answers when t lies strictly inside it.
__device__ __forceinline__ bool pre_find(const PreArgs& a, const PreWindow* w, uint64_t t, uint64_t& s) {
  const uint32_t valid = w->valid;
  if (valid >= 2 && t >= w->trig[0] && t < w->trig[valid - 1]) {
    uint32_t lo = 0;                      // largest j with trig[j] <= t, j in [0, valid - 1)
#pragma unroll
    for (uint32_t step = kPreWin / 2; step; step >>= 1)
      if (lo + step < valid && w->trig[lo + step] <= t) lo += step;
    s = w->h0 + lo;
    return true;
  }
  const uint64_t lo = pre_search(a, t);
  if (lo == 0) return false;
  s = lo - 1;
  return true;
}

// ToA' of event k, or kPreDropped (no trigger yet, or ToF beyond the cut).
__device__ __forceinline__ uint64_t pre_event(const PreArgs& a, const PreWindow* w, uint64_t t, uint32_t tt,
                                              bool with_tot) {
  uint64_t s = 0;
  if (!pre_find(a, w, t, s)) return kPreDropped;
  const uint64_t tof = t - a.trig[s];
  if (tof > a.cut) return kPreDropped;
  if (!with_tot) return 0ull;            // the mark pass only needs kept / dropped
  long long corr = 0;
  if (a.table_len) corr = a.table[tt < a.table_len ? tt : a.table_len - 1u];
  long long tc = (long long)tof - corr;   // tof <= cut < 2^63
  if (tc < 0) tc = 0;
  if ((uint64_t)tc > a.P - 1ull) tc = (long long)(a.P - 1ull);
  return (a.shot_base + s) * a.P + (uint64_t)tc;
}

__global__ void __launch_bounds__(kPreThreads) k_pre_mark(PreArgs a) {
  __shared__ uint32_t s_cnt;
  __shared__ PreWindow s_win;
  const uint64_t base = (uint64_t)blockIdx.x * kPreTile;
  if (threadIdx.x == 0) s_cnt = 0;
  pre_window_fill(a, base, &s_win);
  uint32_t cnt = 0;
  uint64_t t[kPreItems];
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {      // all loads first: independent and coalesced
    const uint64_t k = base + (uint64_t)i * kPreThreads + threadIdx.x;
    t[i] = k < a.n ? a.toa[k] : 0ull;
  }
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {
    const uint64_t k = base + (uint64_t)i * kPreThreads + threadIdx.x;
    if (k < a.n) cnt += pre_event(a, &s_win, t[i], 0u, false) != kPreDropped;
  }
  cnt = __reduce_add_sync(0xffffffffu, cnt);
  if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&s_cnt, cnt);
  __syncthreads();
  if (threadIdx.x == 0) a.blk[blockIdx.x] = s_cnt;
}

// Fused route (tpx3_preprocess_cluster_centroid): the tile kernel drops events in its load phase, so all it needs
// from a pre-pass is the number of SURVIVING events in front of every segment of G events (its sorted positions
// count only those). Block g counts segment g, 4096 events at a time; reads ToA only, like k_pre_mark.
__global__ void __launch_bounds__(kPreThreads) k_pre_seg_count(PreArgs a, uint32_t G, uint32_t* seg_kept) {
  __shared__ uint32_t s_cnt;
  __shared__ PreWindow s_win;
  const uint64_t seg_begin = (uint64_t)blockIdx.x * G;
  const uint64_t seg_end = seg_begin + G < a.n ? seg_begin + G : a.n;
  if (threadIdx.x == 0) s_cnt = 0;
  uint32_t cnt = 0;
  for (uint64_t base = seg_begin; base < seg_end; base += kPreTile) {     // block-uniform trip count
    pre_window_fill(a, base, &s_win);
    uint64_t t[kPreItems];
#pragma unroll
    for (int i = 0; i < kPreItems; ++i) {
      const uint64_t k = base + (uint64_t)i * kPreThreads + threadIdx.x;
      t[i] = k < seg_end ? a.toa[k] : 0ull;
    }
#pragma unroll
    for (int i = 0; i < kPreItems; ++i) {
      const uint64_t k = base + (uint64_t)i * kPreThreads + threadIdx.x;
      if (k < seg_end) cnt += pre_event(a, &s_win, t[i], 0u, false) != kPreDropped;
    }
    __syncthreads();                                                       // the window is refilled next round
  }
  cnt = __reduce_add_sync(0xffffffffu, cnt);
  if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&s_cnt, cnt);
  __syncthreads();
  if (threadIdx.x == 0) seg_kept[blockIdx.x] = s_cnt;
}

// Exclusive scan over the segments (one block); the total is the number of surviving events.
__global__ void __launch_bounds__(1024) k_pre_seg_scan(uint32_t* seg_kept, uint32_t nseg, uint32_t* n_kept) {
  const uint32_t x = scan_inplace_1024(seg_kept, nseg);
  if (threadIdx.x == 0) *n_kept = x;
}

__global__ void __launch_bounds__(1024) k_pre_scan(PreArgs a) {
  const uint32_t x = scan_inplace_1024(a.blk, a.nblk);
  if (threadIdx.x == 0) *a.n_out = x;
}

__global__ void __launch_bounds__(kPreThreads, 3) k_pre_scatter(PreArgs a) {
  __shared__ __align__(16) uint8_t s_keep[kPreTile];
  __shared__ uint16_t s_rank[kPreTile];
  __shared__ uint32_t sm[33];
  __shared__ PreWindow s_win;
  const uint64_t base = (uint64_t)blockIdx.x * kPreTile;
  pre_window_fill(a, base, &s_win);
  // striped (coalesced) pass: ToA' of every event
  uint64_t v[kPreItems];
  uint16_t tt[kPreItems];
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {      // all loads first: independent and coalesced
    const uint64_t k = base + (uint64_t)i * kPreThreads + threadIdx.x;
    v[i] = k < a.n ? a.toa[k] : 0ull;
    tt[i] = k < a.n ? a.tot[k] : (uint16_t)0;
  }
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {
    const uint32_t loc = (uint32_t)i * kPreThreads + threadIdx.x;
    const uint64_t k = base + loc;
    v[i] = k < a.n ? pre_event(a, &s_win, v[i], tt[i], true) : kPreDropped;
    s_keep[loc] = v[i] != kPreDropped;
  }
  __syncthreads();
  // blocked pass over the flags: a thread owns 8 consecutive events, so ranks follow the stream order
  static_assert(kPreItems == 8, "one 8-byte load of flags per thread");
  const uint2 q = *reinterpret_cast<const uint2*>(&s_keep[threadIdx.x * kPreItems]);
  const uint32_t qw[2] = {q.x, q.y};
  const uint32_t cnt = __popc(q.x) + __popc(q.y);
  uint32_t off = block_exclusive_scan_256(cnt, sm, nullptr);
#pragma unroll
  for (int j = 0; j < kPreItems; ++j)
    if ((qw[j >> 2] >> (8 * (j & 3))) & 1u) s_rank[threadIdx.x * kPreItems + j] = (uint16_t)off++;
  __syncthreads();
  // striped pass again: neighbouring threads hold neighbouring ranks, so the copies are coalesced
  const uint32_t blk_off = a.blk[blockIdx.x];
  // all loads before the first store (the compiler cannot prove that the outputs do not alias the inputs)
  uint32_t exy[kPreItems];
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {
    const uint64_t k = base + (uint32_t)i * kPreThreads + threadIdx.x;
    exy[i] = v[i] != kPreDropped ? (uint32_t)a.x[k] | ((uint32_t)a.y[k] << 16) : 0u;
  }
#pragma unroll
  for (int i = 0; i < kPreItems; ++i) {
    if (v[i] == kPreDropped) continue;
    const uint32_t loc = (uint32_t)i * kPreThreads + threadIdx.x;
    const uint64_t k = base + loc;
    const uint32_t o = blk_off + s_rank[loc];
    a.x_out[o] = (uint16_t)exy[i];
    a.y_out[o] = (uint16_t)(exy[i] >> 16);
    a.tot_out[o] = tt[i];
    a.toa_out[o] = v[i];
    if (a.index_out) a.index_out[o] = (uint32_t)k;
  }
}

}  // namespace tpx3
