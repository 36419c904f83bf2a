// General path, S0/S1: stable LSD radix sort of the events by ToA (key = ToA - min ToA; the
// (shot, ToA) order of the contract is the ToA order because shot = ToA div P is monotone in
// ToA — SURVEY.md §8a S0). 8-bit digits; the number of passes is decided on the
// device from the key span, so no host synchronisation is needed: every pass is enqueued and
// the ones past `npass` return immediately.
//
// Per pass: digit histogram per block -> exclusive scan (digit-major) -> stable scatter.
// Packed mode (key span <= 36 bits, the usual case: 2^36 ticks = 107 s of data): key and input position travel
// as ONE 64-bit word (ToA - min) << 28 | position (a plan takes at most 2^28 events), 8 instead of 12 bytes per
// key and pass, and the scatter (k_radix_scatter_packed) orders a tile of 4096 keys in shared memory first, so
// that consecutive threads write consecutive addresses of a digit's run. The last pass writes the plain key and
// perm, so everything behind the sort sees the same buffers in both modes.
// Stability inside a tile comes from warp-ordered ranking with __match_any_sync (each warp owns
// a contiguous slice of the tile; items are visited in ascending position).
#pragma once
#include "tpx3_common.cuh"

namespace tpx3 {

constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortItems = 8;                               // per thread per tile
constexpr int kSortTile = kSortThreads * kSortItems;        // 2048
constexpr int kSortMaxBlocks = kNumSMs * 8;                 // 1184 (one wave of 740 for the packed scatter, 5 blocks per SM: 3 % slower)
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kMaxPasses = 8;

struct SortGeom {
  uint32_t nblk;            // blocks
  uint32_t tiles_per_blk;   // tiles each block walks sequentially
};

__host__ __device__ inline SortGeom sort_geom(uint64_t n) {
  uint64_t tiles = (n + kSortTile - 1) / kSortTile;
  SortGeom g;
  g.nblk = (uint32_t)(tiles < (uint64_t)kSortMaxBlocks ? (tiles ? tiles : 1) : kSortMaxBlocks);
  g.tiles_per_blk = (uint32_t)((tiles + g.nblk - 1) / g.nblk);
  if (g.tiles_per_blk == 0) g.tiles_per_blk = 1;
  return g;
}

// ---- min / max ToA ------------------------------------------------------------------------
// Also clears the fused path's tile status words and the caller's hit counter.
__global__ void __launch_bounds__(256) k_ctrl_init(Ctrl* c, uint64_t n, unsigned long long* tiles, uint32_t num_tiles,
                                                 uint32_t* n_clusters, const uint32_t* n_dev = nullptr,
                                                 const uint32_t* dead = nullptr) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    c->status.error = 0; c->status.path = 0; c->status.n_clusters = 0; c->status.sort_passes = 0;
    c->status.n = n_dev ? (uint64_t)*n_dev : n;                              // stream push: the device's count
    if (dead && *dead) c->status.error = (uint32_t)(-TPX3_ERR_CAPACITY);   // ... and a carry overflow of the stream
    c->toa_min = ~0ull; c->toa_max = 0ull; c->npass = 1; c->fused_state = 0; c->tile_ticket = 0; c->n_roots = 0;
    c->tiles_done = 0; c->fused_fail = 0; c->tight_tiles = 0; c->tiles_run = 0;
    if (n_clusters) *n_clusters = 0;
  }
  for (uint32_t t = i; t < num_tiles; t += gridDim.x * blockDim.x) tiles[t] = 0ull;
}

__global__ void __launch_bounds__(256) k_minmax(Ctrl* c, const uint64_t* __restrict__ toa, uint64_t n) {
  if (c->fused_state == 1) return;
  unsigned long long lo = ~0ull, hi = 0ull;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    unsigned long long t = toa[i];
    lo = t < lo ? t : lo;
    hi = t > hi ? t : hi;
  }
  for (int o = 16; o; o >>= 1) {
    unsigned long long a = __shfl_xor_sync(0xffffffffu, lo, o), b = __shfl_xor_sync(0xffffffffu, hi, o);
    lo = a < lo ? a : lo;
    hi = b > hi ? b : hi;
  }
  if ((threadIdx.x & 31) == 0) { atomic_min_u64(&c->toa_min, lo); atomic_max_u64(&c->toa_max, hi); }
}

__global__ void k_sort_setup(Ctrl* c) {
  if (c->fused_state == 1) return;
  unsigned long long span = c->toa_max >= c->toa_min ? c->toa_max - c->toa_min : 0ull;
  int bits = span ? 64 - __clzll((long long)span) : 1;
  uint32_t np = (uint32_t)((bits + kRadixBits - 1) / kRadixBits);
  c->npass = np ? np : 1;
  c->sort_packed = bits <= 36 ? 1u : 0u;
  c->status.sort_passes = c->npass;
  c->status.path = 2;
}

// ---- one radix pass -----------------------------------------------------------------------
// Source of pass p: p == 0 reads ToA (key = toa - min, idx = position); p >= 1 reads key/idx
// buffer (p-1)&1. Destination: key buffer p&1; idx buffer p&1, or `perm` on the last pass.
struct SortBufs {
  uint64_t* key[2];
  uint32_t* idx[2];
  uint32_t* counts;   // [kRadix][nblk]
};

__device__ __forceinline__ uint64_t sort_load_key(int pass, const Ctrl* c, const uint64_t* toa, const SortBufs& b, uint64_t i) {
  return pass == 0 ? toa[i] - c->toa_min : b.key[(pass - 1) & 1][i];
}

__global__ void __launch_bounds__(kSortThreads) k_radix_hist(Ctrl* c, int pass, const uint64_t* __restrict__ toa,
                                                           SortBufs b, uint64_t n, SortGeom g) {
  if (c->fused_state == 1 || (uint32_t)pass >= c->npass) return;
  __shared__ uint32_t hist[kRadix];
  hist[threadIdx.x] = 0;
  __syncthreads();
  // (packed mode: from pass 1 on the source holds (ToA - min) << 28 | position)
  const int shift = pass * kRadixBits + (c->sort_packed && pass > 0 ? 28 : 0);
  uint64_t t0 = (uint64_t)blockIdx.x * g.tiles_per_blk * kSortTile;
  uint64_t t1 = t0 + (uint64_t)g.tiles_per_blk * kSortTile;
  if (t1 > n) t1 = n;
  for (uint64_t i = t0 + threadIdx.x; i < t1; i += kSortThreads) {
    uint64_t k = sort_load_key(pass, c, toa, b, i);
    const uint32_t d = (uint32_t)(k >> shift) & (kRadix - 1);
    // the high digits of a time-ordered stream are the same across a warp: one add instead of 32 serialised ones
    const uint32_t act = __activemask();
    const uint32_t d0 = __shfl_sync(act, d, __ffs(act) - 1);
    if (__all_sync(act, d == d0)) {
      if ((threadIdx.x & 31) == (uint32_t)(__ffs(act) - 1)) atomicAdd(&hist[d], (uint32_t)__popc(act));
    } else {
      atomicAdd(&hist[d], 1u);
    }
  }
  __syncthreads();
  b.counts[(size_t)threadIdx.x * g.nblk + blockIdx.x] = hist[threadIdx.x];
}

// Exclusive scan of counts[kRadix][nblk] in place, digit by digit: one warp per digit value (32 blocks of 8 warps)
// scans that digit's nblk block counts and leaves the digit's total in counts[kRadix * nblk + d]; the scatter
// kernel adds the exclusive prefix over the 256 totals itself. (One block scanning all 303 K counters took
// 0.33 ms per pass on cfg1, as much as the histogram and half of the scatter.)
__global__ void __launch_bounds__(256) k_radix_scan(Ctrl* c, int pass, uint32_t* counts, uint32_t nblk) {
  if (c->fused_state == 1 || (uint32_t)pass >= c->npass) return;
  const uint32_t lane = threadIdx.x & 31u, d = blockIdx.x * 8u + (threadIdx.x >> 5);
  if (d >= (uint32_t)kRadix) return;
  uint32_t* row = counts + (size_t)d * nblk;
  uint32_t run = 0;
  for (uint32_t b0 = 0; b0 < nblk; b0 += 32u) {
    const uint32_t b = b0 + lane;
    const uint32_t v = b < nblk ? row[b] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (uint32_t)o) inc += t;
    }
    if (b < nblk) row[b] = run + inc - v;
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  if (lane == 0) counts[(size_t)kRadix * nblk + d] = run;
}

__global__ void __launch_bounds__(kSortThreads) k_radix_scatter(Ctrl* c, int pass, const uint64_t* __restrict__ toa,
                                                              SortBufs b, uint32_t* __restrict__ perm, uint64_t n,
                                                              SortGeom g) {
  if (c->fused_state == 1 || (uint32_t)pass >= c->npass || c->sort_packed) return;
  __shared__ uint32_t running[kRadix];
  __shared__ uint32_t warp_cnt[kSortWarps][kRadix];
  const int shift = pass * kRadixBits;
  const bool last = (uint32_t)pass + 1 == c->npass;
  uint64_t* __restrict__ dkey = b.key[pass & 1];
  uint32_t* __restrict__ didx = last ? perm : b.idx[pass & 1];
  const uint32_t* __restrict__ sidx = pass == 0 ? nullptr : b.idx[(pass - 1) & 1];
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5, lt = lanemask_lt();
  {   // exclusive prefix over the 256 digit totals (thread d = digit d), plus this block's offset inside the digit
    const uint32_t tot_d = b.counts[(size_t)kRadix * g.nblk + threadIdx.x];
    uint32_t inc = tot_d;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (uint32_t)o) inc += t;
    }
    __shared__ uint32_t wtot[kSortWarps];
    if (lane == 31) wtot[w] = inc;
    __syncthreads();
    uint32_t base = inc - tot_d;
    for (uint32_t ww = 0; ww < w; ++ww) base += wtot[ww];
    running[threadIdx.x] = base + b.counts[(size_t)threadIdx.x * g.nblk + blockIdx.x];
  }
  uint64_t t0 = (uint64_t)blockIdx.x * g.tiles_per_blk * kSortTile;
  for (uint32_t t = 0; t < g.tiles_per_blk; ++t, t0 += kSortTile) {
    if (t0 >= n) break;
    for (int i = threadIdx.x; i < kSortWarps * kRadix; i += kSortThreads) (&warp_cnt[0][0])[i] = 0;
    __syncthreads();
    uint64_t key[kSortItems];
    uint32_t rank[kSortItems];
    const uint64_t wbase = t0 + (uint64_t)w * (32 * kSortItems) + lane;
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
      uint64_t pos = wbase + (uint64_t)i * 32;
      bool valid = pos < n;
      key[i] = valid ? sort_load_key(pass, c, toa, b, pos) : 0;
      uint32_t d = valid ? ((uint32_t)(key[i] >> shift) & (kRadix - 1)) : (uint32_t)kRadix;
      // lanes holding the same digit: one ballot per digit bit (match.any is far dearer on sm_100)
      uint32_t peers = __ballot_sync(0xffffffffu, valid);
      if (!valid) peers = ~peers;
#pragma unroll
      for (int bit = 0; bit < kRadixBits; ++bit) {
        const bool one = (d >> bit) & 1u;
        const uint32_t bal = __ballot_sync(0xffffffffu, one);
        peers &= one ? bal : ~bal;
      }
      uint32_t lr = __popc(peers & lt);
      uint32_t base = valid ? warp_cnt[w][d] : 0;
      __syncwarp();
      if (valid && lr == 0) warp_cnt[w][d] = base + __popc(peers);
      __syncwarp();
      rank[i] = base + lr;
    }
    __syncthreads();
    {  // thread d: exclusive prefix over warps, seeded with the block's running global offset
      uint32_t d = threadIdx.x, run = running[d];
#pragma unroll
      for (int ww = 0; ww < kSortWarps; ++ww) {
        uint32_t cnt = warp_cnt[ww][d];
        warp_cnt[ww][d] = run;
        run += cnt;
      }
      running[d] = run;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
      uint64_t pos = wbase + (uint64_t)i * 32;
      if (pos < n) {
        uint32_t d = (uint32_t)(key[i] >> shift) & (kRadix - 1);
        uint32_t dst = warp_cnt[w][d] + rank[i];
        dkey[dst] = key[i];
        didx[dst] = pass == 0 ? (uint32_t)pos : sidx[pos];
      }
    }
    __syncthreads();
  }
}

// ---- packed mode: one pass of the scatter ---------------------------------------------------------------------
// A block walks the same key range as in k_radix_hist (so the scanned counts are its offsets), 4096 keys at a
// time: ranks inside the tile by warp ballots (warp w owns the tile's w-th slice of 512 keys, visited in ascending
// position: stable), the tile ordered by digit in shared memory, then written out run by run, coalesced.
constexpr int kPackItems = 16;
constexpr int kPackTile = kSortThreads * kPackItems;   // 4096
static_assert(kPackTile % kSortTile == 0, "a block's key range is a multiple of the histogram's tile");

__global__ void __launch_bounds__(kSortThreads, 4) k_radix_scatter_packed(Ctrl* c, int pass, const uint64_t* __restrict__ toa,
                                                                     SortBufs b, uint32_t* __restrict__ perm, uint64_t n,
                                                                     SortGeom g) {
  if (c->fused_state == 1 || (uint32_t)pass >= c->npass || !c->sort_packed) return;
  __shared__ uint64_t stage[kPackTile];                 // 32 KB: the tile in digit order
  __shared__ uint32_t running[kRadix];                  // global offset of the block's next key per digit
  __shared__ uint32_t warp_cnt[kSortWarps][kRadix];     // per warp and digit: count, then tile-local offset
  __shared__ uint32_t dig_base[kRadix + 1];             // tile-local start of a digit's run
  __shared__ uint32_t wtot[kSortWarps];
  const int shift = pass * kRadixBits + 28;             // digit of the PACKED word
  const bool last = (uint32_t)pass + 1 == c->npass;
  const uint64_t tmin = c->toa_min;
  const uint64_t* __restrict__ skey = pass == 0 ? nullptr : b.key[(pass - 1) & 1];
  uint64_t* __restrict__ dkey = b.key[pass & 1];
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5, lt = lanemask_lt();
  auto block_scan256 = [&](uint32_t v) -> uint32_t {    // exclusive prefix over the 256 threads' values
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (uint32_t)o) inc += t;
    }
    __syncthreads();                                    // wtot of the previous use has been read
    if (lane == 31) wtot[w] = inc;
    __syncthreads();
    uint32_t base = inc - v;
    for (uint32_t ww = 0; ww < w; ++ww) base += wtot[ww];
    return base;
  };
  {   // exclusive prefix over the 256 digit totals (thread d = digit d), plus this block's offset inside the digit
    const uint32_t tot_d = b.counts[(size_t)kRadix * g.nblk + threadIdx.x];
    running[threadIdx.x] = block_scan256(tot_d) + b.counts[(size_t)threadIdx.x * g.nblk + blockIdx.x];
  }
  const uint64_t r0 = (uint64_t)blockIdx.x * g.tiles_per_blk * kSortTile;
  uint64_t r1 = r0 + (uint64_t)g.tiles_per_blk * kSortTile;
  if (r1 > n) r1 = n;
  for (uint64_t t0 = r0; t0 < r1; t0 += kPackTile) {
    const uint32_t cnt = r1 - t0 < (uint64_t)kPackTile ? (uint32_t)(r1 - t0) : (uint32_t)kPackTile;
    for (int i = threadIdx.x; i < kSortWarps * kRadix; i += kSortThreads) (&warp_cnt[0][0])[i] = 0;
    __syncthreads();
    uint64_t key[kPackItems];
    uint16_t rank[kPackItems];
    const uint32_t wbase = w * (32u * kPackItems) + lane;
#pragma unroll
    for (int i = 0; i < kPackItems; ++i) {              // all loads first: independent, 256 coalesced bytes per warp
      const uint32_t q = wbase + (uint32_t)i * 32u;
      key[i] = 0;
      if (q < cnt) key[i] = pass == 0 ? (((toa[t0 + q] - tmin) << 28) | (t0 + q)) : skey[t0 + q];
    }
#pragma unroll
    for (int i = 0; i < kPackItems; ++i) {
      const uint32_t q = wbase + (uint32_t)i * 32u;
      const bool valid = q < cnt;
      const uint32_t d = valid ? ((uint32_t)(key[i] >> shift) & (kRadix - 1)) : 0u;
      uint32_t peers = __ballot_sync(0xffffffffu, valid);
      if (!valid) peers = 0u;
#pragma unroll
      for (int bit = 0; bit < kRadixBits; ++bit) {
        const bool one = (d >> bit) & 1u;
        const uint32_t bal = __ballot_sync(0xffffffffu, one);
        peers &= one ? bal : ~bal;
      }
      const uint32_t lr = __popc(peers & lt);
      const uint32_t base = valid ? warp_cnt[w][d] : 0u;
      __syncwarp();
      if (valid && lr == 0) warp_cnt[w][d] = base + __popc(peers);
      __syncwarp();
      rank[i] = (uint16_t)(base + lr);
    }
    __syncthreads();
    uint32_t tot_d = 0;
    {  // thread d: exclusive prefix over the warps; then over the digits
#pragma unroll
      for (int ww = 0; ww < kSortWarps; ++ww) {
        const uint32_t cw = warp_cnt[ww][threadIdx.x];
        warp_cnt[ww][threadIdx.x] = tot_d;
        tot_d += cw;
      }
      const uint32_t db = block_scan256(tot_d);
      dig_base[threadIdx.x] = db;
      if (threadIdx.x == kRadix - 1) dig_base[kRadix] = db + tot_d;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kPackItems; ++i) {
      const uint32_t q = wbase + (uint32_t)i * 32u;
      if (q < cnt) {
        const uint32_t d = (uint32_t)(key[i] >> shift) & (kRadix - 1);
        stage[dig_base[d] + warp_cnt[w][d] + rank[i]] = key[i];
      }
    }
    __syncthreads();
    for (uint32_t q = threadIdx.x; q < cnt; q += kSortThreads) {   // consecutive q of one digit -> consecutive addresses
      const uint64_t k = stage[q];
      const uint32_t d = (uint32_t)(k >> shift) & (kRadix - 1);
      const uint32_t dst = running[d] + (q - dig_base[d]);
      if (last) { dkey[dst] = k >> 28; perm[dst] = (uint32_t)k & 0x0FFFFFFFu; }
      else dkey[dst] = k;
    }
    __syncthreads();
    running[threadIdx.x] += tot_d;
    // (the next round's first barrier orders this update before its use)
  }
}

}  // namespace tpx3
