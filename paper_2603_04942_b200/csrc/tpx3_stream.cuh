// Chunked stream with cuts that are not shot-aligned (last clause; R24).
//
// "Each pixel [is] associated with the most recent laser trigger" and no hit crosses a shot
// (R6), so a chunk of an endless stream may be cut anywhere as long as every shot is clustered in ONE piece.
// One push of a chunk:
//   k_stream_cut      t_max = max(t_max, ToA of the last 65536 events of the chunk) (atomicMax per block); with
//                     the stream's disorder bound D (pixels report out of order) every shot
//                     below s_cut = max(s_emitted, (t_max - D) div P) is complete (stream_cut, per block)
//   k_stream_mark     working set = carried events ++ chunk (stream order); per block of 4096 the number of
//                     events to emit (s_emitted <= shot < s_cut) and to carry (shot >= s_cut); the rest is late
//   k_stream_scan     exclusive scans of both counts (one block), totals and the new stream state
//   k_stream_scatter  order-preserving compaction into the emit arrays and the new carry arrays
//   k_stream_dispatch (tpx3_lib.cu, one thread) reads the emit count and launches the clustering of the emit arrays
//                     from the device (tile kernel, compaction, fallback dispatcher): the host never waits for
//                     the count. The compaction adds the events emitted by earlier pushes to the label column,
//                     so the rows continue the batch numbering.
// Shots are compared as times (t_lo = s_emitted * P <= ToA < t_cut = s_cut * P): no division per event.
#pragma once
#include "tpx3_centroid.cuh"
#include "tpx3_common.cuh"

namespace tpx3 {

constexpr int kStreamThreads = 512;
constexpr int kStreamItems = 8;
constexpr int kStreamTile = kStreamThreads * kStreamItems;   // 4096 events per block
constexpr uint32_t kStreamSample = 65536;                    // chunk tail that feeds the running maximum

struct StreamCtrl {
  uint64_t t_max;        // running maximum (a lower bound of the largest ToA seen)
  uint64_t s_emitted;    // every shot below went out
  uint64_t s_cut;        // this push
  uint64_t t_lo, t_cut;  // s_emitted * P, s_cut * P
  uint64_t label_base;   // events emitted by earlier pushes
  uint64_t label_next;   // ... including this one
  uint64_t late_total;
  uint32_t n_work, n_carry, n_late, overflow;
  uint32_t final_push, dead;   // dead: a push overflowed the carry; every later push reports TPX3_ERR_CAPACITY
  uint32_t n_carry_in, pad;    // the carry this push started with (n_carry is overwritten by its scan)
};

struct StreamArgs {
  StreamCtrl* c;
  uint64_t n;            // chunk
  uint32_t carry_cap;    // (the number of carried events is device state: c->n_carry_in)
  const uint16_t *x, *y, *tot;      // chunk
  const uint64_t* toa;
  const uint16_t *cx, *cy, *ctot;   // carried in
  const uint64_t* ctoa;
  uint16_t *nx, *ny, *ntot;         // carried out
  uint64_t* ntoa;
  uint16_t *wx, *wy, *wtot;         // emitted
  uint64_t* wtoa;
  uint32_t *blk_emit, *blk_keep;
  uint32_t nblk;
  uint64_t P, D;
  int final_push;
};

__global__ void __launch_bounds__(256) k_stream_open(StreamCtrl* c) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    c->t_max = 0; c->s_emitted = 0; c->s_cut = 0; c->t_lo = 0; c->t_cut = 0; c->label_base = 0; c->label_next = 0; c->late_total = 0;
    c->n_work = 0; c->n_carry = 0; c->n_late = 0; c->overflow = 0; c->final_push = 0; c->dead = 0; c->n_carry_in = 0; c->pad = 0;
  }
}

// Running maximum over the chunk's last kStreamSample events: 64 blocks, one atomicMax each. Also the first
// kernel of a push: records the carry the push starts with.
__global__ void __launch_bounds__(256) k_stream_cut(StreamArgs a) {
  if (blockIdx.x == 0 && threadIdx.x == 0) a.c->n_carry_in = a.c->n_carry;
  const uint64_t m = a.n < kStreamSample ? a.n : kStreamSample;
  const uint64_t beg = a.n - m;
  unsigned long long v = 0;
  for (uint64_t i = (uint64_t)blockIdx.x * 256 + threadIdx.x; i < m; i += (uint64_t)gridDim.x * 256) {
    const unsigned long long t = a.toa[beg + i];
    v = t > v ? t : v;
  }
  for (int o = 16; o; o >>= 1) {
    const unsigned long long t = __shfl_xor_sync(0xffffffffu, v, o);
    v = t > v ? t : v;
  }
  if ((threadIdx.x & 31) == 0 && v) atomicMax(reinterpret_cast<unsigned long long*>(&a.c->t_max), v);
}

// Every block derives the cut of this push from the state (unchanged until k_stream_scan); block 0 records it.
__device__ __forceinline__ void stream_cut(const StreamArgs& a, uint64_t& t_lo, uint64_t& t_cut) {
  const StreamCtrl* c = a.c;
  const uint64_t t_max = c->t_max, s_emitted = c->s_emitted;
  uint64_t s_cut = t_max >= a.D ? (t_max - a.D) / a.P : 0ull;
  if (s_cut < s_emitted) s_cut = s_emitted;
  t_lo = s_emitted * a.P;
  t_cut = s_cut * a.P;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    a.c->s_cut = s_cut; a.c->t_lo = t_lo; a.c->t_cut = t_cut; a.c->final_push = (uint32_t)a.final_push;
  }
}

// 0 = late, 1 = emit, 2 = carry
__device__ __forceinline__ uint32_t stream_class(uint64_t t, uint64_t t_lo, uint64_t t_cut, int final_push) {
  if (t < t_lo) return 0u;
  return (final_push || t < t_cut) ? 1u : 2u;
}

__device__ __forceinline__ uint64_t stream_toa(const StreamArgs& a, uint32_t n_carry, uint64_t v) {
  return v < n_carry ? a.ctoa[v] : a.toa[v - n_carry];
}

__global__ void __launch_bounds__(kStreamThreads) k_stream_mark(StreamArgs a) {
  __shared__ uint32_t s_cnt[2];
  if (threadIdx.x < 2) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  uint64_t t_lo, t_cut;
  stream_cut(a, t_lo, t_cut);
  const uint32_t n_carry = a.c->n_carry_in;
  const uint64_t nv = a.n + n_carry;
  const uint64_t base = (uint64_t)blockIdx.x * kStreamTile;     // the grid covers n + carry_cap: blocks past nv count 0
  uint32_t e = 0, k = 0;
#pragma unroll 4
  for (int i = 0; i < kStreamItems; ++i) {
    const uint64_t v = base + (uint64_t)i * kStreamThreads + threadIdx.x;
    if (v < nv) {
      const uint32_t cl = stream_class(stream_toa(a, n_carry, v), t_lo, t_cut, a.final_push);
      e += cl == 1u;
      k += cl == 2u;
    }
  }
  e = __reduce_add_sync(0xffffffffu, e);
  k = __reduce_add_sync(0xffffffffu, k);
  if ((threadIdx.x & 31) == 0) {
    if (e) atomicAdd(&s_cnt[0], e);
    if (k) atomicAdd(&s_cnt[1], k);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    a.blk_emit[blockIdx.x] = s_cnt[0];
    a.blk_keep[blockIdx.x] = s_cnt[1];
  }
}

__global__ void __launch_bounds__(1024) k_stream_scan(StreamArgs a) {
  const uint32_t e = scan_inplace_1024(a.blk_emit, a.nblk);
  __syncthreads();
  const uint32_t k = scan_inplace_1024(a.blk_keep, a.nblk);
  if (threadIdx.x == 0) {
    StreamCtrl* c = a.c;
    const uint64_t nv = a.n + c->n_carry_in;
    if (a.nblk == 0) {   // nothing to mark: record the (unchanged) cut here
      uint64_t t_lo, t_cut;
      stream_cut(a, t_lo, t_cut);
    }
    c->label_base = c->label_next;
    c->label_next += e;
    c->n_carry = k > a.carry_cap ? a.carry_cap : k;
    c->overflow = k > a.carry_cap ? 1u : 0u;
    if (c->overflow) c->dead = 1u;                  // more events to carry than the buffer holds: the stream is dead
    c->n_work = c->dead ? 0u : e;                   // (a dead stream clusters nothing; the status word says CAPACITY)
    c->n_late = (uint32_t)(nv - e - k);
    c->late_total += nv - e - k;
    if (!a.final_push) c->s_emitted = c->s_cut;
  }
}

__global__ void __launch_bounds__(kStreamThreads, 3) k_stream_scatter(StreamArgs a) {
  __shared__ __align__(16) uint8_t s_cls[kStreamTile];
  __shared__ uint16_t s_rank[kStreamTile];
  __shared__ uint32_t sm[33];
  const uint32_t n_carry = a.c->n_carry_in;
  const uint64_t t_lo = a.c->t_lo, t_cut = a.c->t_cut, nv = a.n + n_carry;
  const uint64_t base = (uint64_t)blockIdx.x * kStreamTile;
  if (base >= nv) return;
  // striped (coalesced) pass: ToA and class of every event
  uint64_t t[kStreamItems];
#pragma unroll
  for (int i = 0; i < kStreamItems; ++i) {
    const uint32_t loc = (uint32_t)i * kStreamThreads + threadIdx.x;
    const uint64_t v = base + loc;
    uint32_t cl = 0;
    t[i] = 0;
    if (v < nv) {
      t[i] = stream_toa(a, n_carry, v);
      cl = stream_class(t[i], t_lo, t_cut, a.final_push);
    }
    s_cls[loc] = (uint8_t)cl;
  }
  __syncthreads();
  // blocked pass over the classes: a thread owns 8 consecutive events, so ranks follow the stream order
  static_assert(kStreamItems == 8, "one 8-byte load of classes per thread");
  const uint2 q = *reinterpret_cast<const uint2*>(&s_cls[threadIdx.x * kStreamItems]);
  const uint32_t qw[2] = {q.x, q.y};
  uint32_t e = 0, k = 0;
#pragma unroll
  for (int j = 0; j < kStreamItems; ++j) {
    const uint32_t cl = (qw[j >> 2] >> (8 * (j & 3))) & 0xFFu;
    e += cl == 1u;
    k += cl == 2u;
  }
  uint32_t eo = block_exclusive_scan_256(e, sm, nullptr);
  uint32_t ko = block_exclusive_scan_256(k, sm, nullptr);
#pragma unroll
  for (int j = 0; j < kStreamItems; ++j) {
    const uint32_t cl = (qw[j >> 2] >> (8 * (j & 3))) & 0xFFu;
    if (cl == 1u) s_rank[threadIdx.x * kStreamItems + j] = (uint16_t)eo++;
    else if (cl == 2u) s_rank[threadIdx.x * kStreamItems + j] = (uint16_t)ko++;
  }
  __syncthreads();
  // striped pass again: neighbouring threads hold neighbouring ranks, so the copies are coalesced
  const uint32_t e_base = a.blk_emit[blockIdx.x], k_base = a.blk_keep[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kStreamItems; ++i) {
    const uint32_t loc = (uint32_t)i * kStreamThreads + threadIdx.x;
    const uint32_t cl = s_cls[loc];
    if (cl == 0u) continue;
    const uint64_t v = base + loc;
    uint16_t ex, ey, et;
    if (v < n_carry) { ex = a.cx[v]; ey = a.cy[v]; et = a.ctot[v]; }
    else { const uint64_t j = v - n_carry; ex = a.x[j]; ey = a.y[j]; et = a.tot[j]; }
    const uint32_t r = s_rank[loc];
    if (cl == 1u) {
      const uint32_t o = e_base + r;
      a.wx[o] = ex; a.wy[o] = ey; a.wtot[o] = et; a.wtoa[o] = t[i];
    } else {
      const uint32_t o = k_base + r;
      if (o < a.carry_cap) { a.nx[o] = ex; a.ny[o] = ey; a.ntot[o] = et; a.ntoa[o] = t[i]; }
    }
  }
}

}  // namespace tpx3
