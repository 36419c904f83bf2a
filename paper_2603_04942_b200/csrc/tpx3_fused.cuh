// Fused shot-tile path: S0-S5 in ONE kernel for shot-contiguous streams (shot = ToA div P never
// decreases along the input, as in a TimePix3 readout where disorder is confined to a readout
// window — PAPER.md:62, 68, 96; BASELINE.json configs 0-4).
//
// No link crosses a shot (PAPER.md:68 assigns every pixel to one laser trigger; R6), and
// with a shot-contiguous stream the stable (shot, ToA) order only permutes events INSIDE a shot.
// So the stream is cut into tiles of whole shots and each tile is finished in shared memory:
//
//   tile b owns the shots that START inside input slice [b*S, (b+1)*S); it reads up to T = S + L
//   events (L = the largest shot the variant supports) to reach the end of its last shot. The
//   global sorted position of an event is tile start + local rank: perm and label need no
//   inter-tile communication. Only the ordinal of a hit in the ascending-label cluster table
//   needs a prefix over tiles: a decoupled look-back over per-tile status words (tiles are
//   handed out by an atomic ticket, so every predecessor of a running tile has started).
//
// Per tile (all in shared memory, one CTA):
//   load     128-bit coalesced loads of toa / x / y / tot; shot = toa div P by multiply-high with
//            a precomputed magic number; composite key = (shot - first shot) << tof_bits | ToF
//   sort     skipped when the keys are already ascending; otherwise stable LSD radix sort of
//            16-bit local indices, digits ranked per warp with match.any (S1)
//   link     multimap hash table (cell -> event) in shared memory; every event probes its own
//            cell and the 4 "forward" neighbour cells (E, SW, S, SE), tests same shot and
//            |dToA| <= W (Eq. 5) and unites in a lock-free union-find that
//            always hooks the larger root under the smaller (S2)
//   compress label = root = smallest sorted index of the component; ordinals by block scan (S3)
//   reduce   members chained to their root (one atomicExch each); one thread per hit walks
//            the chain: exact 64-bit sums, brightest pixel by (ToT, sorted index) (S4, :150)
//   centroid fp32(sum tot*x) / fp32(sum tot), IEEE RN (S5, Eq. 9)
//
// A tile that cannot be handled (a shot longer than L, a decreasing shot number, key wider than
// 32 bits) marks the call as failed; the general kernels, enqueued behind this one, then run.
#pragma once
#include "tpx3_common.cuh"

namespace tpx3 {

// ---- exact 64-bit division by an invariant divisor (multiply-high + shift) -------------------
// Round-up method (Granlund & Montgomery 1994; the form used here keeps a 65-bit multiplier by
// an add-and-halve fix-up): for d not a power of two, l = floor(log2 d),
//   m = floor(2^(64+l) / d) + 1 if that is exact enough (error term e = d - 2^(64+l) mod d < 2^l),
//   otherwise the 65-bit multiplier floor(2^(65+l) / d) + 1 whose top bit is implicit.
struct Div64 {
  uint64_t magic;  // 0: power of two (shift only)
  uint32_t shift;
  uint32_t add;    // 1: 65-bit multiplier
};

inline Div64 make_div64(uint64_t d) {
  Div64 r{0, 0, 0};
  if (d == 0) return r;
  uint32_t l = 63u - (uint32_t)__builtin_clzll(d);
  if ((d & (d - 1)) == 0) { r.shift = l; return r; }
  unsigned __int128 num = (unsigned __int128)1 << (64 + l);
  uint64_t m = (uint64_t)(num / d);
  uint64_t rem = (uint64_t)(num % d);
  uint64_t e = d - rem;
  if (e < ((uint64_t)1 << l)) {
    r.shift = l;
  } else {
    m += m;
    uint64_t twice = rem + rem;
    if (twice >= d || twice < rem) m += 1;
    r.shift = l;
    r.add = 1;
  }
  r.magic = m + 1;
  return r;
}

__device__ __forceinline__ uint64_t div64(uint64_t n, const Div64& d) {
  if (d.magic == 0) return n >> d.shift;
  uint64_t q = __umul64hi(n, d.magic);
  if (d.add) q = ((n - q) >> 1) + q;
  return q >> d.shift;
}

// ---- tile status words for the decoupled look-back -------------------------------------------
constexpr unsigned long long kTileAggregate = 1ull << 62;  // value = hits of this tile
constexpr unsigned long long kTilePrefix = 2ull << 62;     // value = hits of tiles 0..this
constexpr unsigned long long kTileValueMask = 0xFFFFFFFFull;

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ uint4 ldg_nc_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

struct FusedArgs {
  Ctrl* ctrl;
  unsigned long long* tiles;
  uint64_t n;
  uint64_t P;
  Div64 divP;
  uint32_t W;
  uint32_t S;          // slice length (events); tile b owns shots starting in [b*S, (b+1)*S)
  uint32_t num_tiles;
  uint32_t sensor_w, sensor_h;
  uint32_t flags;
  const uint16_t* x;
  const uint16_t* y;
  const uint64_t* toa;
  const uint16_t* tot;
  uint32_t* perm;
  uint32_t* label;
  uint64_t max_clusters;
  tpx3_clusters_t out;
  uint32_t* n_clusters;
};

constexpr uint32_t kNone = 0xFFFFFFFFu;

template <int T>
struct FusedSmem {
  // byte offsets inside the dynamic shared memory block
  static constexpr int kRegA = 0;            // 8T  unsorted->sorted records OR hash / lists
  static constexpr int kRegB = 8 * T;        // 8T  records as loaded (input order)
  static constexpr int kRegC = 16 * T;       // 4T  sort index double buffer -> chain heads
  static constexpr int kRegD = 20 * T;       // 4T  warp digit counters (sort) -> parent
  static constexpr int kMisc = 24 * T;       // small block-wide scalars
  static constexpr int kMiscBytes = 512;
  static constexpr int kBytes = kMisc + kMiscBytes;
};

struct FusedMisc {
  unsigned long long s_lo;     // shot number of the first owned event
  unsigned int lo, hi;         // owned range, relative to the tile base
  unsigned int fail;
  unsigned int unsorted;
  unsigned int max_tof, max_local;
  unsigned int ticket;
  unsigned int n_roots;
  unsigned int ord_base;
  unsigned int warp_sums[33];
  unsigned int is_last;
};
static_assert(sizeof(FusedMisc) <= 512, "FusedMisc must fit kMiscBytes");

// One tile per CTA. T = tile capacity (events), THREADS = T / 8.
template <int T, int THREADS>
__global__ void __launch_bounds__(THREADS, (T <= 4096 ? 2 : 1)) k_fused_shot_tiles(FusedArgs a) {
  constexpr int IPT = T / THREADS;  // 8 consecutive events per thread in the load phase
  static_assert(IPT == 8, "the 128-bit load phase assumes 8 events per thread");
  constexpr int WARPS = THREADS / 32;
  constexpr uint32_t HS = 2u * T;   // hash slots
  using L = FusedSmem<T>;
  extern __shared__ __align__(16) unsigned char smem[];
  FusedMisc* misc = reinterpret_cast<FusedMisc*>(smem + L::kMisc);
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;

  // ---- ticket: tiles are processed in start order (look-back needs started predecessors) ----
  if (tid == 0) {
    misc->ticket = atomicAdd(&a.ctrl->tile_ticket, 1u);
    misc->lo = kNone;
    misc->hi = kNone;
    misc->fail = 0;
    misc->unsorted = 0;
    misc->max_tof = 0;
    misc->max_local = 0;
    misc->n_roots = 0;
    misc->ord_base = 0;
    misc->is_last = 0;
  }
  __syncthreads();
  const uint32_t b = misc->ticket;
  const uint64_t base = (uint64_t)b * a.S;             // first event this tile looks at
  const uint64_t avail = a.n - base;                   // > 0 by construction
  const uint32_t cnt = avail < (uint64_t)T ? (uint32_t)avail : (uint32_t)T;  // events readable
  const uint32_t p0 = tid * IPT;                       // this thread's 8 tile-relative positions

  // ---- load ToA (2 events per 128-bit load), shot numbers, boundaries --------------------------
  uint64_t toa_r[IPT];
  if (p0 + IPT <= cnt) {
    const uint4* src = reinterpret_cast<const uint4*>(a.toa + base + p0);
#pragma unroll
    for (int j = 0; j < IPT / 2; ++j) {
      uint4 v = ldg_nc_v4(src + j);
      toa_r[2 * j] = ((uint64_t)v.y << 32) | v.x;
      toa_r[2 * j + 1] = ((uint64_t)v.w << 32) | v.z;
    }
  } else {
#pragma unroll
    for (int j = 0; j < IPT; ++j) toa_r[j] = (p0 + j < cnt) ? a.toa[base + p0 + j] : 0ull;
  }
  // shot of the event just before this thread's first one (previous lane, or a global load)
  uint64_t s_first = div64(toa_r[0], a.divP);
  uint64_t s_last = div64(toa_r[IPT - 1], a.divP);
  uint64_t s_prev;
  {
    uint32_t lo32 = __shfl_up_sync(0xffffffffu, (uint32_t)s_last, 1);
    uint32_t hi32 = __shfl_up_sync(0xffffffffu, (uint32_t)(s_last >> 32), 1);
    s_prev = ((uint64_t)hi32 << 32) | lo32;
    if (lane == 0) {
      if (base + p0 > 0 && p0 < cnt) s_prev = div64(a.toa[base + p0 - 1], a.divP);
      else s_prev = ~0ull;  // position 0 of the stream: always a shot start
    }
  }
  uint32_t bnd = 0;  // bit j: event p0+j starts a shot
  bool viol = false;
  {
    uint64_t sp = s_prev;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      if (p0 + j < cnt) {
        uint64_t s = (j == 0) ? s_first : ((j == IPT - 1) ? s_last : div64(toa_r[j], a.divP));
        bool start = (base + p0 + j == 0) || (s != sp);
        if (start) bnd |= 1u << j;
        if (base + p0 + j != 0 && s < sp && p0 + j < a.S) viol = true;  // each position checked once
        sp = s;
      }
    }
  }
  // lo = first shot start in [0, S); hi = first shot start in [S, cnt) (or cnt == end of stream)
  {
    uint32_t my_lo = kNone, my_hi = kNone;
#pragma unroll
    for (int j = IPT - 1; j >= 0; --j) {
      if (bnd & (1u << j)) {
        if (p0 + j < a.S) my_lo = p0 + j;
        else my_hi = p0 + j;
      }
    }
    // my_hi must be the FIRST start at or after S: the loop runs downwards, so it is
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      my_lo = min(my_lo, __shfl_xor_sync(0xffffffffu, my_lo, o));
      my_hi = min(my_hi, __shfl_xor_sync(0xffffffffu, my_hi, o));
    }
    uint32_t any_viol = __any_sync(0xffffffffu, viol);
    if (lane == 0) {
      if (my_lo != kNone) atomicMin(&misc->lo, my_lo);
      if (my_hi != kNone) atomicMin(&misc->hi, my_hi);
      if (any_viol) misc->fail = 1;
    }
  }
  __syncthreads();
  uint32_t lo = misc->lo, hi = misc->hi;
  if (hi == kNone) {
    if (base + cnt >= a.n) hi = cnt;          // the stream ends inside this tile's window
    else if (lo != kNone) { hi = lo; if (tid == 0) misc->fail = 1; }  // last shot longer than the window
  }
  if (lo == kNone) { lo = 0; hi = 0; }        // no shot starts in this slice: nothing owned
  const uint32_t m = hi - lo;                 // owned events; sorted position k <-> p = lo + k
  // shot number of the first owned event
  if (m && lo >= p0 && lo < p0 + IPT) {
    uint64_t s = 0;
#pragma unroll
    for (int j = 0; j < IPT; ++j)
      if (p0 + j == lo) s = div64(toa_r[j], a.divP);
    misc->s_lo = s;
  }
  __syncthreads();
  const uint64_t s_lo = misc->s_lo;

  // ---- ToF and shot offset of every owned event; widths of the composite key ------------------
  uint32_t tof_r[IPT], loc_r[IPT];
  {
    uint32_t mt = 0, ml = 0;
    bool bad = false;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t p = p0 + j;
      tof_r[j] = 0;
      loc_r[j] = 0;
      if (p >= lo && p < hi) {
        uint64_t s = div64(toa_r[j], a.divP);
        uint64_t d = s - s_lo;
        if (d > 0xFFFFFFFFull) bad = true;
        tof_r[j] = (uint32_t)(toa_r[j] - s * a.P);
        loc_r[j] = (uint32_t)d;
        mt = max(mt, tof_r[j]);
        ml = max(ml, loc_r[j]);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      mt = max(mt, __shfl_xor_sync(0xffffffffu, mt, o));
      ml = max(ml, __shfl_xor_sync(0xffffffffu, ml, o));
    }
    uint32_t any_bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
      if (mt) atomicMax(&misc->max_tof, mt);
      if (ml) atomicMax(&misc->max_local, ml);
      if (any_bad) misc->fail = 1;
    }
  }
  __syncthreads();
  const uint32_t tof_bits = misc->max_tof ? 32u - (uint32_t)__clz(misc->max_tof) : 1u;
  const uint32_t shot_bits = misc->max_local ? 32u - (uint32_t)__clz(misc->max_local) : 0u;
  const uint32_t key_bits = tof_bits + shot_bits;
  const bool failed = misc->fail || key_bits > 32u;
  const uint32_t mm = failed ? 0u : m;   // a failed tile owns nothing (the general path redoes the call)

  // ---- records as loaded -> region B (key, xy, tot), 128-bit loads of x / y / tot ---------------
  uint32_t* keyB = reinterpret_cast<uint32_t*>(smem + L::kRegB);
  uint16_t* xyB = reinterpret_cast<uint16_t*>(smem + L::kRegB + 4 * T);
  uint16_t* totB = reinterpret_cast<uint16_t*>(smem + L::kRegB + 6 * T);
  uint32_t key_r[IPT];
#pragma unroll
  for (int j = 0; j < IPT; ++j) key_r[j] = (loc_r[j] << tof_bits) | tof_r[j];
  if (mm && p0 < hi && p0 + IPT > lo) {
    uint4 vx, vy, vt;
    if (p0 + IPT <= cnt) {
      vx = ldg_nc_v4(a.x + base + p0);
      vy = ldg_nc_v4(a.y + base + p0);
      vt = ldg_nc_v4(a.tot + base + p0);
    } else {
      uint16_t tx[IPT], ty[IPT], tt[IPT];
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        bool ok = p0 + j < cnt;
        tx[j] = ok ? a.x[base + p0 + j] : (uint16_t)0;
        ty[j] = ok ? a.y[base + p0 + j] : (uint16_t)0;
        tt[j] = ok ? a.tot[base + p0 + j] : (uint16_t)1;
      }
      vx = make_uint4(tx[0] | ((uint32_t)tx[1] << 16), tx[2] | ((uint32_t)tx[3] << 16),
                      tx[4] | ((uint32_t)tx[5] << 16), tx[6] | ((uint32_t)tx[7] << 16));
      vy = make_uint4(ty[0] | ((uint32_t)ty[1] << 16), ty[2] | ((uint32_t)ty[3] << 16),
                      ty[4] | ((uint32_t)ty[5] << 16), ty[6] | ((uint32_t)ty[7] << 16));
      vt = make_uint4(tt[0] | ((uint32_t)tt[1] << 16), tt[2] | ((uint32_t)tt[3] << 16),
                      tt[4] | ((uint32_t)tt[5] << 16), tt[6] | ((uint32_t)tt[7] << 16));
    }
    if (a.flags & TPX3_FLAG_VALIDATE_INPUT) {
      const uint32_t xs[4] = {vx.x, vx.y, vx.z, vx.w}, ys[4] = {vy.x, vy.y, vy.z, vy.w},
                     ts[4] = {vt.x, vt.y, vt.z, vt.w};
      bool oob = false;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int hw = 0; hw < 2; ++hw) {
          const uint32_t p = p0 + 2 * q + hw;
          if (p >= lo && p < hi) {
            uint32_t xx = (xs[q] >> (16 * hw)) & 0xFFFFu, yy = (ys[q] >> (16 * hw)) & 0xFFFFu,
                     tt = (ts[q] >> (16 * hw)) & 0xFFFFu;
            if (xx >= a.sensor_w || yy >= a.sensor_h || tt == 0) oob = true;
          }
        }
      }
      if (oob) set_error(a.ctrl, TPX3_ERR_OUT_OF_RANGE);
    }
    // xy = x | y << 8, two events per 32-bit word
    uint4 vxy;
    vxy.x = (vx.x & 0x00FF00FFu) | ((vy.x & 0x00FF00FFu) << 8);
    vxy.y = (vx.y & 0x00FF00FFu) | ((vy.y & 0x00FF00FFu) << 8);
    vxy.z = (vx.z & 0x00FF00FFu) | ((vy.z & 0x00FF00FFu) << 8);
    vxy.w = (vx.w & 0x00FF00FFu) | ((vy.w & 0x00FF00FFu) << 8);
    *reinterpret_cast<uint4*>(xyB + p0) = vxy;
    *reinterpret_cast<uint4*>(totB + p0) = vt;
    *reinterpret_cast<uint4*>(keyB + p0) = make_uint4(key_r[0], key_r[1], key_r[2], key_r[3]);
    *reinterpret_cast<uint4*>(keyB + p0 + 4) = make_uint4(key_r[4], key_r[5], key_r[6], key_r[7]);
  }
  __syncthreads();
  // already in (shot, ToA) order? (configs 0-3 arrive sorted; config 4 does not)
  {
    bool uns = false;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t p = p0 + j;
      if (p > lo && p < lo + mm) {
        uint32_t prev = (j == 0) ? keyB[p - 1] : key_r[j - 1];
        if (key_r[j] < prev) uns = true;
      }
    }
    if (__any_sync(0xffffffffu, uns) && lane == 0) misc->unsorted = 1;
  }
  __syncthreads();
  const bool unsorted = misc->unsorted != 0;

  // ---- S1: stable LSD radix sort of local indices by composite key (only if needed) ------------
  uint32_t* keyA = reinterpret_cast<uint32_t*>(smem + L::kRegA);
  uint16_t* xyA = reinterpret_cast<uint16_t*>(smem + L::kRegA + 4 * T);
  uint16_t* totA = reinterpret_cast<uint16_t*>(smem + L::kRegA + 6 * T);
  const uint32_t out_base = (uint32_t)(base + lo);  // global sorted position of local rank 0 (n <= 2^28)
  if (unsorted) {
    uint16_t* buf0 = reinterpret_cast<uint16_t*>(smem + L::kRegC);
    uint16_t* buf1 = buf0 + T;
    uint32_t* wcnt = reinterpret_cast<uint32_t*>(smem + L::kRegD);  // [WARPS][256]
    const uint32_t npass = (key_bits + 7u) / 8u;
    const uint32_t dbits = (key_bits + npass - 1u) / npass;         // <= 8
    const uint32_t radix = 1u << dbits, dmask = radix - 1u;
    const uint32_t lt = lanemask_lt();
    for (uint32_t pass = 0; pass < npass; ++pass) {
      const uint16_t* src = (pass & 1u) ? buf1 : buf0;
      uint16_t* dst = (pass & 1u) ? buf0 : buf1;
      const uint32_t shift = pass * dbits;
      for (uint32_t i = tid; i < WARPS * 256u; i += THREADS) wcnt[i] = 0;
      __syncthreads();
      uint32_t e_src[IPT], e_dig[IPT], e_rank[IPT];
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        const uint32_t k = warp * (32u * IPT) + (uint32_t)j * 32u + lane;   // warps own ascending slices
        const bool valid = k < mm;
        uint32_t s = valid ? (pass == 0 ? k : (uint32_t)src[k]) : 0u;
        uint32_t d = valid ? ((keyB[lo + s] >> shift) & dmask) : 256u;      // 256: "no event"
        uint32_t peers = __match_any_sync(0xffffffffu, d);
        uint32_t lr = __popc(peers & lt);
        uint32_t c0 = valid ? wcnt[warp * 256u + d] : 0u;
        __syncwarp();
        if (valid && lr == 0) wcnt[warp * 256u + d] = c0 + __popc(peers);
        __syncwarp();
        e_src[j] = s;
        e_dig[j] = d;
        e_rank[j] = c0 + lr;
      }
      __syncthreads();
      // digit d (thread d): exclusive prefix over warps, then over digits
      uint32_t tot_d = 0;
      if (tid < radix) {
#pragma unroll 4
        for (int w = 0; w < WARPS; ++w) {
          uint32_t c = wcnt[w * 256 + tid];
          wcnt[w * 256 + tid] = tot_d;
          tot_d += c;
        }
      }
      uint32_t inc = tot_d;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc += t;
      }
      if (lane == 31 && warp < 8) misc->warp_sums[warp] = inc;
      __syncthreads();
      if (tid < radix) {
        uint32_t wbase = 0;
        for (uint32_t w = 0; w < warp; ++w) wbase += misc->warp_sums[w];
        const uint32_t dbase = wbase + inc - tot_d;
#pragma unroll 4
        for (int w = 0; w < WARPS; ++w) wcnt[w * 256 + tid] += dbase;
      }
      __syncthreads();
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        if (e_dig[j] < 256u) dst[wcnt[warp * 256u + e_dig[j]] + e_rank[j]] = (uint16_t)e_src[j];
      }
      __syncthreads();
    }
    const uint16_t* fin = (npass & 1u) ? buf1 : buf0;
    // gather the records into sorted order (region A) and emit perm
    for (uint32_t k = tid; k < mm; k += THREADS) {
      const uint32_t s = fin[k];
      keyA[k] = keyB[lo + s];
      xyA[k] = xyB[lo + s];
      totA[k] = totB[lo + s];
      a.perm[out_base + k] = out_base + s;
    }
  } else {
    for (uint32_t k = tid; k < mm; k += THREADS) a.perm[out_base + k] = out_base + k;
  }
  __syncthreads();
  const uint32_t* keyS = unsorted ? keyA : keyB + lo;
  const uint16_t* xyS = unsorted ? xyA : xyB + lo;
  const uint16_t* totS = unsorted ? totA : totB + lo;
  unsigned char* freeR = smem + (unsorted ? L::kRegB : L::kRegA);   // 8T bytes no longer needed

  // ---- S2: chained hash cell -> events, probe own + 4 forward cells, union-find -----------------
  // bucket head and chain links both carry (cell << 16 | event), so a chain is walked without
  // touching the records; only a cell match reads the candidate's key (same shot, |dToA| <= W).
  uint32_t* bhead = reinterpret_cast<uint32_t*>(freeR);               // [HS] kNone = empty bucket
  uint32_t* nextc = reinterpret_cast<uint32_t*>(smem + L::kRegC);     // [T]  next node of the bucket chain
  uint32_t* parent = reinterpret_cast<uint32_t*>(smem + L::kRegD);    // [T]
  {
    uint4 e = make_uint4(kNone, kNone, kNone, kNone);
    uint4* t4 = reinterpret_cast<uint4*>(bhead);
#pragma unroll
    for (int q = 0; q < (int)(HS / 4 / THREADS); ++q) t4[q * THREADS + tid] = e;
    for (uint32_t k = tid; k < mm; k += THREADS) parent[k] = k;
  }
  __syncthreads();
  constexpr uint32_t kHashShift = 32u - (T == 8192 ? 14u : (T == 4096 ? 13u : (T == 2048 ? 12u : 11u)));
  static_assert(T == 8192 || T == 4096 || T == 2048 || T == 1024, "hash shift table");
  for (uint32_t k = tid; k < mm; k += THREADS) {
    const uint32_t cell = xyS[k], loc = keyS[k] >> tof_bits;
    const uint32_t h = ((cell | (loc << 16)) * 0x9E3779B1u) >> kHashShift;
    nextc[k] = atomicExch(&bhead[h], (cell << 16) | k);
  }
  __syncthreads();
  for (uint32_t k0 = 0; k0 < mm; k0 += THREADS) {   // block-uniform trip count; lanes past mm idle
    const uint32_t k = k0 + tid;
    const bool act = k < mm;
    const uint32_t cell = act ? xyS[k] : 0u, key = act ? keyS[k] : 0u, loc = key >> tof_bits;
    const uint32_t x = cell & 0xFFu, y = cell >> 8;
    // neighbour cells still to visit: bit q of {own, E, SW, S, SE}; sensor edges removed
    uint32_t todo = 0;
    if (act) {
      const bool xe = x + 1u < a.sensor_w, xw = x > 0u, ys = y + 1u < a.sensor_h;
      todo = 1u | (xe ? 2u : 0u) | ((xw && ys) ? 4u : 0u) | (ys ? 8u : 0u) | ((xe && ys) ? 16u : 0u);
    }
    // one flattened loop over all five chains keeps the lanes of a warp in step; matching
    // candidates are only recorded here (up to 8, packed 2 per register) and united afterwards
    uint32_t cand[4] = {0u, 0u, 0u, 0u};
    uint32_t ncand = 0, cur = kNone, c = 0, q = 0;
    uint32_t rk = k;   // current guess of k's root
    auto unite = [&](uint32_t j) {
      uint32_t ra = rk, rb = j;
      for (;;) {
        uint32_t p;
        while ((p = parent[ra]) != ra) { uint32_t g = parent[p]; if (g != p) parent[ra] = g; ra = p; }
        while ((p = parent[rb]) != rb) { uint32_t g = parent[p]; if (g != p) parent[rb] = g; rb = p; }
        if (ra == rb) break;
        if (ra < rb) { uint32_t t = ra; ra = rb; rb = t; }
        const uint32_t old = atomicMin(&parent[ra], rb);   // hook the larger root under the smaller
        if (old == ra) { ra = rb; break; }
        ra = old;
      }
      rk = ra;
    };
    while (todo != 0u || cur != kNone) {
      if (cur == kNone) {
        q = (uint32_t)__ffs(todo) - 1u;
        todo &= todo - 1u;
        const uint32_t off = (q == 0u) ? 0u : (q == 1u ? 1u : 253u + q);   // 0, +1, +255, +256, +257
        c = cell + off;
        cur = bhead[((c | (loc << 16)) * 0x9E3779B1u) >> kHashShift];
      } else {
        const uint32_t j = cur & 0xFFFFu, tag = cur >> 16;
        cur = nextc[j];
        if (tag == c && (q != 0u || j < k)) {
          const uint32_t kj = keyS[j];
          const uint32_t dt = key > kj ? key - kj : kj - key;
          if ((kj >> tof_bits) == loc && dt <= a.W) {
            if (ncand < 8u) {
              cand[ncand >> 1] |= j << ((ncand & 1u) * 16u);
              ++ncand;
            } else {
              unite(j);   // more than 8 neighbours (heavy overlap): unite on the spot
            }
          }
        }
      }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if ((uint32_t)i < ncand) unite((cand[i >> 1] >> ((i & 1) * 16)) & 0xFFFFu);
    }
  }
  __syncthreads();

  uint32_t* head = reinterpret_cast<uint32_t*>(smem + L::kRegC);   // [T] member chain head per root (nextc is dead)
  // ---- S3: label = root (smallest sorted index of the component); ordinals of the roots ---------
  {
    uint32_t root_r[IPT];
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t k = (uint32_t)j * THREADS + tid;
      uint32_t r = k;
      if (k < mm) {
        uint32_t p;
        while ((p = parent[r]) != r) r = p;
      }
      root_r[j] = r;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t k = (uint32_t)j * THREADS + tid;
      if (k < mm) {
        parent[k] = root_r[j];
        head[k] = kNone;
        a.label[out_base + k] = out_base + root_r[j];
      }
    }
  }
  __syncthreads();
  uint16_t* nxt = reinterpret_cast<uint16_t*>(freeR);            // [T] next member of the same hit
  uint16_t* rootpos = reinterpret_cast<uint16_t*>(freeR + 2 * T);  // [T] ordinal -> sorted index of the root
  uint32_t n_roots;
  {
    // blocked arrangement: thread owns sorted positions [8 tid, 8 tid + 8)
    const uint4 q0 = *reinterpret_cast<const uint4*>(parent + p0);
    const uint4 q1 = *reinterpret_cast<const uint4*>(parent + p0 + 4);
    const uint32_t pr[IPT] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
    uint32_t flags = 0, cntr = 0;
#pragma unroll
    for (int j = 0; j < IPT; ++j)
      if (p0 + j < mm && pr[j] == p0 + j) { flags |= 1u << j; ++cntr; }
    uint32_t inc = cntr;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= (uint32_t)o) inc += t;
    }
    if (lane == 31) misc->warp_sums[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      uint32_t ws = lane < (uint32_t)WARPS ? misc->warp_sums[lane] : 0u, xs = ws;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, xs, o);
        if (lane >= (uint32_t)o) xs += t;
      }
      if (lane < (uint32_t)WARPS) misc->warp_sums[lane] = xs - ws;
      if (lane == 31) misc->n_roots = xs;
    }
    __syncthreads();
    uint32_t ord = misc->warp_sums[warp] + inc - cntr;
#pragma unroll
    for (int j = 0; j < IPT; ++j)
      if (flags & (1u << j)) rootpos[ord++] = (uint16_t)(p0 + j);
    n_roots = misc->n_roots;
  }
  // publish this tile's hit count as early as possible
  if (tid == 0) {
    st_volatile_u64(a.tiles + b, (b == 0 ? kTilePrefix : kTileAggregate) | (unsigned long long)n_roots);
  }

  // ---- S4: chain every member to its root --------------------------------------------------------
  for (uint32_t k = tid; k < mm; k += THREADS) {
    const uint32_t r = parent[k];
    if (r != k) nxt[k] = (uint16_t)atomicExch(&head[r], k);   // kNone truncates to 0xFFFF = end
  }
  // ---- ordinal of this tile's first hit: decoupled look-back over the predecessors (warp 0) ----
  if (warp == 0 && b > 0) {
    uint32_t prefix = 0;
    int jb = (int)b - 1;
    for (;;) {
      const int idx = jb - (int)lane;
      unsigned long long v = kTilePrefix;   // before tile 0: an empty prefix
      if (idx >= 0) {
        while (((v = ld_volatile_u64(a.tiles + idx)) >> 62) == 0ull) __nanosleep(64);
      }
      const uint32_t pm = __ballot_sync(0xffffffffu, (v >> 62) == 2ull);
      const uint32_t first = pm ? (uint32_t)__ffs(pm) - 1u : 31u;   // nearest predecessor holding a prefix
      uint32_t val = lane <= first ? (uint32_t)(v & kTileValueMask) : 0u;
#pragma unroll
      for (int o = 16; o; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
      prefix += val;
      if (pm) break;
      jb -= 32;
    }
    if (lane == 0) {
      misc->ord_base = prefix;
      st_volatile_u64(a.tiles + b, kTilePrefix | (unsigned long long)(prefix + n_roots));
    }
  }
  __syncthreads();

  // ---- S4/S5: one thread per hit walks its chain: exact sums, brightest pixel, centroid ---------
  {
    const uint32_t ord_base = misc->ord_base;
    const uint32_t tof_mask = (tof_bits >= 32u) ? 0xFFFFFFFFu : ((1u << tof_bits) - 1u);
    bool over = false;
    for (uint32_t c = tid; c < n_roots; c += THREADS) {
      const uint32_t r = rootpos[c];
      unsigned long long st = 0, sx = 0, sy = 0;
      uint32_t size = 0, best = 0, k = r;
      do {
        const uint32_t cell = xyS[k], t = totS[k];
        st += t;
        sx += (unsigned long long)(t * (cell & 0xFFu));
        sy += (unsigned long long)(t * (cell >> 8));
        ++size;
        best = max(best, (t << 16) | k);   // (ToT, sorted index): the later pixel wins ties
        if (k == r) k = head[r];
        else { const uint32_t nk = nxt[k]; k = (nk == 0xFFFFu) ? kNone : nk; }
      } while (k != kNone);
      const uint64_t o = (uint64_t)ord_base + c;
      if (o < a.max_clusters) {
        const uint32_t kp = best & 0xFFFFu, keyp = keyS[kp];
        a.out.label[o] = out_base + r;
        a.out.size[o] = size;
        a.out.shot[o] = (uint32_t)(s_lo + (uint64_t)(keyS[r] >> tof_bits));
        a.out.sum_tot[o] = (long long)st;
        a.out.sum_tot_x[o] = (long long)sx;
        a.out.sum_tot_y[o] = (long long)sy;
        a.out.toa_peak[o] = (s_lo + (uint64_t)(keyp >> tof_bits)) * a.P + (uint64_t)(keyp & tof_mask);
        const float fst = __ll2float_rn((long long)st);
        a.out.cx[o] = __fdiv_rn(__ll2float_rn((long long)sx), fst);
        a.out.cy[o] = __fdiv_rn(__ll2float_rn((long long)sy), fst);
      } else {
        over = true;
      }
    }
    if (over) set_error(a.ctrl, TPX3_ERR_CAPACITY);
  }

  // ---- completion: the last tile to finish publishes the outcome of the call --------------------
  if (tid == 0) {
    if (failed) atomicExch(&a.ctrl->fused_fail, 1u);
    __threadfence();
    const uint32_t done = atomicAdd(&a.ctrl->tiles_done, 1u);
    if (done + 1u == a.num_tiles) {
      __threadfence();
      const uint32_t any_fail = atomicAdd(&a.ctrl->fused_fail, 0u);
      if (any_fail) {
        a.ctrl->fused_state = 2;   // the general kernels behind this one redo the call
        if (a.ctrl->status.error == (uint32_t)(-TPX3_ERR_CAPACITY)) a.ctrl->status.error = 0;
      } else {
        const uint32_t total = (uint32_t)(ld_volatile_u64(a.tiles + (a.num_tiles - 1u)) & kTileValueMask);
        *a.n_clusters = total;
        a.ctrl->status.n_clusters = total;
        a.ctrl->status.path = 1;
        a.ctrl->status.sort_passes = 0;
        a.ctrl->fused_state = 1;
      }
    }
  }
}

// Which variant serves a plan: L = largest supported shot (events), T = tile capacity, S = T - L.
struct FusedGeom {
  int variant;      // 0 = fused path not available for this plan, 1 = T 4096 / 512 thr, 2 = T 8192 / 1024 thr
  uint32_t T, S;
};

inline FusedGeom fused_geom(uint64_t P, uint32_t W, uint32_t max_shot_hits) {
  FusedGeom g{0, 0, 0};
  if (P == 0 || P > (1ull << 24) || W >= (1u << 24)) return g;   // ToF must fit the 32-bit composite key
  const uint32_t Lh = max_shot_hits ? max_shot_hits : 4096u;
  if (Lh <= 1024u) { g.variant = 1; g.T = 4096; }
  else if (Lh <= 4096u) { g.variant = 2; g.T = 8192; }
  else return g;
  g.S = (g.T - Lh) & ~7u;
  return g;
}

template <int T, int THREADS>
inline int launch_fused(const FusedArgs& a, cudaStream_t st) {
  auto kern = k_fused_shot_tiles<T, THREADS>;
  static bool configured = false;   // per process; the attribute is per function and device-wide
  if (!configured) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, FusedSmem<T>::kBytes) != cudaSuccess)
      return TPX3_ERR_CUDA;
    configured = true;
  }
  kern<<<a.num_tiles, THREADS, FusedSmem<T>::kBytes, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? TPX3_OK : TPX3_ERR_CUDA;
}

// Returns TPX3_OK (launched or not applicable; *launched says which) or an error.
inline int enqueue_fused(const FusedGeom& g, uint64_t* launches, Ctrl* ctrl, unsigned long long* tiles,
                         cudaStream_t st, const Params& prm, const uint16_t* x, const uint16_t* y,
                         const uint64_t* toa, const uint16_t* tot, uint32_t* perm, uint32_t* label,
                         uint64_t max_clusters, const tpx3_clusters_t& out, uint32_t* n_clusters, bool* launched) {
  *launched = false;
  if (g.variant == 0 || prm.n == 0) return TPX3_OK;
  // the 128-bit load phase needs 16-byte aligned inputs (PyTorch allocations are 256-byte aligned)
  if ((((uintptr_t)x | (uintptr_t)y | (uintptr_t)toa | (uintptr_t)tot) & 15u) != 0) return TPX3_OK;
  FusedArgs a;
  a.ctrl = ctrl;
  a.tiles = tiles;
  a.n = prm.n;
  a.P = prm.P;
  a.divP = make_div64(prm.P);
  a.W = prm.W;
  a.S = g.S;
  a.num_tiles = (uint32_t)((prm.n + g.S - 1) / g.S);
  a.sensor_w = prm.sensor_w;
  a.sensor_h = prm.sensor_h;
  a.flags = prm.flags;
  a.x = x; a.y = y; a.toa = toa; a.tot = tot;
  a.perm = perm; a.label = label;
  a.max_clusters = max_clusters;
  a.out = out;
  a.n_clusters = n_clusters;
  int rc = g.variant == 1 ? launch_fused<4096, 512>(a, st) : launch_fused<8192, 1024>(a, st);
  if (rc == TPX3_OK) { ++*launches; *launched = true; }
  return rc;
}

}  // namespace tpx3
