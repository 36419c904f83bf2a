// Fused shot-tile path: S0-S5 in ONE kernel for shot-contiguous streams (shot = ToA div P never
// decreases along the input, as in a TimePix3 readout where disorder is confined to a readout
// window — PAPER.md:62, 68, 96; BASELINE.json configs 0-4).
//
// No link crosses a shot (PAPER.md:68 assigns every pixel to one laser trigger; R6), and
// with a shot-contiguous stream the stable (shot, ToA) order only permutes events INSIDE a shot.
// So the stream is cut into tiles of whole shots and each tile is finished in shared memory:
//
//   the stream is cut into SEGMENTS of G events; CTA g walks segment g tile by tile. A tile starts at a
//   shot start (the first tile of a segment finds the first shot start at or after g*G), reads a window
//   of T events and owns the whole shots that lie inside the window and start before (g+1)*G; the next
//   tile starts where this one ended, so nothing but the shot that straddles the window's end is read
//   twice (round 1 cut fixed slices and read S + L events to own S: 58 % overlap on config 4). The
//   global sorted position of an event is tile start + local rank: perm and label need no
//   inter-tile communication. Only the ordinal of a hit in the ascending-label cluster table
//   needs a prefix over tiles: tiles write their hits to a staging table at their own position
//   and a small second kernel (k_fused_compact) moves them to their ordinals, so that no tile
//   ever waits for another one (a look-back inside the kernel cost 24-59 % of the warp time).
//
// Per tile (all in shared memory, one CTA; k = sorted position inside the tile):
//   load     128-bit coalesced loads of toa / x / y / tot. rel = toa - (first shot of the tile)*P
//            fits 32 bits; shot offset sl = rel div P by a 32-bit multiply-high; tof = rel - sl*P.
//            key = sl << tb | tof with 2^tb > max tof + W, so |key_i - key_j| <= W already implies
//            "same shot" and ONE compare is the whole time test of Eq. 5.
//   sort     skipped when the keys are already ascending; otherwise the rank of every event in the
//            stable (shot, ToA) order by counting: bitmap of the keys that occur -> dense key number
//            (prefix popcount) -> count per dense key -> offsets; events of one key (a few) are ordered
//            by input position. Keys too wide for the bitmap, or one key held by very many events: stable
//            LSD radix sort of 16-bit local indices, digits ranked per warp with ballots (S1)
//   hash     open table of 4-slot buckets (one 128-bit load reads a bucket), key (shot, cell),
//            entry = cell << 16 | k+1; a bucket that overflows spills to the next one and marks
//            itself, so the common probe is straight-line code
//   link     every event probes S, E, SE, SW and its own cell ("forward" cells), applies the time
//            test and keeps only links that are not implied by other neighbour pairs (two
//            candidates that are themselves adjacent in space and time are linked by one of them).
//            The first kept link is a plain store parent[k] = j (forward order => no cycles); the
//            few others go to a list that is united afterwards with compare-and-swap hooks (S2)
//   label    root per event by pointer chasing, label = smallest k of the component (shared-memory
//            atomicMin per event), ordinals of the labels by block scan (S3)
//   reduce   members chained to their label (one atomicExch each); one thread per hit walks the
//            chain: exact 64-bit sums, brightest pixel by (ToT, sorted index) (S4)
//            (+ sum tot*tof for the time-of-flight centroid)
//   centroid fp32(sum tot*x) / fp32(sum tot), IEEE RN (S5, Eq. 9), in k_fused_compact
//
// Template MODE 1 is the paper-literal mode (tpx3_localmax_centroid, R21): same tiling, load, sort,
// hash, staging and compaction, but in place of link / label / reduce an event is a hit when its box holds no
// greater (ToT, sorted index), and the sums run over that box. Boxes of <= 81 cells are scanned cell by cell
// through the hash, larger ones by walking the time window of the sorted tile.
//
// A tile that cannot be handled (a shot longer than the window, a decreasing shot number, shot offset and time
// of flight too wide for one 32-bit key) marks the call as failed; the general kernels, enqueued from the device
// behind this one (k_fallback_dispatch), then redo the call.
#pragma once
#include <type_traits>

#include "tpx3_common.cuh"
#include "tpx3_localmax.cuh"
#include "tpx3_preprocess.cuh"

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

// ---- exact 32-bit division by an invariant divisor -------------------------------------------
// Granlund & Montgomery 1994, Fig. 4.1 (N = 32): l = ceil(log2 d), m' = floor(2^32 (2^l - d) / d) + 1,
// q = (t + ((n - t) >> sh1)) >> sh2 with t = mulhi(m', n), sh1 = min(l, 1), sh2 = max(l - 1, 0).
struct Div32 {
  uint32_t m, sh1, sh2;
};

inline Div32 make_div32(uint32_t d) {
  uint32_t l = 0;
  while (((uint64_t)1 << l) < d) ++l;
  Div32 r;
  r.m = (uint32_t)((((uint64_t)1 << 32) * (((uint64_t)1 << l) - d)) / d + 1);
  r.sh1 = l < 1 ? l : 1;
  r.sh2 = l ? l - 1 : 0;
  return r;
}

__device__ __forceinline__ uint32_t div32(uint32_t n, const Div32& d) {
  const uint32_t t = __umulhi(d.m, n);
  return (t + ((n - t) >> d.sh1)) >> d.sh2;
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
  Div32 divP32;
  uint32_t W;
  uint32_t G;          // segment length (events, multiple of 8); CTA g owns the shots starting in [g*G, (g+1)*G)
  uint32_t nseg;       // segments = CTAs
  uint32_t maxt;       // tile status words per segment
  uint32_t num_tiles;  // nseg * maxt: status words (most of them stay 0)
  uint32_t num_sms;
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
  uint4* stage_a;      // staging table, indexed by sorted position: {label, size, sum tot, -}
  uint4* stage_b;      //                                            {sum tot*x (lo, hi), sum tot*y (lo, hi)}
  uint64_t* stage_c;   //                                            ToA of the brightest pixel
  uint64_t* stage_d;   //                                            sum tot*tof
  uint32_t mode;       // (2: as 0 but S0-S3 only; 3: S4-S5 on the caller's perm / label)
                       // 0: hit = connected component (north_star); 1: paper-literal mode, hit = local ToT
                       //    maximum of the box (lm_wx, lm_wy, W) and sums over that box (tpx3_localmax.cuh)
  uint32_t lm_wx, lm_wy;
  const uint64_t* label_base;   // [dev] or null: added (low 32 bits) to the label column (stream pushes, R24)
  PreArgs pre;                  // mode 4 only: trigger list, cut, timewalk table (tpx3_preprocess.cuh)
  const uint32_t* seg_kept;     // mode 4 only: events that survive the preprocessing in front of every segment
  uint32_t head;                // Inputs that are not 16-byte aligned (a chunk of a resident stream that starts at any event):
                                // the position-indexed arrays are passed moved DOWN by `head` elements to the alignment
                                // boundary, n counts those elements too, and the kernel starts at position `head`.
                                // Position p of the kernel is element p - head of the caller's arrays; the values it
                                // writes (perm, label) are in the caller's numbering.
  uint32_t labels_only;         // mode 5 only: stop after the labels (the general route of tpx3_cluster)
  const uint32_t* n_dev;        // [dev] or null: the event count is device state (a stream push): n, G, nseg, maxt and
                                // num_tiles above are upper bounds then (they size the grids) and every kernel
                                // derives the true ones from *n_dev; the staging table is laid out for the bound
};

// Segment length and status words per segment for n events in tiles of T (host and device: the ladder's rungs
// are sized on the device). Segments of 8 windows keep the re-read of a segment's first window at a few per
// cent; short inputs get shorter segments so that every SM has work. Two consecutive tiles that own something
// advance by at least T - 7 events together (what one leaves behind, at most a shot, the next one takes), hence
// the bound on status words. Measured and dropped: the stream's last wave in segments a quarter as long (cfg1
// 4 % slower: every segment start re-reads half a shot).
struct FusedSegs {
  uint32_t G, nseg, maxt;
};

__host__ __device__ inline FusedSegs fused_segs(uint64_t n, uint32_t T, uint32_t num_sms) {
  FusedSegs s;
  uint64_t G = 8ull * T;
  const uint64_t slots = (uint64_t)num_sms * (T <= 2048u ? 4u : (T <= 4096u ? 2u : 1u));   // resident CTAs
  const uint64_t want = slots * 8ull;                        // segments to aim for (load balance)
  if (n / G < want) {
    G = (n / want + 7ull) & ~7ull;
    // at least two windows per segment (a segment's first window re-reads half a shot), one when even that leaves
    // CTA slots empty (2^20 events: 0.105 -> 0.093 ms; 2^22-event stream pushes prefer two: 2.24 against 2.37 ms)
    const uint64_t gmin = n / (2ull * T) < slots ? (uint64_t)T : 2ull * T;
    if (G < gmin) G = gmin;
  }
  s.G = (uint32_t)G;
  s.nseg = (uint32_t)((n + G - 1) / G);
  s.maxt = 2u * (uint32_t)(G / T + 2u) + 2u;
  return s;
}

__host__ __device__ inline void compact_grid(uint32_t num_tiles, uint32_t num_sms, uint32_t* ctas, uint32_t* tiles_per_cta) {
  uint32_t c = num_tiles < num_sms * 8u ? num_tiles : num_sms * 8u;
  if (c == 0) c = 1;
  const uint32_t t = (num_tiles + c - 1) / c;
  *tiles_per_cta = t ? t : 1u;
  *ctas = t ? (num_tiles + t - 1) / t : 1u;
}

constexpr uint32_t kNone = 0xFFFFFFFFu;
constexpr int kHalvePre = 2;    // pointer-halving rounds before the deferred unions
constexpr int kHalvePost = 0;   // and before the root search
constexpr uint32_t kGold = 0x9E3779B1u;
constexpr uint32_t kTaskBase = 0xFFF8u;   // deferred-list entries k << 16 | (kTaskBase + direction) are scan tasks

// Shared-memory map (bytes). Records are uint2 {key, xy | tot << 16}.
//   A [0, 8T)    sorted records (unsorted input only)            } the hash table takes the 16T bytes
//   X [8T, 16T)  sort index buffers + warp digit counters        } next to the live records: A+X when
//   B [16T, 24T) records as loaded (input order)                 } the input was sorted, X+B otherwise
//   P [24T, 26T) bucket fill counters (u16) -> parent (u16)
//   L [26T, 27.5T) deferred links
// After the link step the hash region is reused: minidx u32[T] | head u32[T] | lab u16[T] |
// rootpos u16[T] | nxt u16[T]  (14T <= 16T).
template <int T>
struct FusedSmem {
  static constexpr int kRegA = 0;
  static constexpr int kRegX = 8 * T;
  static constexpr int kRegB = 16 * T;
  static constexpr int kPar = 24 * T;
  static constexpr int kList = 26 * T;
  static constexpr int kListCap = 3 * T / 8;           // deferred links the list holds
  static constexpr int kMisc = kList + 4 * kListCap;   // 27.5 T
  static constexpr int kMiscBytes = 512;
#ifdef TPX3_BULK_TOA   // experiment: the next window's ToA by cp.async.bulk + mbarrier into 8T more bytes
  static constexpr int kBulk = kMisc + kMiscBytes;
  static constexpr int kBytes = kBulk + (T <= 4096 ? 8 * T + 16 : 0);   // 8192-event windows: no room
#else
  static constexpr int kBytes = kMisc + kMiscBytes;
#endif
};

#ifdef TPX3_BULK_TOA
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, void* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\nWAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
#endif

struct FusedMisc {
  unsigned int lo, hi;         // first shot start of the window; first one at or after the segment's end
  unsigned int last;           // last shot start of the window
  unsigned int fail;
  unsigned int max_tof, max_sl;
  unsigned int n_roots;
  unsigned int n_list;         // deferred links pushed (may exceed the capacity: overflow)
  unsigned int skip;           // the call already failed in another tile
  unsigned int loose;          // some time cluster of the tile is wider than W ("within W" is not transitive)
  unsigned int min_tof;        // smallest time of flight among the events the tile loaded
  unsigned int s_next;               // mode 4: shot offset of the event the next tile starts at
  unsigned int kept_own, kept_pre;   // mode 4: events of the owned range / in front of it that survive the preprocessing
  unsigned int n_klist;        // other tiles: events whose S cell is empty (second pass of the link step)
  unsigned int warp_sums[33];
  unsigned int warp_cnt[33], warp_max[33];   // mode 4: surviving events / largest surviving key per warp (compaction)
};
static_assert(sizeof(FusedMisc) <= 512, "FusedMisc must fit kMiscBytes");

__device__ __forceinline__ uint32_t absdiff_u32(uint32_t a, uint32_t b) { return a > b ? a - b : b - a; }

// ---- union-find on 16-bit parents (two per 32-bit word) ----------------------------------------
__device__ __forceinline__ uint32_t uf_find(const uint16_t* par, uint32_t x) {
  uint32_t p;
  while ((p = par[x]) != x) x = p;
  return x;
}

// Hooks the larger root under the smaller with a compare-and-swap on the word that holds it; only a
// node that still is a root (parent == self) is ever changed, so no cycle can form.
__device__ __forceinline__ void uf_unite(uint16_t* par, uint32_t a, uint32_t b) {
  for (;;) {
    a = uf_find(par, a);
    b = uf_find(par, b);
    if (a == b) return;
    if (a < b) { const uint32_t t = a; a = b; b = t; }
    uint32_t* w = reinterpret_cast<uint32_t*>(par + (a & ~1u));
    const uint32_t sh = (a & 1u) * 16u;
    uint32_t old = *reinterpret_cast<volatile uint32_t*>(w);
    for (;;) {
      if (((old >> sh) & 0xFFFFu) != a) break;   // a was hooked meanwhile: find again
      const uint32_t nw = (old & ~(0xFFFFu << sh)) | (b << sh);
      const uint32_t prev = atomicCAS(w, old, nw);
      if (prev == old) return;
      old = prev;
    }
  }
}

// One tile per CTA. T = tile capacity (events), THREADS = T / 8.
// MODE 0: hit = connected component (north_star), S0-S5. MODE 1: paper-literal mode. MODE 2: S0-S3 only
// (tpx3_cluster). MODE 3: S4-S5 on the caller's (perm, label) (tpx3_centroid): the events are read THROUGH perm,
// in the caller's order, and the tile takes label[] as it is. (FusedArgs::mode holds the same number.)
template <int T, int THREADS, int MODE>
__global__ void __launch_bounds__(THREADS, (T <= 2048 ? 4 : (T <= 4096 ? 2 : 1))) k_fused_shot_tiles(FusedArgs a) {
  constexpr int IPT = T / THREADS;  // 8 events per thread
  constexpr bool kLM = MODE == 1 || MODE == 6;   // paper-literal mode (tpx3_localmax_centroid); 6: behind the general sort
  constexpr bool kLabelsOnly = MODE == 2;    // S0-S3 only: perm, label, hit count (tpx3_cluster)
  constexpr bool kGiven = MODE == 3;         // S4-S5 for a given (perm, label) (tpx3_centroid): no sort, no link
  constexpr bool kPerm = MODE == 3 || MODE == 5 || MODE == 6;   // the events are read through a given perm, which is not written
  constexpr bool kPre = MODE == 4;           // S0-S5 on a RAW stream: trigger assignment, ToF cut, timewalk, rebase in the load phase
  constexpr bool kCC = MODE == 0 || MODE == 2 || MODE == 4 || MODE == 5;   // hits are connected components found here
  static_assert(IPT == 8, "the 128-bit load phase assumes 8 events per thread");
  constexpr int WARPS = THREADS / 32;
  constexpr uint32_t NB = T;        // hash buckets of 4 slots (16 bytes each)
  constexpr uint32_t kHashShift = 32u - (T == 8192 ? 13u : (T == 4096 ? 12u : 11u));
  static_assert(T == 8192 || T == 4096 || T == 2048, "hash shift table");
  using L = FusedSmem<T>;
  extern __shared__ __align__(16) unsigned char smem[];
  FusedMisc* misc = reinterpret_cast<FusedMisc*>(smem + L::kMisc);
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;

  // ---- the CTA walks its segment tile by tile ---------------------------------------------------------
  const uint32_t seg = blockIdx.x;
  uint32_t n_ev = (uint32_t)a.n;     // positions fit 32 bits: a plan takes at most 2^28 events
  uint32_t seg_G = a.G, seg_n = a.nseg, seg_maxt = a.maxt;
  if (a.n_dev) {                     // a stream push: the count was decided on the device
    n_ev = *a.n_dev;
    const FusedSegs sg = fused_segs((uint64_t)n_ev, (uint32_t)T, a.num_sms);
    seg_G = sg.G; seg_n = sg.nseg; seg_maxt = sg.maxt;
    if (seg >= seg_n) return;        // the grid was sized for the largest count
  }
  const uint32_t seg_begin = seg * seg_G;
  const uint32_t seg_end = seg_begin + seg_G < n_ev ? seg_begin + seg_G : n_ev;
  const uint32_t P32 = (uint32_t)a.P;
  const uint32_t seg_first = seg == 0 ? a.head : seg_begin;   // (the elements below `head` are not the caller's)
  uint32_t tile_at = seg_first;     // where the next tile starts; a shot start except for the segment's first tile
  uint32_t kept_run = kPre ? a.seg_kept[seg] : 0u;   // mode 4: surviving events in front of tile_at
  uint64_t pre_next_s = 0;          // mode 4: trigger index of the event at tile_at, when the previous tile saw it
  bool pre_have_s = false;
  bool at_start = seg == 0;         // tile_at is known to be a shot start
  uint32_t tile_i = 0;              // status words written so far
  uint32_t seg_hits_run = 0;        // hits of the segment's tiles so far
  bool seg_failed = false;
#ifdef TPX3_BULK_TOA
  uint64_t* toa_s = reinterpret_cast<uint64_t*>(smem + L::kBulk);
  void* bulk_bar = smem + L::kBulk + 8 * T;
  uint32_t bulk_phase = 0;
  bool bulk_have = false;            // the window at tile_at has been requested into toa_s (block-uniform)
  constexpr bool kBulkOn = !kPerm && T <= 4096;
  if (kBulkOn) {
    if (tid == 0) {
      mbar_init(bulk_bar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    bulk_have = n_ev - (tile_at & ~7u) >= (uint32_t)T;
    if (bulk_have && tid == 0) {
      mbar_expect_tx(bulk_bar, 8u * T);
      bulk_g2s(toa_s, a.toa + (tile_at & ~7u), 8u * T, bulk_bar);
    }
  }
#endif
  for (;;) {
  // the next window's ToA is requested BEFORE the barrier that ends the previous tile: the loads touch no shared
  // memory, so the DRAM round trip runs under the wait for the previous tile's slowest warp
  const uint32_t base = tile_at & ~7u;                 // window start: aligned for the 128-bit loads
  const uint32_t skp = tile_at - base;                 // window positions below skp belong to the previous tile
  const uint32_t avail = n_ev - base;                  // > 0 by construction
  const uint32_t cnt = avail < (uint32_t)T ? avail : (uint32_t)T;  // events readable
  const uint32_t e_rel = seg_end - base > (uint32_t)T ? kNone : seg_end - base;   // segment end in the window
  const uint32_t p0 = tid * IPT;                       // this thread's 8 window positions

  // ---- load ToA (2 events per 128-bit load) ----------------------------------------------------
  uint64_t toa_r[IPT];
  if (kPerm) {      // position p of the given order is input event perm[p]
    if (p0 + IPT <= cnt) {
      const uint4 i0 = ldg_nc_v4(a.perm + base + p0), i1 = ldg_nc_v4(a.perm + base + p0 + 4);
      const uint32_t ix[IPT] = {i0.x, i0.y, i0.z, i0.w, i1.x, i1.y, i1.z, i1.w};
#pragma unroll
      for (int j = 0; j < IPT; ++j) toa_r[j] = a.toa[ix[j]];
    } else {
#pragma unroll
      for (int j = 0; j < IPT; ++j) toa_r[j] = (p0 + j < cnt) ? a.toa[a.perm[base + p0 + j]] : 0ull;
    }
#ifdef TPX3_BULK_TOA
  } else if (bulk_have) {
    mbar_wait(bulk_bar, bulk_phase);
    bulk_phase ^= 1u;
    const uint4* src = reinterpret_cast<const uint4*>(toa_s + p0);
#pragma unroll
    for (int j = 0; j < IPT / 2; ++j) {
      uint4 v = src[j];
      toa_r[2 * j] = ((uint64_t)v.y << 32) | v.x;
      toa_r[2 * j + 1] = ((uint64_t)v.w << 32) | v.z;
    }
#endif
  } else if (p0 + IPT <= cnt) {
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
  // the event just before this warp's first one (lanes > 0 get it from the previous lane); only the segment's
  // first tile needs it: a later tile starts at a known shot start
  uint64_t t_prev = 0;
  const bool has_prev = lane == 0 && p0 < cnt && base + p0 > 0 && !(at_start && p0 <= skp);
  if (has_prev) t_prev = kPerm ? a.toa[a.perm[base + p0 - 1]] : a.toa[base + p0 - 1];
  const uint64_t t_first = kPerm ? a.toa[a.perm[tile_at]] : a.toa[tile_at];
  // mode 4 needs the ToT for the timewalk correction before the keys can be laid out: requested here as well
  uint4 vt_early = make_uint4(0u, 0u, 0u, 0u);
  uint32_t tot_prev = 0;
  if (kPre) {
    if (p0 + IPT <= cnt) vt_early = ldg_nc_v4(a.tot + base + p0);
    else {
      uint32_t tt[IPT];
#pragma unroll
      for (int j = 0; j < IPT; ++j) tt[j] = p0 + j < cnt ? (uint32_t)a.tot[base + p0 + j] : 1u;
      vt_early = make_uint4(tt[0] | (tt[1] << 16), tt[2] | (tt[3] << 16), tt[4] | (tt[5] << 16), tt[6] | (tt[7] << 16));
    }
    if (has_prev) tot_prev = a.tot[base + p0 - 1];
  }
  __syncthreads();                  // the previous tile is done with the shared memory
  if (tid == 0) {
    misc->lo = kNone;
    misc->hi = kNone;
    misc->last = 0;
    // another tile already gave up: this attempt is lost, do not spend time on it (the next attempt — a
    // variant with longer shots, or the general kernels — is enqueued behind; k_fallback_dispatch)
    misc->skip = tile_at == seg_first ? atomicAdd(&a.ctrl->fused_fail, 0u) : 0u;
    misc->fail = 0;
    misc->max_tof = 0;
    misc->loose = 0;
    misc->min_tof = kNone;
    misc->n_klist = 0;
    misc->kept_own = 0;
    misc->kept_pre = 0;
    misc->max_sl = 0;
    misc->n_roots = 0;
    misc->n_list = 0;
  }
  __syncthreads();
  if (misc->skip != 0u || tile_i >= seg_maxt) { seg_failed = tile_i >= seg_maxt; break; }
  // reference time of the tile: start of the shot its first event belongs to
  uint64_t ref;
  uint64_t s_ref = 0;               // mode 4: trigger index of the tile's first event
  // ---- shot offsets and times of flight; shot boundaries ----------------------------------------
  uint32_t sl[IPT], tof[IPT];
  uint32_t keepm = 0xFFu;           // mode 4: bit j = event p0 + j survives the preprocessing
  bool keepp = true;                // ... and so does the event in front of this thread's first one
  uint32_t slp, tofp;
  bool start0, viol0;
  bool bad = false;
  if constexpr (kPre) {
    // Preprocessing in the load phase (R23; the arithmetic of tpx3_preprocess.cuh): shot =
    // index of the most recent trigger, ToF = ToA - trigger, dropped beyond the cut, ToF' = ToF - table[ToT] clamped
    // to [0, P - 1]. No division: the shot offset is a difference of trigger indices. Every event keeps the shot
    // of its trigger period, dropped or not, so shot boundaries are found on the raw stream.
    PreWindow* win = reinterpret_cast<PreWindow*>(smem + L::kList);     // the list region is free until the link step
    if (pre_have_s) {     // the previous tile knew the trigger of this tile's first event: no search for the window
      if (tid == 0) {
        const uint64_t h0 = pre_next_s > 8ull ? pre_next_s - 8ull : 0ull;
        win->h0 = h0;
        win->valid = (uint32_t)(a.pre.n_trig - h0 < (uint64_t)kPreWin ? a.pre.n_trig - h0 : (uint64_t)kPreWin);
      }
      __syncthreads();
      if (tid < kPreWin) win->trig[tid] = tid < win->valid ? a.pre.trig[win->h0 + tid] : ~0ull;
      __syncthreads();
    } else {
      pre_window_fill(a.pre, tile_at, win);
    }
    {
      uint64_t s0;
      s_ref = pre_find(a.pre, win, t_first, s0) ? s0 : 0ull;
    }
    ref = (a.pre.shot_base + s_ref) * a.P;
    // a thread's 8 events are neighbours in the stream, so nearly always in the trigger period of the one before:
    // the last period found is kept ([c_lo, c_hi) = trigger c_s up to the next one) and tried first
    uint64_t c_s = 0, c_lo = 1, c_hi = 0;            // empty interval
    auto trig_at = [&](uint64_t s1) -> uint64_t {
      const uint64_t o = s1 - win->h0;
      return o < (uint64_t)win->valid ? win->trig[o] : a.pre.trig[s1];
    };
    auto pre_one = [&](uint64_t t, uint32_t tt, uint64_t& s_out, uint32_t& tof_out) -> bool {   // true: kept
      uint64_t s1 = c_s;
      if (!(t >= c_lo && t < c_hi)) {
        const bool has = pre_find(a.pre, win, t, s1);
        if (!has) { s_out = 0ull; tof_out = 0; return false; }   // no trigger yet: counted to shot 0, dropped
        c_s = s1;
        c_lo = trig_at(s1);
        c_hi = s1 + 1ull < a.pre.n_trig ? trig_at(s1 + 1ull) : ~0ull;
      }
      s_out = s1;
      tof_out = 0;
      const uint64_t tf = t - c_lo;
      if (tf > a.pre.cut) return false;
      long long corr = 0;
      if (a.pre.table_len) corr = a.pre.table[tt < a.pre.table_len ? tt : a.pre.table_len - 1u];
      long long tc = (long long)tf - corr;
      if (tc < 0) tc = 0;
      if ((uint64_t)tc > a.P - 1ull) tc = (long long)(a.P - 1ull);
      tof_out = (uint32_t)tc;                        // P <= 2^24
      return true;
    };
    keepm = 0;
    const uint32_t tw[4] = {vt_early.x, vt_early.y, vt_early.z, vt_early.w};
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const bool in = p0 + j < cnt && p0 + j >= skp;
      sl[j] = 0; tof[j] = 0;
      if (in) {
        uint64_t s1;
        const bool keep = pre_one(toa_r[j], (tw[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu, s1, tof[j]);
        const uint64_t d = s1 - s_ref;
        if (d >> 31) bad = true;                     // an earlier shot behind a later one, or out of range
        sl[j] = (uint32_t)d;
        if (keep) keepm |= 1u << j;
      }
    }
    slp = __shfl_up_sync(0xffffffffu, sl[IPT - 1], 1);
    tofp = __shfl_up_sync(0xffffffffu, tof[IPT - 1], 1);
    keepp = __shfl_up_sync(0xffffffffu, (keepm >> (IPT - 1)) & 1u, 1) != 0u;
    start0 = sl[0] != slp; viol0 = sl[0] < slp;
    if (lane == 0) {
      if (!has_prev) { start0 = p0 < cnt; viol0 = false; slp = 0; tofp = 0; keepp = false; }
      else {
        uint64_t s1;
        keepp = pre_one(t_prev, tot_prev, s1, tofp);
        if (s1 < s_ref) { start0 = true; viol0 = false; slp = 0; keepp = false; }       // previous shot
        else {
          const uint64_t d = s1 - s_ref;
          slp = (d >> 31) ? kNone : (uint32_t)d;
          start0 = sl[0] != slp;
          viol0 = sl[0] < slp;
        }
      }
    }
  } else {
  const uint64_t s_base = div64(t_first, a.divP);
  ref = s_base * a.P;
#pragma unroll
  for (int j = 0; j < IPT; ++j) {
    const uint64_t r64 = toa_r[j] - ref;
    const bool in = p0 + j < cnt && p0 + j >= skp;
    const uint32_t rel = in ? (uint32_t)r64 : 0u;
    sl[j] = div32(rel, a.divP32);
    tof[j] = rel - sl[j] * P32;
    if (in && (r64 >> 32) != 0ull) {   // rare: more than 2^32 ticks after the tile's first shot (or before it)
      const uint64_t q = div64(r64, a.divP);
      if (q >> 32) bad = true;
      sl[j] = (uint32_t)q;
      tof[j] = (uint32_t)(r64 - q * a.P);
    }
  }
  slp = __shfl_up_sync(0xffffffffu, sl[IPT - 1], 1);
  tofp = __shfl_up_sync(0xffffffffu, tof[IPT - 1], 1);
  start0 = sl[0] != slp; viol0 = sl[0] < slp;
  if (lane == 0) {
    if (!has_prev) { start0 = p0 < cnt; viol0 = false; slp = 0; tofp = 0; }          // position 0 of the stream
    else if (t_prev < ref) { start0 = true; viol0 = false; slp = 0; tofp = 0; }        // previous shot
    else {
      const uint64_t r64 = t_prev - ref;
      const uint64_t q = div64(r64, a.divP);
      slp = (q >> 32) ? kNone : (uint32_t)q;
      tofp = (uint32_t)(r64 - q * a.P);
      start0 = sl[0] != slp;
      viol0 = sl[0] < slp;
    }
  }
  }   // not mode 4
  uint32_t bnd = 0;  // bit j: event p0+j starts a shot
  bool viol = false;
  {
    if (p0 < cnt && p0 >= skp) {
      if (start0 || (at_start && p0 == skp)) bnd |= 1u;
      if (viol0 && !(at_start && p0 == skp)) viol = true;
    }
#pragma unroll
    for (int j = 1; j < IPT; ++j) {
      if (p0 + j < cnt && p0 + j >= skp) {
        const bool first = at_start && p0 + j == skp;   // the known shot start of a chained tile
        if (first || sl[j] != sl[j - 1]) bnd |= 1u << j;
        if (!first && sl[j] < sl[j - 1]) viol = true;
      }
    }
  }
  // lo = first shot start of the window; last = the last one; hi = the first one at or after the segment's end
  {
    uint32_t my_lo = kNone, my_hi = kNone, my_last = 0, mt = 0, ml = 0, mn = kNone;
#pragma unroll
    for (int j = IPT - 1; j >= 0; --j) {
      if (bnd & (1u << j)) {
        my_lo = p0 + j;
        if (p0 + j >= e_rel) my_hi = p0 + j;
        my_last = max(my_last, p0 + (uint32_t)j);
      }
      mt = max(mt, tof[j]);
      ml = max(ml, sl[j]);
      if (p0 + j < cnt && p0 + j >= skp && ((keepm >> j) & 1u)) mn = min(mn, tof[j]);
    }
    mn = __reduce_min_sync(0xffffffffu, mn);
    my_lo = __reduce_min_sync(0xffffffffu, my_lo);
    my_hi = __reduce_min_sync(0xffffffffu, my_hi);
    my_last = __reduce_max_sync(0xffffffffu, my_last);
    mt = __reduce_max_sync(0xffffffffu, mt);
    ml = __reduce_max_sync(0xffffffffu, ml);
    const uint32_t any_bad = __any_sync(0xffffffffu, bad || viol);
    if (lane == 0) {
      if (my_lo != kNone) atomicMin(&misc->lo, my_lo);
      if (my_hi != kNone) atomicMin(&misc->hi, my_hi);
      if (my_last) atomicMax(&misc->last, my_last);
      if (mt) atomicMax(&misc->max_tof, mt);
      if (mn != kNone) atomicMin(&misc->min_tof, mn);
      if (ml) atomicMax(&misc->max_sl, ml);
      if (any_bad) misc->fail = 1;
    }
  }
  // meanwhile: clear the hash region for sorted input (A + X) and the bucket counters
  {
    uint4* z = reinterpret_cast<uint4*>(smem + L::kRegA);
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int q = 0; q < 16 * T / 16 / THREADS; ++q) z[q * THREADS + tid] = zero;
    uint4* zc = reinterpret_cast<uint4*>(smem + L::kPar);
    if (tid < 2 * T / 16) zc[tid] = zero;
    static_assert(2 * T / 16 <= THREADS, "counter clear");
  }
  __syncthreads();
  // Owned range [lo, hi) of the window: whole shots that start before the segment's end and end inside the
  // window. The end of the stream counts as a shot start.
  uint32_t lo = misc->lo, hi;
  bool failed = misc->fail != 0;
  uint32_t next_at;               // where the next tile of this segment starts (>= seg_end: none)
  {
    const bool to_end = base + cnt >= n_ev;
    const uint32_t last = to_end ? cnt : misc->last;          // misc->last >= lo whenever lo exists
    if (lo == kNone) {            // no shot starts in this window: nothing owned, look further on
      lo = hi = 0;
      next_at = base + cnt;
    } else if (lo >= e_rel) {     // the first shot start belongs to the next segment
      hi = lo;
      next_at = seg_end;
    } else {
      hi = min(last, misc->hi);   // misc->hi: kNone when the segment's end is not in sight
      next_at = base + hi;
      if (hi == lo) {             // not even the first shot ends inside the window
        if (lo > skp) next_at = base + lo;     // start again with the window at that shot's start
        else failed = true;                    // a shot longer than the window
      }
    }
    if (to_end && next_at >= base + cnt) next_at = n_ev;
  }
#ifdef TPX3_BULK_TOA
  if (kBulkOn) {  // every thread has its ToA in registers (two barriers ago): the buffer may take the next window
    bulk_have = !failed && next_at < seg_end && n_ev - (next_at & ~7u) >= (uint32_t)T;
    if (bulk_have && tid == 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(bulk_bar, 8u * T);
      bulk_g2s(toa_s, a.toa + (next_at & ~7u), 8u * T, bulk_bar);
    }
  }
#endif
  // key layout: 2^tb > max tof + W, so keys of different shots differ by more than W
  const uint32_t tspan = misc->max_tof + a.W;
  const uint32_t tb = tspan ? 32u - (uint32_t)__clz(tspan) : 0u;
  const uint32_t sbits = misc->max_sl ? 32u - (uint32_t)__clz(misc->max_sl) : 0u;
  if (tb + sbits > (kPre ? 31u : 32u)) failed = true;      // mode 4 keeps the key 0xFFFFFFFF for dropped events
  const uint32_t mm_raw = failed ? 0u : hi - lo;   // owned events of the window; a failed tile owns nothing
  uint32_t mm = mm_raw;                            // owned events that are clustered (mode 4: those that survive)
  const uint32_t tmask = tb >= 32u ? 0xFFFFFFFFu : ((1u << tb) - 1u);
  const uint32_t raw_base = base + lo;              // input position of the window's first owned event (n <= 2^28)
  uint32_t out_base = raw_base;                     // global sorted position of local rank 0
  if constexpr (kPre) {
    // surviving events of the owned range and of what this window skips in front of it (counted into kept_run)
    const uint32_t pre_end = misc->lo == kNone ? cnt : lo;
    uint32_t c_own = 0, c_pre = 0;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t q = p0 + (uint32_t)j, kb = (keepm >> j) & 1u;
      c_own += (q >= lo && q < lo + mm_raw) ? kb : 0u;
      c_pre += (q >= skp && q < pre_end) ? kb : 0u;
    }
    c_own = __reduce_add_sync(0xffffffffu, c_own);
    c_pre = __reduce_add_sync(0xffffffffu, c_pre);
    if (lane == 0) {
      if (c_own) atomicAdd(&misc->kept_own, c_own);
      if (c_pre) atomicAdd(&misc->kept_pre, c_pre);
    }
    // the trigger of the event the next tile starts at (read at the end of this tile)
    const uint32_t nrel = next_at - base;
    if (nrel >= p0 && nrel < p0 + IPT && nrel < cnt && nrel >= skp) misc->s_next = sl[nrel - p0];
  }

  // ---- records as loaded -> region B, 128-bit loads of x / y / tot ------------------------------
  uint2* recB = reinterpret_cast<uint2*>(smem + L::kRegB);
  // The time-cluster check (below) is skipped when all times of flight lie within W anyway, and when the last
  // call on this workspace found hardly any tight tile (the hint; every 16th call looks again).
  const bool cl_wide = misc->max_tof - misc->min_tof > a.W;
  const bool cl_scan = kCC && cl_wide && (a.ctrl->scan_hint != kScanSkip || (a.ctrl->calls & 15u) == 0u);
  bool uns = false;
  uint32_t cl_last_start = 0, cl_lead_last = 0;   // time-cluster check on the keys in registers
  bool cl_have_lead = false, cl_loose = false;
  uint32_t kp_cnt = 0, kp_max = 0, kp_first = kNone;   // mode 4: surviving owned events of this thread, their largest / first key
  bool kp_viol = false;                                 // ... and whether they descend somewhere
  if (mm_raw && p0 < hi && p0 + IPT > lo) {
    uint32_t key_r[IPT];
#pragma unroll
    for (int j = 0; j < IPT; ++j)
      key_r[j] = ((keepm >> j) & 1u) ? ((tb >= 32u ? 0u : (sl[j] << tb)) | tof[j]) : 0xFFFFFFFFu;   // dropped: behind all others
    const uint32_t keyp = keepp ? ((tb >= 32u ? 0u : (slp << tb)) | tofp) : 0xFFFFFFFFu;
    if constexpr (kPre) {   // for the compaction below: this thread's surviving owned events
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        const uint32_t q = p0 + (uint32_t)j;
        if (q >= lo && q < hi && ((keepm >> j) & 1u)) {
          if (kp_cnt && key_r[j] < kp_max) kp_viol = true;
          if (!kp_cnt) kp_first = key_r[j];
          kp_max = max(kp_max, key_r[j]);
          ++kp_cnt;
        }
      }
    }
    // already in (shot, ToA) order? (configs 0-3 arrive sorted; config 4 does not)
    if (p0 > lo && key_r[0] < keyp) uns = true;
#pragma unroll
    for (int j = 1; j < IPT; ++j)
      if (p0 + j > lo && p0 + j < hi && key_r[j] < key_r[j - 1]) uns = true;
    // time clusters (see "are the time clusters of the tile tight?" below): for a tile that is in order the
    // keys are at hand here, in registers, in the blocked arrangement the check wants
    if (cl_scan) {
      uint32_t cur = 0;
      bool have_cur = false;
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        const uint32_t q = p0 + (uint32_t)j;
        if (q >= lo && q < hi) {
          const uint32_t key = key_r[j], prev = j ? key_r[j - 1] : keyp;
          if (q == lo || key - prev > a.W) { cur = key; have_cur = true; cl_last_start = key; }
          else if (have_cur) { if (key - cur > a.W) cl_loose = true; }
          else { cl_lead_last = key; cl_have_lead = true; }
        }
      }
    }
    uint4 vx, vy, vt;
    if (!kPerm && p0 + IPT <= cnt) {
      vx = ldg_nc_v4(a.x + base + p0);
      vy = ldg_nc_v4(a.y + base + p0);
      vt = kPre ? vt_early : ldg_nc_v4(a.tot + base + p0);
    } else {
      uint16_t tx[IPT], ty[IPT], tt[IPT];
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        bool ok = p0 + j < cnt;
        const uint64_t src = ok ? (kPerm ? (uint64_t)a.perm[base + p0 + j] : base + p0 + j) : 0ull;
        tx[j] = ok ? a.x[src] : (uint16_t)0;
        ty[j] = ok ? a.y[src] : (uint16_t)0;
        tt[j] = ok ? a.tot[src] : (uint16_t)1;
      }
      vx = make_uint4(tx[0] | ((uint32_t)tx[1] << 16), tx[2] | ((uint32_t)tx[3] << 16),
                      tx[4] | ((uint32_t)tx[5] << 16), tx[6] | ((uint32_t)tx[7] << 16));
      vy = make_uint4(ty[0] | ((uint32_t)ty[1] << 16), ty[2] | ((uint32_t)ty[3] << 16),
                      ty[4] | ((uint32_t)ty[5] << 16), ty[6] | ((uint32_t)ty[7] << 16));
      vt = make_uint4(tt[0] | ((uint32_t)tt[1] << 16), tt[2] | ((uint32_t)tt[3] << 16),
                      tt[4] | ((uint32_t)tt[5] << 16), tt[6] | ((uint32_t)tt[7] << 16));
    }
    const uint32_t xs[4] = {vx.x, vx.y, vx.z, vx.w}, ys[4] = {vy.x, vy.y, vy.z, vy.w},
                   ts[4] = {vt.x, vt.y, vt.z, vt.w};
    if (a.flags & TPX3_FLAG_VALIDATE_INPUT) {
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
    // record word 1: x | y << 8 | tot << 16
    uint32_t w1[IPT];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      w1[2 * q] = (xs[q] & 0xFFu) | ((ys[q] & 0xFFu) << 8) | (ts[q] << 16);
      w1[2 * q + 1] = ((xs[q] >> 16) & 0xFFu) | (((ys[q] >> 16) & 0xFFu) << 8) | (ts[q] & 0xFFFF0000u);
    }
    uint4* dst = reinterpret_cast<uint4*>(recB + p0);
#pragma unroll
    for (int q = 0; q < 4; ++q) dst[q] = make_uint4(key_r[2 * q], w1[2 * q], key_r[2 * q + 1], w1[2 * q + 1]);
  }
  uint32_t cl_carry = 0;
  if (cl_scan) {
    uint32_t cl_inc = cl_last_start;   // prefix maximum of the cluster starts: 0 = "none" is the identity
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, cl_inc, o);
      if (lane >= (uint32_t)o) cl_inc = max(cl_inc, t);
    }
    if (lane == 31) misc->warp_sums[warp] = cl_inc;
    cl_carry = __shfl_up_sync(0xffffffffu, cl_inc, 1);
    if (lane == 0) cl_carry = 0;
  }
  uint32_t kp_excl = 0, kp_pmax = 0;
  if constexpr (kPre) {   // warp scans: surviving events in front of this thread (sum) and their largest key (max)
    uint32_t ic = kp_cnt, im = kp_max;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t tc = __shfl_up_sync(0xffffffffu, ic, o), tm = __shfl_up_sync(0xffffffffu, im, o);
      if (lane >= (uint32_t)o) { ic += tc; im = max(im, tm); }
    }
    if (lane == 31) { misc->warp_cnt[warp] = ic; misc->warp_max[warp] = im; }
    kp_excl = ic - kp_cnt;
    kp_pmax = __shfl_up_sync(0xffffffffu, im, 1);
    if (lane == 0) kp_pmax = 0;
  }
  const bool out_of_order = __syncthreads_or(!kGiven && uns ? 1 : 0) != 0;
  const bool unsorted = !kPerm && out_of_order;    // a given perm is never re-sorted (mode 5: it IS the (shot, ToA) order)
  if ((MODE == 5 || MODE == 6) && out_of_order) failed = true;
  if constexpr (kPre) {     // (a tile whose keys ascend has its dropped events, key 0xFFFFFFFF, at the end: first mm records)
    mm = failed ? 0u : misc->kept_own;
    out_base = kept_run + misc->kept_pre;
    kept_run = out_base + mm;
  }
  // what the tile writes as VALUES is in the caller's numbering (FusedArgs::head)
  const uint32_t out_val = out_base - a.head, raw_val = raw_base - a.head;
  if (cl_wide && !cl_scan && tid == 0) misc->loose = 1u;   // not checked: treated as not tight
  if (!unsorted && cl_scan) {
    for (uint32_t w = 0; w < warp; ++w) cl_carry = max(cl_carry, misc->warp_sums[w]);
    if (cl_have_lead && cl_lead_last - cl_carry > a.W) cl_loose = true;   // position lo starts a cluster
    if (cl_loose) misc->loose = 1u;
  }

  // ---- S1: stable order of the owned events by (shot offset, tof) (only if needed) -------------------
  uint2* recA = reinterpret_cast<uint2*>(smem + L::kRegA);
  if (unsorted) {
    uint16_t* buf0 = reinterpret_cast<uint16_t*>(smem + L::kRegX);
    uint16_t* buf1 = buf0 + T;
    // sort key without the gap between the tof bits and the shot bits
    const uint32_t tofb = misc->max_tof ? 32u - (uint32_t)__clz(misc->max_tof) : 1u;
    const uint32_t key_bits = tofb + sbits;
    const uint16_t* fin;
    // (0) Mode 4: a tile is usually out of order only because dropped events (key 0xFFFFFFFF) sit between the
    // surviving ones. If the surviving keys ascend, their ranks are a prefix count: no sort.
    bool compacted = false;
    if constexpr (kPre) {
      for (uint32_t w = 0; w < warp; ++w) { kp_excl += misc->warp_cnt[w]; kp_pmax = max(kp_pmax, misc->warp_max[w]); }
      const bool desc = kp_viol || (kp_cnt && kp_first < kp_pmax);
      compacted = __syncthreads_or(desc ? 1 : 0) == 0;
      if (compacted) {
        uint32_t r = kp_excl;
#pragma unroll
        for (int j = 0; j < IPT; ++j) {
          const uint32_t q = p0 + (uint32_t)j;
          if (q >= lo && q < hi && ((keepm >> j) & 1u)) buf1[r++] = (uint16_t)(q - lo);
        }
        fin = buf1;
        __syncthreads();
      }
    }
    if (!compacted) {
    // (a) Rank by counting. What has to be computed is the RANK of every event among the composite values
    // (key, input position), which are all different, so nothing here needs to be stable. Detector streams hold
    // few distinct keys per tile (time of flight is quantised and bunched: 5 mass peaks of about 100 ticks on
    // config 4), so: bitmap of the keys that occur (region A, already zero) -> dense key number by a prefix
    // popcount -> events per dense key (shared-memory atomics; the returned value is the event's arrival slot
    // inside its key group) -> offsets by an exclusive scan -> the few events of one key are ordered by input
    // position: by position block through the counts, inside a block with a count of smaller positions. About 60 thread instructions per event; the two-pass LSD sort
    // below (one ballot per digit bit) took 42 % of the kernel's instructions on config 4 (profiles/r02_*).
    constexpr uint32_t kBitmapBits = 32u * (uint32_t)T;           // 4T bytes of region A
    uint32_t* bitmap = reinterpret_cast<uint32_t*>(smem + L::kRegA);             // [T] words
    uint16_t* wpre = reinterpret_cast<uint16_t*>(smem + L::kRegA + 4 * T);       // [T] dense number of a word's first key
    uint16_t* gbase = reinterpret_cast<uint16_t*>(smem + L::kRegA + 4 * T);      // [T + 1] offsets (over wpre, once dead)
    // events per (dense key, block of THREADS input positions): eight 4-bit counts per word. A key group's
    // members of different position blocks are ordered by the block; only the members of one block (rarely
    // more than one) are left to the count of smaller positions.
    uint32_t* gcnt = reinterpret_cast<uint32_t*>(smem + L::kRegX + 4 * T);       // [T] words
    static_assert(IPT == 8, "eight position blocks = eight 4-bit counts per word");
    bool counted = key_bits <= 31u && (1u << key_bits) <= kBitmapBits;
    if (counted) {
      const uint32_t nwords = ((1u << key_bits) + 31u) >> 5;
      uint32_t sk_r[IPT];
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        const uint32_t k = (uint32_t)j * THREADS + tid;
        uint32_t sk = kNone;                  // kNone: no event here (mode 4: or one the preprocessing dropped)
        if (k < mm_raw) {
          const uint32_t key = recB[lo + k].x;
          if (!kPre || key != 0xFFFFFFFFu) {
            sk = ((key >> tb) << tofb) | (key & tmask);
            atomicOr(&bitmap[sk >> 5], 1u << (sk & 31u));
          }
        }
        sk_r[j] = sk;
      }
      __syncthreads();
      {   // dense key numbers: exclusive prefix popcount over the bitmap words, 8 consecutive words per thread
        uint32_t c[IPT], sum = 0;
        const uint4 w0 = *reinterpret_cast<const uint4*>(bitmap + p0), w1 = *reinterpret_cast<const uint4*>(bitmap + p0 + 4);
        const uint32_t ww[IPT] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
        for (int j = 0; j < IPT; ++j) { c[j] = p0 + j < nwords ? (uint32_t)__popc(ww[j]) : 0u; sum += c[j]; }
        uint32_t inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
          if (lane >= (uint32_t)o) inc += t;
        }
        if (lane == 31) misc->warp_sums[warp] = inc;
        __syncthreads();
        uint32_t run = inc - sum;
        for (uint32_t w = 0; w < warp; ++w) run += misc->warp_sums[w];
        uint32_t pk[4];
#pragma unroll
        for (int j = 0; j < IPT; j += 2) {
          pk[j >> 1] = run | ((run + c[j]) << 16);
          run += c[j] + c[j + 1];
        }
        *reinterpret_cast<uint4*>(wpre + p0) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      }
      __syncthreads();
      // Counter fields: first eight 4-bit counts per key (position blocks of THREADS events). If one of them
      // overflows — 16 events of one key inside one position block: electron VMI, where a shot's few hundred
      // events share 95 ticks — the step is redone with four 8-bit counts (blocks of 2 * THREADS events); the
      // members of one field are then ordered by the count of smaller positions, whatever their number.
      // (Two instantiations of one generic lambda: the field width is a compile-time constant in both.)
      auto rank_by_fields = [&](auto cb_tag) -> bool {              // false: a field overflowed, nothing usable written
        constexpr uint32_t cb = decltype(cb_tag)::value, fmask = (1u << cb) - 1u;
        auto fsum = [](uint32_t w) -> uint32_t {                    // sum of the fields of a counter word
          if (cb == 4u) {
            w = (w & 0x0F0F0F0Fu) + ((w >> 4) & 0x0F0F0F0Fu);
            return (w * 0x01010101u) >> 24;
          }
          return (w & 0xFFu) + ((w >> 8) & 0xFFu) + ((w >> 16) & 0xFFu) + (w >> 24);
        };
        uint32_t dk_r[IPT];   // dense key | arrival slot inside (key, position block) << 16
        bool big = false;
#pragma unroll
        for (int j = 0; j < IPT; ++j) {
          dk_r[j] = kNone;
          if (sk_r[j] != kNone) {
            const uint32_t sk = sk_r[j], w = sk >> 5;
            const uint32_t dk = (uint32_t)wpre[w] + (uint32_t)__popc(bitmap[w] & ((1u << (sk & 31u)) - 1u));
            const uint32_t sh = cb == 4u ? 4u * (uint32_t)j : 8u * ((uint32_t)j >> 1);
            const uint32_t r = (atomicAdd(&gcnt[dk], 1u << sh) >> sh) & fmask;
            big = big || r == fmask;
            dk_r[j] = dk | (r << 16);
          }
        }
        if (__syncthreads_or(big ? 1 : 0)) return false;
        {   // offsets: exclusive scan of the group sizes, 8 consecutive dense keys per thread (at most mm <= T keys)
          const uint4 q0 = *reinterpret_cast<const uint4*>(gcnt + p0), q1 = *reinterpret_cast<const uint4*>(gcnt + p0 + 4);
          const uint32_t qw[IPT] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w};
          uint32_t c[IPT], sum = 0;
#pragma unroll
          for (int j = 0; j < IPT; ++j) { c[j] = fsum(qw[j]); sum += c[j]; }
          uint32_t inc = sum;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= (uint32_t)o) inc += t;
          }
          if (lane == 31) misc->warp_sums[warp] = inc;
          __syncthreads();
          uint32_t run = inc - sum;
          for (uint32_t w = 0; w < warp; ++w) run += misc->warp_sums[w];
          uint32_t pk[4];
#pragma unroll
          for (int j = 0; j < IPT; j += 2) {
            pk[j >> 1] = run | ((run + c[j]) << 16);
            run += c[j] + c[j + 1];
          }
          *reinterpret_cast<uint4*>(gbase + p0) = make_uint4(pk[0], pk[1], pk[2], pk[3]);   // wpre is dead
        }
        __syncthreads();
        uint32_t b0_r[IPT];
#pragma unroll
        for (int j = 0; j < IPT; ++j) {
          const uint32_t k = (uint32_t)j * THREADS + tid;
          b0_r[j] = 0;
          if (dk_r[j] != kNone) {
            const uint32_t dk = dk_r[j] & 0xFFFFu, r = dk_r[j] >> 16;
            const uint32_t w = gcnt[dk];
            const uint32_t sh = cb == 4u ? 4u * (uint32_t)j : 8u * ((uint32_t)j >> 1);
            // the group's members of earlier position blocks come first
            const uint32_t b0 = (uint32_t)gbase[dk] + fsum(w & ((1u << sh) - 1u)), m = (w >> sh) & fmask;
            b0_r[j] = b0 | (m << 16);
            if (m == 1u) buf1[b0] = (uint16_t)k;      // alone with its key in its position block: final position
            else buf0[b0 + r] = (uint16_t)k;          // the sub-group's members in arrival order
          }
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < IPT; ++j) {
          const uint32_t k = (uint32_t)j * THREADS + tid;
          const uint32_t b0 = b0_r[j] & 0xFFFFu, m = b0_r[j] >> 16;
          if (m > 1u) {
            uint32_t c = 0;
            for (uint32_t q = 0; q < m; ++q) c += (uint32_t)buf0[b0 + q] < k ? 1u : 0u;   // members at earlier input positions
            buf1[b0 + c] = (uint16_t)k;
          }
        }
        return true;
      };
      bool ranked = rank_by_fields(std::integral_constant<uint32_t, 4u>{});
      if (!ranked) {
        for (uint32_t i = tid; i < (uint32_t)T; i += THREADS) gcnt[i] = 0u;     // again, with wider fields
        __syncthreads();
        ranked = rank_by_fields(std::integral_constant<uint32_t, 8u>{});
      }
      if (ranked) fin = buf1;
      else counted = false;      // 256 events of one key in one position block: the LSD sort below
      __syncthreads();
    }
    if (!counted) {
    // (b) Stable LSD radix sort of 16-bit local indices, digits ranked per warp with ballots.
    // digit counters per warp, 16 bit (a count is <= T); one thread per digit value, so up to 9-bit digits
    // with >= 512 threads
    constexpr uint32_t DB = THREADS >= 512 ? 9u : 8u;
    constexpr uint32_t RMAX = 1u << DB;
    uint16_t* wcnt = reinterpret_cast<uint16_t*>(smem + L::kRegX + 4 * T);  // [WARPS][RMAX]
    static_assert(WARPS * RMAX * 2 <= 4 * T && T <= 65535, "warp digit counters");
    const uint32_t npass = (key_bits + DB - 1u) / DB;
    const uint32_t dbits = (key_bits + npass - 1u) / npass;         // <= DB
    const uint32_t radix = 1u << dbits, dmask = radix - 1u;
    const uint32_t lt = lanemask_lt();
    for (uint32_t pass = 0; pass < npass; ++pass) {
      const uint16_t* src = (pass & 1u) ? buf1 : buf0;
      uint16_t* dst = (pass & 1u) ? buf0 : buf1;
      const uint32_t shift = pass * dbits;
      for (uint32_t i = tid; i < WARPS * RMAX / 2u; i += THREADS) reinterpret_cast<uint32_t*>(wcnt)[i] = 0u;
      __syncthreads();
      uint32_t e_src[IPT], e_dig[IPT], e_rank[IPT];
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        const uint32_t k = warp * (32u * IPT) + (uint32_t)j * 32u + lane;   // warps own ascending slices
        // first pass: the owned events as loaded (mode 4: but for the dropped ones); later passes: the mm survivors
        bool valid = pass == 0 ? k < mm_raw : k < mm;
        const uint32_t s = valid ? (pass == 0 ? k : (uint32_t)src[k]) : 0u;
        const uint32_t key = valid ? recB[lo + s].x : 0u;
        if (kPre && key == 0xFFFFFFFFu) valid = false;
        const uint32_t sk = ((key >> tb) << tofb) | (key & tmask);
        const uint32_t d = (sk >> shift) & dmask;
        // lanes holding the same digit (ballot per digit bit; match.any is 20x dearer on sm_100)
        uint32_t peers = __ballot_sync(0xffffffffu, valid);
        for (uint32_t bit = 0; bit < dbits; ++bit) {
          const bool one = (d >> bit) & 1u;
          const uint32_t bal = __ballot_sync(0xffffffffu, one);
          peers &= one ? bal : ~bal;
        }
        const uint32_t lr = __popc(peers & lt);
        const uint32_t c0 = valid ? (uint32_t)wcnt[warp * RMAX + d] : 0u;
        __syncwarp();
        if (valid && lr == 0) wcnt[warp * RMAX + d] = (uint16_t)(c0 + __popc(peers));
        __syncwarp();
        e_src[j] = s;
        e_dig[j] = valid ? d : RMAX;                                        // RMAX: "no event"
        e_rank[j] = c0 + lr;
      }
      __syncthreads();
      // digit d (thread d): exclusive prefix over warps, then over digits
      uint32_t tot_d = 0;
      if (tid < radix) {
#pragma unroll 4
        for (int w = 0; w < WARPS; ++w) {
          const uint32_t c = wcnt[w * RMAX + tid];
          wcnt[w * RMAX + tid] = (uint16_t)tot_d;
          tot_d += c;
        }
      }
      uint32_t inc = tot_d;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc += t;
      }
      if (lane == 31 && warp < RMAX / 32u) misc->warp_sums[warp] = inc;
      __syncthreads();
      if (tid < radix) {
        uint32_t wbase = 0;
        for (uint32_t w = 0; w < warp; ++w) wbase += misc->warp_sums[w];
        const uint32_t dbase = wbase + inc - tot_d;
#pragma unroll 4
        for (int w = 0; w < WARPS; ++w) wcnt[w * RMAX + tid] = (uint16_t)(wcnt[w * RMAX + tid] + dbase);
      }
      __syncthreads();
#pragma unroll
      for (int j = 0; j < IPT; ++j) {
        if (e_dig[j] < RMAX) dst[(uint32_t)wcnt[warp * RMAX + e_dig[j]] + e_rank[j]] = (uint16_t)e_src[j];
      }
      __syncthreads();
    }
    fin = (npass & 1u) ? buf1 : buf0;
    }
    }   // not compacted
    // gather the records into sorted order (region A) and emit perm. The sorted keys pass through the registers of
    // consecutive lanes here, so the time-cluster check ("are the time clusters of the tile tight?", below) rides
    // along: per block of 32 sorted positions the largest cluster-start key and the key of the last event in front
    // of the block's first start go to the (still free) list region, and are stitched together after the barrier.
    // (Reading the keys again afterwards, 8 consecutive records per thread, was a 16-way bank conflict: 7 % of the
    // kernel's shared-memory wavefronts on config 4.)
    uint32_t* cl_blk = reinterpret_cast<uint32_t*>(smem + L::kList);      // [T / 32][2]
    bool cl_loose2 = false;
    for (uint32_t k0 = warp * 32u; k0 < mm; k0 += THREADS) {               // warp-uniform trip count
      const uint32_t k = k0 + lane;
      const bool valid = k < mm;
      uint2 rec = make_uint2(0xFFFFFFFFu, 0u);
      if (valid) {
        const uint32_t s = fin[k];
        rec = recB[lo + s];
        recA[k] = rec;
        a.perm[out_base + k] = raw_val + s;
      }
      if (cl_scan) {
        const uint32_t key = rec.x;
        uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
        if (lane == 0) prev = k0 ? recB[lo + fin[k0 - 1u]].x : 0u;
        const bool st = valid && (k == 0u || key - prev > a.W);
        uint32_t ps = st ? key : 0u;                                       // prefix maximum of the start keys (0: none)
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t t = __shfl_up_sync(0xffffffffu, ps, o);
          if (lane >= (uint32_t)o) ps = max(ps, t);
        }
        // a start at key 0 looks like "none": its followers are then checked against the carry, which is 0 too
        const bool lead = valid && ps == 0u;
        if (valid && ps != 0u && key - ps > a.W) cl_loose2 = true;
        const uint32_t lead_last = __reduce_max_sync(0xffffffffu, lead ? key + 1u : 0u);   // + 1: 0 = no lead event
        if (lane == 31) { cl_blk[2u * (k0 >> 5)] = ps; cl_blk[2u * (k0 >> 5) + 1u] = lead_last; }
      }
    }
    __syncthreads();
    // the hash table now takes X + B: clear it
    uint4* z = reinterpret_cast<uint4*>(smem + L::kRegX);
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int q = 0; q < 16 * T / 16 / THREADS; ++q) z[q * THREADS + tid] = zero;
    if (cl_scan) {
      const uint32_t nb = (mm + 31u) >> 5;
      if (tid < nb && cl_blk[2u * tid + 1u]) {          // block tid begins inside a cluster that started before it
        uint32_t carry = 0;
        for (uint32_t b2 = 0; b2 < tid; ++b2) carry = max(carry, cl_blk[2u * b2]);
        if (cl_blk[2u * tid + 1u] - 1u - carry > a.W) cl_loose2 = true;
      }
      if (cl_loose2) misc->loose = 1u;
    }
    __syncthreads();
  } else {
    if (!kPerm)
      for (uint32_t k = tid; k < mm; k += THREADS) a.perm[out_base + k] = raw_val + k;
  }
  const uint2* recS = unsorted ? recA : recB + lo;
  unsigned char* hreg = smem + (unsorted ? L::kRegX : L::kRegA);   // 16T bytes: hash table, later the label / chain arrays
  uint32_t* tab = reinterpret_cast<uint32_t*>(hreg);               // [NB][4]
  uint32_t* cnt32 = reinterpret_cast<uint32_t*>(smem + L::kPar);   // bucket fill counters, u16 pairs
  uint16_t* par = reinterpret_cast<uint16_t*>(smem + L::kPar);     // parent (after the insert step)
  uint32_t* list = reinterpret_cast<uint32_t*>(smem + L::kList);   // deferred links k << 16 | j
  uint32_t* head = reinterpret_cast<uint32_t*>(hreg + 4 * T);           // [T] member chain head per label
  // mode 1 keeps the hash table alive until the end: its marks go where mode 0 keeps the parents, and the
  // ordinal list may overwrite them (the ordinal step has read every mark before it writes the first ordinal)
  uint16_t* lab = kLM ? reinterpret_cast<uint16_t*>(smem + L::kPar)
                       : reinterpret_cast<uint16_t*>(hreg + 8 * T);     // [T] label per event
  uint16_t* rootpos = kLM ? lab : reinterpret_cast<uint16_t*>(hreg + 10 * T);   // [T] ordinal -> label
  uint16_t* nxt = reinterpret_cast<uint16_t*>(hreg + 12 * T);           // [T] next member of the same hit

  // Scans one neighbour cell completely (home bucket and, while marked, the following ones) and
  // hands every event that passes the time test to `sink`. Used for the rare cases only.
  auto scan_cell = [&](uint32_t c, uint32_t slk, uint32_t key, uint32_t lim, auto&& sink) {
    uint32_t h = ((c | (slk << 16)) * kGold) >> kHashShift;
    const uint32_t want = c << 16;
    for (;;) {
      const uint4 e = *reinterpret_cast<const uint4*>(tab + 4u * h);
      const uint32_t es[4] = {e.x, e.y, e.z, e.w & ~0x8000u};
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        const uint32_t d = (es[s] ^ want) - 1u;
        if (d < lim) {
          const uint32_t kj = recS[d].x;
          if (absdiff_u32(kj, key) <= a.W) sink(d);
        }
      }
      if (!(e.w & 0x8000u)) break;
      h = (h + 1u) & (NB - 1u);
    }
  };
  // hash insert: entry = cell << 16 | k+1 into bucket hash(shot offset, cell). Slot c of a bucket is taken by
  // the c-th arrival (counter); arrivals past the 4th mark the bucket (bit 15 of slot 3) and spill to the next.
  auto hash_insert = [&]() {
    for (uint32_t k = tid; k < mm; k += THREADS) {
      const uint2 r = recS[k];
      const uint32_t cell = r.y & 0xFFFFu, slk = r.x >> tb;
      uint32_t h = ((cell | (slk << 16)) * kGold) >> kHashShift;
      const uint32_t entry = (cell << 16) | (k + 1u);
      for (;;) {
        const uint32_t sh = (h & 1u) * 16u;
        const uint32_t c = (atomicAdd(&cnt32[h >> 1], 1u << sh) >> sh) & 0xFFFFu;
        if (c < 4u) { atomicOr(&tab[4u * h + c], entry); break; }
        atomicOr(&tab[4u * h + 3u], 0x8000u);
        h = (h + 1u) & (NB - 1u);
      }
    }
  };
  // The same, fast for the common cases: a cell that is empty or holds one or two events (below lim) is settled
  // with the min/max match network; only a third event or an overflowed bucket takes the slot-by-slot scan
  // (which then skips the first two).
  auto scan_cell2 = [&](uint32_t c, uint32_t slk, uint32_t key, uint32_t lim, auto&& sink) {
    const uint32_t h = ((c | (slk << 16)) * kGold) >> kHashShift;
    const uint4 e = *reinterpret_cast<const uint4*>(tab + 4u * h);
    const uint32_t want = c << 16;
    const uint32_t d0 = (e.x ^ want) - 1u, d1 = (e.y ^ want) - 1u, d2 = (e.z ^ want) - 1u,
                   d3 = ((e.w & ~0x8000u) ^ want) - 1u;
    const uint32_t mn01 = min(d0, d1), mx01 = max(d0, d1), mn23 = min(d2, d3), mx23 = max(d2, d3);
    const uint32_t lo2 = max(mn01, mn23), hi2 = min(mx01, mx23);
    const uint32_t s1 = min(mn01, mn23), s2 = min(lo2, hi2), s3 = max(lo2, hi2);
    if (s1 < lim && absdiff_u32(recS[s1].x, key) <= a.W) sink(s1);
    if (s2 < lim && absdiff_u32(recS[s2].x, key) <= a.W) sink(s2);
    if (s3 < lim || (e.w & 0x8000u))
      scan_cell(c, slk, key, lim, [&](uint32_t j) { if (j != s1 && j != s2) sink(j); });
  };
  // mode 1 with a small box: the neighbours are found through the hash, (2 wx + 1)(2 wy + 1) cells per event;
  // a large box is cheaper to serve by walking the time window of the sorted tile
  const bool lm_grid = kLM && (2u * a.lm_wx + 1u) * (2u * a.lm_wy + 1u) <= 81u;
  // calls sink(j) for every event j of the box of event (cell, slk, key), the event itself included
  auto scan_box = [&](uint32_t cell, uint32_t slk, uint32_t key, auto&& sink) {
    const uint32_t x = cell & 0xFFu, y = cell >> 8;
    const uint32_t x0 = x > a.lm_wx ? x - a.lm_wx : 0u, x1 = min(x + a.lm_wx, a.sensor_w - 1u);
    const uint32_t y0 = y > a.lm_wy ? y - a.lm_wy : 0u, y1 = min(y + a.lm_wy, a.sensor_h - 1u);
    for (uint32_t yy = y0; yy <= y1; ++yy)
      for (uint32_t xx = x0; xx <= x1; ++xx) {
        scan_cell2((yy << 8) | xx, slk, key, (uint32_t)T, sink);
      }
  };

  if (kLM && lm_grid) {
    // ---- paper-literal mode (Eq. 5-7, :122-150) through the hash: k is a hit if no event of its box —
    //      same shot, |dX| <= wx, |dY| <= wy, |dToF| <= W, all inclusive — has a greater (ToT, sorted index)
    hash_insert();
    __syncthreads();
    for (uint32_t k = tid; k < mm; k += THREADS) {
      const uint2 r = recS[k];
      const uint32_t ti = r.y >> 16;
      bool is_max = true;
      scan_box(r.y & 0xFFFFu, r.x >> tb, r.x, [&](uint32_t j) {
        const uint32_t tj = recS[j].y >> 16;
        if (tj > ti || (tj == ti && j > k)) is_max = false;      // equal ToT: the later pixel wins (:150)
      });
      // the marks overwrite the bucket counters (dead since the insert barrier), not the table
      a.label[out_base + k] = is_max ? out_val + k : kNone;
      lab[k] = is_max ? (uint16_t)k : (uint16_t)0xFFFFu;
    }
    __syncthreads();
  } else if (kLM) {
    // ---- paper-literal mode (Eq. 5-7, :122-150): k is a hit if no event of its box — same shot,
    //      |dX| <= wx, |dY| <= wy, |dToF| <= W, all inclusive — has a greater (ToT, sorted index). The keys
    //      ascend and keys of different shots differ by more than W, so the time neighbours of k are one
    //      contiguous run of the sorted tile around k: walk it in shared memory, stop at the first brighter one
    for (uint32_t k = tid; k < mm; k += THREADS) {
      const uint2 r = recS[k];
      const uint32_t ti = r.y >> 16;
      bool is_max = true;
      for (uint32_t j = k; is_max && j-- > 0u;) {
        const uint2 q = recS[j];
        if (r.x - q.x > a.W) break;
        if ((q.y >> 16) > ti && lm_near(r.y, q.y, a.lm_wx, a.lm_wy)) is_max = false;    // earlier: strictly brighter
      }
      for (uint32_t j = k + 1u; is_max && j < mm; ++j) {
        const uint2 q = recS[j];
        if (q.x - r.x > a.W) break;
        if ((q.y >> 16) >= ti && lm_near(r.y, q.y, a.lm_wx, a.lm_wy)) is_max = false;   // later: wins ties (:150)
      }
      lab[k] = is_max ? (uint16_t)k : (uint16_t)0xFFFFu;
      a.label[out_base + k] = is_max ? out_val + k : kNone;
    }
    __syncthreads();
  } else if (kGiven) {
    // ---- mode 3 (tpx3_centroid): the caller's labels. A hit must lie inside the tile (labels of tpx3_cluster do:
    //      no hit crosses a shot); one that does not sends the call to the general kernels --------------------
    {
      uint4* f = reinterpret_cast<uint4*>(hreg);
      const uint4 ones = make_uint4(kNone, kNone, kNone, kNone);
#pragma unroll
      for (int q = 0; q < 8 * T / 16 / THREADS; ++q) f[q * THREADS + tid] = ones;   // (minidx and) head
    }
    __syncthreads();
    bool outside = false;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t k = (uint32_t)j * THREADS + tid;
      if (k < mm) {
        const uint32_t l = a.label[out_base + k] - out_val;       // a label before the tile wraps to a huge value
        if (l >= mm) { outside = true; lab[k] = (uint16_t)0xFFFFu; }
        else {
          lab[k] = (uint16_t)l;
          nxt[k] = (uint16_t)atomicExch(&head[l], k);
        }
      }
    }
    if (__syncthreads_or(outside ? 1 : 0)) failed = true;
  } else {
  // ---- are the time clusters of the tile tight? --------------------------------------------------------
  // Cut the ascending keys into clusters wherever two neighbours are more than W apart (a new shot always is).
  // If every cluster spans at most W, "within W" is an equivalence relation on the tile: two events that are
  // both within W of a third are within W of each other. The link step below then needs one probe for most
  // events. One pass over the sorted keys; the start of the cluster that runs into a warp's range is the largest
  // cluster-start key of the warps before it (the keys ascend, so a prefix maximum).
  // (Nothing to check when all times of flight of the tile lie within W: electron VMI. Tiles that arrived in
  // order did this on the keys in registers while building their records; see there.)
  // ---- hash insert ----------------------------------------------------------------------------------
  hash_insert();
  __syncthreads();

  // ---- S2: probe the forward cells, prune implied links, first link = parent, others deferred ---
  uint32_t list_cap = (uint32_t)L::kListCap;   // tight tiles lend the top of the list region to the second pass
  auto push_link = [&](uint32_t k, uint32_t j) {
    const uint32_t pos = atomicAdd(&misc->n_list, 1u);
    if (pos < list_cap) list[pos] = (k << 16) | j;
  };
  // tt: the tile is tight (see below). Then a candidate that passes the time test stands for every event of
  // its cell and time cluster (they are connected among themselves: through their common S event, or by the
  // later one's own-cell probe), and the cell needs no scan task.
  auto link_event = [&](const uint32_t k, const bool tt) {
    {
      const uint2 r = recS[k];
      const uint32_t key = r.x, cell = r.y & 0xFFFFu, slk = key >> tb, hs = slk << 16;
      const uint32_t x = cell & 0xFFu, y = cell >> 8;
      const bool xe = x + 1u < a.sensor_w, xw = x > 0u, ys = y + 1u < a.sensor_h;
      uint32_t slow = 0;
      // one forward cell: candidate index (or k), its key, and whether it passed the time test
      auto probe = [&](uint32_t off, bool valid, uint32_t lim, uint32_t bit, uint32_t& jc, uint32_t& kc) -> bool {
        const uint32_t c = cell + off;
        const uint32_t h = ((c | hs) * kGold) >> kHashShift;
        const uint4 e = *reinterpret_cast<const uint4*>(tab + 4u * h);
        const uint32_t want = c << 16;
        const uint32_t d0 = (e.x ^ want) - 1u, d1 = (e.y ^ want) - 1u, d2 = (e.z ^ want) - 1u,
                       d3 = ((e.w & ~0x8000u) ^ want) - 1u;
        // a slot of this cell gives d < lim, any other slot (other cell, empty) a d >= 65535: the smallest d
        // is the candidate, and a second-smallest d below lim means the cell holds several events
        const uint32_t mn01 = min(d0, d1), mx01 = max(d0, d1), mn23 = min(d2, d3), mx23 = max(d2, d3);
        const uint32_t s1 = min(mn01, mn23), s2 = min(max(mn01, mn23), min(mx01, mx23));
        const bool any = valid && s1 < lim;
        jc = any ? s1 : k;
        kc = recS[jc].x;
        const bool pass = any && absdiff_u32(kc, key) <= a.W;
        if (valid && (s2 < lim || (e.w & 0x8000u)) && !(tt && pass)) slow |= bit;
        return pass;
      };
      uint32_t jS, kS, jE, kE, jSE, kSE, jSW, kSW, jO, kO;
      const bool pS = probe(256u, ys, (uint32_t)T, 1u, jS, kS);
      const bool pE = probe(1u, xe, (uint32_t)T, 2u, jE, kE);
      const bool pSE = probe(257u, xe && ys, (uint32_t)T, 4u, jSE, kSE);
      const bool pSW = probe(255u, xw && ys, (uint32_t)T, 8u, jSW, kSW);
      const bool pO = probe(0u, true, k, 16u, jO, kO);   // own cell: only earlier events (d < k)
      // A candidate c is dropped when another candidate a of this event is adjacent to c in space
      // (fixed by the cell geometry) and in time: the pair (a, c) is linked by a or c itself.
      const uint32_t W = a.W;
      const bool keepS = pS;
      const bool keepE = pE && !(pS && absdiff_u32(kE, kS) <= W);
      const bool keepSE = pSE && !(pS && absdiff_u32(kSE, kS) <= W) && !(pE && absdiff_u32(kSE, kE) <= W);
      const bool keepSW = pSW && !(pS && absdiff_u32(kSW, kS) <= W);
      const bool keepO = pO && !(pS && absdiff_u32(kO, kS) <= W) && !(pE && absdiff_u32(kO, kE) <= W) &&
                         !(pSE && absdiff_u32(kO, kSE) <= W) && !(pSW && absdiff_u32(kO, kSW) <= W);
      uint32_t parent = k;
      bool have = false;
      auto take = [&](bool keep, uint32_t j) {
        if (keep) {
          if (!have) { parent = j; have = true; }
          else push_link(k, j);
        }
      };
      take(keepS, jS);
      take(keepE, jE);
      take(keepSE, jSE);
      take(keepSW, jSW);
      take(keepO, jO);
      par[k] = (uint16_t)parent;
      // rare: a neighbour cell holds several events, or its bucket overflowed: all of them must be
      // linked. Queued as a task (k, direction) so that the scans run densely packed afterwards.
      while (slow) {
        const uint32_t q = (uint32_t)__ffs(slow) - 1u;
        slow &= slow - 1u;
        push_link(k, kTaskBase + q);
      }
    }
  };
  // Tight tiles (all time clusters at most W wide: electron VMI, ion VMI with separated mass peaks): two events
  // that pass the time test against a third pass it against each other, so the pruning rule drops every other
  // candidate of an event whose S cell holds an event of its own time cluster. Such an event needs ONE probe.
  // First pass: S only; the events whose S cell is empty, holds another cluster's event first, or overflowed are
  // collected and take the full five-cell step densely packed in a second pass.
  const bool tight = kCC && misc->loose == 0u;
  if (tight && tid == 0) atomicAdd(&a.ctrl->tight_tiles, 1u);
  if (tight) {
    uint16_t* kl_end = reinterpret_cast<uint16_t*>(smem + L::kMisc);   // grows downwards from the list's end
    constexpr uint32_t kKlMax = (uint32_t)(4 * L::kListCap - 1024) / 2u;   // leaves 256 deferred-list entries
    const uint32_t lt_mask = lanemask_lt();
    for (uint32_t k0 = warp * 32u; k0 < mm; k0 += THREADS) {          // warp-uniform trip count (ballot inside)
      const uint32_t k = k0 + lane;
      bool second = false;
      if (k < mm) {
        const uint2 r = recS[k];
        const uint32_t key = r.x, cell = r.y & 0xFFFFu;
        second = true;
        if ((cell >> 8) + 1u < a.sensor_h) {
          const uint32_t c = cell + 256u;
          const uint32_t h = ((c | ((key >> tb) << 16)) * kGold) >> kHashShift;
          const uint4 e = *reinterpret_cast<const uint4*>(tab + 4u * h);
          const uint32_t want = c << 16;
          const uint32_t d0 = (e.x ^ want) - 1u, d1 = (e.y ^ want) - 1u, d2 = (e.z ^ want) - 1u,
                         d3 = ((e.w & ~0x8000u) ^ want) - 1u;
          const uint32_t s1 = min(min(d0, d1), min(d2, d3));
          if (s1 < (uint32_t)T && !(e.w & 0x8000u) && absdiff_u32(recS[s1].x, key) <= a.W) {
            par[k] = (uint16_t)s1;
            second = false;
          }
        }
      }
      const uint32_t bal = __ballot_sync(0xffffffffu, second);
      if (bal) {
        uint32_t basepos = 0;
        if (lane == 0) basepos = atomicAdd(&misc->n_klist, (uint32_t)__popc(bal));
        basepos = __shfl_sync(0xffffffffu, basepos, 0);
        const uint32_t idx = basepos + (uint32_t)__popc(bal & lt_mask);
        if (second && idx < kKlMax) kl_end[-1 - (int)idx] = (uint16_t)k;
      }
    }
    __syncthreads();
    const uint32_t n2 = misc->n_klist;
    if (n2 <= kKlMax) {
      list_cap = ((uint32_t)(4 * L::kListCap) - 2u * n2) / 4u;   // what the collected events leave of the region
      for (uint32_t i = tid; i < n2; i += THREADS) link_event(kl_end[-1 - (int)i], true);
    } else {                                                       // mostly isolated pixels: the plain single pass
      for (uint32_t k = tid; k < mm; k += THREADS) link_event(k, false);
    }
  } else {
    for (uint32_t k = tid; k < mm; k += THREADS) link_event(k, false);
  }
  __syncthreads();
  // ---- deferred links: union by compare-and-swap hooks ---------------------------------------------
  {
    const uint32_t nl = misc->n_list;
    // the plain parent stores left chains as long as a blob is tall: halve them first, so that the finds of
    // the unions (few threads, everybody else waits for them) are short. A halving store never touches a
    // root and any ancestor is a valid parent, so it may race with the hooks.
    for (int hr = 0; hr < kHalvePre; ++hr)
      for (uint32_t k = tid; k < mm; k += THREADS) {
        const uint32_t p1 = par[k], g = par[p1];
        if (g != p1) par[k] = (uint16_t)g;
      }
    if (nl > list_cap) {
      // the list overflowed (very dense tile): redo the probes, uniting on the spot
      for (uint32_t k = tid; k < mm; k += THREADS) {
        const uint2 r = recS[k];
        const uint32_t key = r.x, cell = r.y & 0xFFFFu, slk = key >> tb;
        const uint32_t x = cell & 0xFFu, y = cell >> 8;
        const bool xe = x + 1u < a.sensor_w, xw = x > 0u, ys = y + 1u < a.sensor_h;
        auto un = [&](uint32_t j) { uf_unite(par, k, j); };
        if (ys) scan_cell(cell + 256u, slk, key, (uint32_t)T, un);
        if (xe) scan_cell(cell + 1u, slk, key, (uint32_t)T, un);
        if (xe && ys) scan_cell(cell + 257u, slk, key, (uint32_t)T, un);
        if (xw && ys) scan_cell(cell + 255u, slk, key, (uint32_t)T, un);
        scan_cell(cell, slk, key, k, un);
      }
      __syncthreads();
    } else {
      for (uint32_t i = tid; i < nl; i += THREADS) {
        const uint32_t e = list[i];
        const uint32_t k = e >> 16, j = e & 0xFFFFu;
        if (j < kTaskBase) {
          uf_unite(par, k, j);
        } else {                                   // task: scan one forward cell of k completely
          const uint32_t q = j - kTaskBase;
          const uint2 r = recS[k];
          const uint32_t off = q == 0u ? 256u : (q == 1u ? 1u : (q == 2u ? 257u : (q == 3u ? 255u : 0u)));
          scan_cell2((r.y & 0xFFFFu) + off, r.x >> tb, r.x, q == 4u ? k : (uint32_t)T,
                     [&](uint32_t jj) { uf_unite(par, k, jj); });
        }
      }
    }
  }
  __syncthreads();   // the hash table is dead from here on

  // ---- S3: label = smallest sorted index of the component ------------------------------------------
  uint32_t* minidx = reinterpret_cast<uint32_t*>(hreg);                 // [T] by root
  {
    uint4* f = reinterpret_cast<uint4*>(hreg);
    const uint4 ones = make_uint4(kNone, kNone, kNone, kNone);
#pragma unroll
    for (int q = 0; q < 8 * T / 16 / THREADS; ++q) f[q * THREADS + tid] = ones;   // minidx and head
  }
  // kHalvePost more rounds of pointer halving (any ancestor is a valid parent, so the plain stores may race;
  // measured: 2 rounds before the unions and none here is best),
  // then the roots
#pragma unroll
  for (int round = 0; round < kHalvePost; ++round) {
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t k = (uint32_t)j * THREADS + tid;
      if (k < mm) {
        const uint32_t p1 = par[k], g = par[p1];
        if (g != p1) par[k] = (uint16_t)g;
      }
    }
  }
  uint32_t root_r[IPT];
#pragma unroll
  for (int j = 0; j < IPT; ++j) {
    const uint32_t k = (uint32_t)j * THREADS + tid;
    root_r[j] = k < mm ? uf_find(par, k) : 0u;
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < IPT; ++j) {
    const uint32_t k = (uint32_t)j * THREADS + tid;
    if (k < mm) atomicMin(&minidx[root_r[j]], k);
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < IPT; ++j) {
    const uint32_t k = (uint32_t)j * THREADS + tid;
    if (k < mm) {
      const uint32_t l = minidx[root_r[j]];
      lab[k] = (uint16_t)l;
      a.label[out_base + k] = out_val + l;
      if (!kLabelsOnly && !(MODE == 5 && a.labels_only)) nxt[k] = (uint16_t)atomicExch(&head[l], k);   // every member, the first pixel too; kNone truncates to 0xFFFF = end
    }
  }
  __syncthreads();
  }   // mode 0
  uint32_t n_roots;
  {
    // blocked arrangement: thread owns sorted positions [8 tid, 8 tid + 8)
    const uint4 q0 = *reinterpret_cast<const uint4*>(lab + p0);
    const uint32_t lw[4] = {q0.x, q0.y, q0.z, q0.w};
    uint32_t flags = 0, cntr = 0;
#pragma unroll
    for (int j = 0; j < IPT; ++j) {
      const uint32_t l = (lw[j >> 1] >> ((j & 1) * 16)) & 0xFFFFu;
      if (p0 + j < mm && l == p0 + j) { flags |= 1u << j; ++cntr; }
    }
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
    n_roots = (kGiven && failed) ? 0u : misc->n_roots;
  }
  __syncthreads();   // rootpos complete

  // ---- S4: one thread per hit walks its chain: exact sums, brightest pixel. The hit goes to the
  //      staging table at the tile's own position out_base + c (a tile has no more hits than events);
  //      k_fused_compact moves it to its ordinal once every tile's count is known -------------------
  if (kLM && lm_grid) {
    // paper-literal mode: the row sums of Eq. 9 over the box about every local maximum
    for (uint32_t c = tid; c < n_roots; c += THREADS) {
      const uint32_t r = rootpos[c];
      const uint2 rr = recS[r];
      unsigned long long sx = 0, sy = 0, sf = 0;
      uint32_t st = 0, size = 0;
      scan_box(rr.y & 0xFFFFu, rr.x >> tb, rr.x, [&](uint32_t j) {   // j == r included: A_ii = 1 (Eq. 4 diagonal)
        const uint2 q = recS[j];
        const uint32_t t = q.y >> 16;
        ++size;
        st += t;
        sx += (unsigned long long)(t * (q.y & 0xFFu));
        sy += (unsigned long long)(t * ((q.y >> 8) & 0xFFu));
        sf += (unsigned long long)t * (unsigned long long)(q.x & tmask);
      });
      const uint64_t o = (uint64_t)out_base + c;
      a.stage_a[o] = make_uint4(out_val + r, size, st, 0u);
      a.stage_b[o] = make_uint4((uint32_t)sx, (uint32_t)(sx >> 32), (uint32_t)sy, (uint32_t)(sy >> 32));
      a.stage_c[o] = ref + (uint64_t)(rr.x >> tb) * a.P + (uint64_t)(rr.x & tmask);
      a.stage_d[o] = sf;
    }
  } else if (kLM) {
    // the same by walking the time window of the sorted tile (large boxes)
    for (uint32_t c = tid; c < n_roots; c += THREADS) {
      const uint32_t r = rootpos[c];
      const uint2 rr = recS[r];
      unsigned long long sx = 0, sy = 0, sf = 0;
      uint32_t st = 0, size = 0;
      auto add = [&](const uint2 q) {
        if (lm_near(rr.y, q.y, a.lm_wx, a.lm_wy)) {
          const uint32_t t = q.y >> 16;
          ++size;
          st += t;
          sx += (unsigned long long)(t * (q.y & 0xFFu));
          sy += (unsigned long long)(t * ((q.y >> 8) & 0xFFu));
          sf += (unsigned long long)t * (unsigned long long)(q.x & tmask);
        }
      };
      add(rr);                                    // A_ii = 1 (Eq. 4 diagonal)
      for (uint32_t j = r; j-- > 0u;) {
        const uint2 q = recS[j];
        if (rr.x - q.x > a.W) break;
        add(q);
      }
      for (uint32_t j = r + 1u; j < mm; ++j) {
        const uint2 q = recS[j];
        if (q.x - rr.x > a.W) break;
        add(q);
      }
      const uint64_t o = (uint64_t)out_base + c;
      a.stage_a[o] = make_uint4(out_val + r, size, st, 0u);
      a.stage_b[o] = make_uint4((uint32_t)sx, (uint32_t)(sx >> 32), (uint32_t)sy, (uint32_t)(sy >> 32));
      a.stage_c[o] = ref + (uint64_t)(rr.x >> tb) * a.P + (uint64_t)(rr.x & tmask);
      a.stage_d[o] = sf;
    }
  } else if (!kLabelsOnly && !(MODE == 5 && a.labels_only))
  for (uint32_t c = tid; c < n_roots; c += THREADS) {
    const uint32_t r = rootpos[c];
    unsigned long long sx = 0, sy = 0, sf = 0;
    uint32_t st = 0, size = 0, best = 0, k = head[r];   // the chain holds every member of the hit
    do {
      const uint2 rk = recS[k];
      const uint32_t w1 = rk.y;
      const uint32_t t = w1 >> 16;
      sf += (unsigned long long)t * (unsigned long long)(rk.x & tmask);   // ToF = ToA - shot * P
      st += t;                                             // <= 65535 * 8192 < 2^32
      sx += (unsigned long long)(t * (w1 & 0xFFu));
      sy += (unsigned long long)(t * ((w1 >> 8) & 0xFFu));
      ++size;
      best = max(best, (t << 16) | k);   // (ToT, sorted index): the later pixel wins ties
      k = nxt[k];
    } while (k != 0xFFFFu);
    const uint32_t keyp = recS[best & 0xFFFFu].x;
    const uint64_t o = (uint64_t)out_base + c;
    a.stage_a[o] = make_uint4(out_val + r, size, st, 0u);
    a.stage_b[o] = make_uint4((uint32_t)sx, (uint32_t)(sx >> 32), (uint32_t)sy, (uint32_t)(sy >> 32));
    a.stage_c[o] = ref + (uint64_t)(keyp >> tb) * a.P + (uint64_t)(keyp & tmask);
    a.stage_d[o] = sf;
  }

  // ---- the tile's status word (tiles that own something only); on to the segment's next tile -------------
  if (mm) {
    if (tid == 0) a.tiles[(uint64_t)seg * seg_maxt + tile_i] = ((unsigned long long)out_base << 32) | (unsigned long long)n_roots;
    ++tile_i;
    seg_hits_run += n_roots;
  }
  if (failed) { seg_failed = true; break; }
  at_start = misc->lo != kNone;     // everything but "no shot start in sight" ends at a shot start
  if constexpr (kPre) {
    pre_have_s = next_at < base + cnt && next_at - base >= skp;
    pre_next_s = s_ref + misc->s_next;
  }
  tile_at = next_at;
  if (tile_at >= seg_end) break;
  }   // tiles of the segment

  // ---- completion: the last segment to finish publishes the outcome of the call -------------------
  if (tid == 0) {
    for (uint32_t i = tile_i; i < seg_maxt; ++i) a.tiles[(uint64_t)seg * seg_maxt + i] = 0ull;
    // the segment's hit total, behind the status words: k_fused_compact sums these, not every tile word, for its prefix
    reinterpret_cast<uint32_t*>(a.tiles + a.num_tiles)[seg] = seg_hits_run;
    if (seg_failed) atomicExch(&a.ctrl->fused_fail, 1u);
    if (tile_i) atomicAdd(&a.ctrl->tiles_run, tile_i);
    __threadfence();
    const uint32_t done = atomicAdd(&a.ctrl->tiles_done, 1u);
    if (done + 1u == seg_n) {
      __threadfence();
      const uint32_t any_fail = atomicAdd(&a.ctrl->fused_fail, 0u);
      // 2: the general kernels behind this one redo the call; 1: k_fused_compact finishes it
      a.ctrl->fused_state = any_fail ? 2u : 1u;
    }
  }
}

// ---- S5 + ordering: staging table -> cluster table -----------------------------------------------
// Runs behind k_fused_shot_tiles (same stream), so every tile's hit count is final: no tile waits
// for another one. CTA i takes a contiguous range of tiles, sums the hits in front of its range
// (per-segment totals, L2-resident) and copies its tiles' hits to
// their ordinals, ascending label order. Also computes what needs no tile state: shot = ToA of
// the brightest pixel div P (the pixel belongs to the hit's shot, R6) and the centroid
// fp32(sum tot*x) / fp32(sum tot), IEEE RN (Eq. 9).
constexpr int kCompactThreads = 256;

__global__ void __launch_bounds__(kCompactThreads) k_fused_compact(FusedArgs a, uint32_t tiles_per_cta, uint32_t T) {
  if (a.ctrl->fused_state != 1u) return;   // the fused kernel gave up: the general path redoes the call
  const uint32_t* seg_hits = reinterpret_cast<const uint32_t*>(a.tiles + a.num_tiles);   // per-segment hit totals
  uint32_t maxt = a.maxt;
  if (a.n_dev) {                           // a stream push: the true geometry from the device's count
    const FusedSegs sg = fused_segs((uint64_t)*a.n_dev, T, a.num_sms);
    a.num_tiles = sg.nseg * sg.maxt;
    maxt = sg.maxt;
    uint32_t ctas;
    compact_grid(a.num_tiles, a.num_sms, &ctas, &tiles_per_cta);
    if (blockIdx.x >= ctas) return;
  }
  __shared__ unsigned long long s_part[kCompactThreads / 32];
  __shared__ unsigned long long s_prefix;
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t t0 = blockIdx.x * tiles_per_cta;
  const uint32_t t1 = min(t0 + tiles_per_cta, a.num_tiles);
  if (t0 >= a.num_tiles) return;
  unsigned long long sum = 0;
  // hits in front of the CTA's range: whole segments by their totals, the rest tile by tile (summing all tile words
  // here was 1.7 GB of L2 reads over the grid on the 2^28-hit chunk: as much as the rows the kernel moves)
  const uint32_t seg0 = t0 / maxt;
  for (uint32_t g = tid; g < seg0; g += kCompactThreads) sum += seg_hits[g];
  for (uint32_t t = seg0 * maxt + tid; t < t0; t += kCompactThreads) sum += a.tiles[t] & 0xFFFFFFFFull;
#pragma unroll
  for (int o = 16; o; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if (lane == 0) s_part[warp] = sum;
  __syncthreads();
  if (tid == 0) {
    unsigned long long p = 0;
    for (int w = 0; w < kCompactThreads / 32; ++w) p += s_part[w];
    s_prefix = p;
  }
  __syncthreads();
  unsigned long long prefix = s_prefix;
  const uint32_t label_base = a.label_base ? (uint32_t)*a.label_base : 0u;
  bool over = false;
  // the CTA's tiles in groups of 32: warp 0 turns the group's hit counts into offsets, then all threads walk the
  // group's hits as ONE index range (a tile has about 300 hits: a loop per tile would leave most of the last
  // iteration's lanes idle)
  __shared__ uint32_t s_off[33];
  __shared__ uint32_t s_src[32];
  for (uint32_t g0 = t0; g0 < t1; g0 += 32u) {
    const uint32_t ng = min(32u, t1 - g0);
    __syncthreads();                      // the previous group's tables are no longer read
    if (warp == 0) {
      const unsigned long long w = lane < ng ? a.tiles[g0 + lane] : 0ull;
      const uint32_t cnt = (uint32_t)(w & 0xFFFFFFFFull);
      uint32_t inc = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (uint32_t)o) inc += v;
      }
      s_off[lane] = inc - cnt;
      s_src[lane] = (uint32_t)(w >> 32);
      if (lane == 31) s_off[32] = inc;
    }
    __syncthreads();
    const uint32_t total = s_off[32];
    for (uint32_t i = tid; a.mode != 2u && !a.labels_only && i < total; i += kCompactThreads) {
      // tile of hit i: the last offset <= i (binary search over 32 offsets)
      uint32_t q = 0;
#pragma unroll
      for (uint32_t step = 16; step; step >>= 1)
        if (q + step < ng && s_off[q + step] <= i) q += step;
      const uint64_t src = (uint64_t)s_src[q] + (i - s_off[q]);
      const uint64_t o = prefix + i;
      if (o >= a.max_clusters) { over = true; continue; }
      const uint4 va = a.stage_a[src], vb = a.stage_b[src];
      const uint64_t toa_peak = a.stage_c[src];
      const long long st = (long long)va.z;
      const long long sx = (long long)(((unsigned long long)vb.y << 32) | vb.x);
      const long long sy = (long long)(((unsigned long long)vb.w << 32) | vb.z);
      a.out.label[o] = va.x + label_base;
      a.out.size[o] = va.y;
      a.out.shot[o] = (uint32_t)div64(toa_peak, a.divP);
      a.out.sum_tot[o] = st;
      a.out.sum_tot_x[o] = sx;
      a.out.sum_tot_y[o] = sy;
      a.out.toa_peak[o] = toa_peak;
      const float fst = __ll2float_rn(st);
      a.out.cx[o] = __fdiv_rn(__ll2float_rn(sx), fst);
      a.out.cy[o] = __fdiv_rn(__ll2float_rn(sy), fst);
      const long long sf = (long long)a.stage_d[src];
      a.out.sum_tot_tof[o] = sf;
      a.out.ctof[o] = __fdiv_rn(__ll2float_rn(sf), fst);
    }
    prefix += total;
  }
  if (over) set_error(a.ctrl, TPX3_ERR_CAPACITY);
  if (t1 == a.num_tiles && tid == 0) {
    *a.n_clusters = (uint32_t)prefix;
    a.ctrl->status.n_clusters = (uint32_t)prefix;
    if (a.mode == 6u) a.ctrl->status.path = 3;
    if (a.mode != 5u && a.mode != 6u) {     // modes 5 and 6 run behind the general path's global sort: its pass count stands (mode 5: path 2 too)
      a.ctrl->status.path = a.mode == 1u ? 3 : 1;
      a.ctrl->status.sort_passes = 0;
    }
    if (a.mode == 0u || a.mode == 2u || a.mode == 5u) {   // worth checking the time clusters next time? (fewer than 1 tile in 8 was tight: no)
      a.ctrl->scan_hint = a.ctrl->tight_tiles * 8u < a.ctrl->tiles_run ? kScanSkip : 0u;
      a.ctrl->calls += 1u;
    }
  }
}

// Which variant serves a plan. T = tile capacity = window length (events); a shot of up to T - 8 events fits.
struct FusedGeom {
  int variant;      // 0 = fused path not available for this plan, 1 = T 4096 / 512 thr, 2 = T 8192 / 1024 thr,
                    // 3 = T 2048 / 256 thr (4 CTAs per SM: +2.5 % over variant 1 on cfg 1 at the same hint)
  uint32_t T;
};

inline FusedGeom fused_geom(uint64_t P, uint32_t W, uint32_t max_shot_hits) {
  FusedGeom g{0, 0};
  if (P == 0 || P > (1ull << 24) || W >= (1u << 24)) return g;   // tof + W must fit the 32-bit tile key
  const uint32_t Lh = max_shot_hits ? max_shot_hits : 1024u;      // no hint: first rung of the ladder (below)
  // a window must hold the longest shot (T - 8 events when the tile starts at an odd position); the smaller
  // window wins whenever it does (4 CTAs of 2048 events per SM against 2 of 4096: cfg2 +6.7 %, cfg4 +5 %,
  // cfg1 equal; 8192 against 4096 on cfg3: equal)
  if (Lh <= 1536u) { g.variant = 3; g.T = 2048; }
  else if (Lh <= 3584u) { g.variant = 1; g.T = 4096; }
  else if (Lh <= 8184u) { g.variant = 2; g.T = 8192; }
  else return g;
  return g;
}

template <int T, int THREADS, int MODE>
inline int launch_fused(const FusedArgs& a, cudaStream_t st) {
  k_fused_shot_tiles<T, THREADS, MODE><<<a.nseg, THREADS, FusedSmem<T>::kBytes, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? TPX3_OK : TPX3_ERR_CUDA;
}

// The opt-in to more than 48 KB of dynamic shared memory is per function AND per device: tpx3_plan calls this
// after cudaSetDevice for its device (the 8192-event variants may also be launched from the device later on).
inline int fused_configure_device() {
#define TPX3_FUSED_ATTR(T, THREADS, MODE)                                                                          \
  if (cudaFuncSetAttribute(k_fused_shot_tiles<T, THREADS, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                           FusedSmem<T>::kBytes) != cudaSuccess)                                                  \
    return TPX3_ERR_CUDA;
  TPX3_FUSED_ATTR(2048, 256, 0) TPX3_FUSED_ATTR(2048, 256, 1) TPX3_FUSED_ATTR(2048, 256, 2) TPX3_FUSED_ATTR(2048, 256, 3)
  TPX3_FUSED_ATTR(4096, 512, 0) TPX3_FUSED_ATTR(4096, 512, 1) TPX3_FUSED_ATTR(4096, 512, 2) TPX3_FUSED_ATTR(4096, 512, 3)
  TPX3_FUSED_ATTR(8192, 1024, 0) TPX3_FUSED_ATTR(8192, 1024, 1) TPX3_FUSED_ATTR(8192, 1024, 2)
  TPX3_FUSED_ATTR(8192, 1024, 3) TPX3_FUSED_ATTR(8192, 1024, 5) TPX3_FUSED_ATTR(8192, 1024, 6)
  TPX3_FUSED_ATTR(2048, 256, 4) TPX3_FUSED_ATTR(4096, 512, 4) TPX3_FUSED_ATTR(8192, 1024, 4)
#undef TPX3_FUSED_ATTR
  return TPX3_OK;
}

// Without a hint the window length is tried in rungs: 2048 events, then 4096, then 8192. A rung whose tiles meet
// a shot that does not fit fails within its first wave (every later segment returns at once), and
// k_fallback_dispatch launches the next rung from the device; after the last one the general kernels run.
constexpr int kLadderMax = 2;   // rungs after the first
struct FusedLadder {
  int n;                        // rungs still to try after the one the host enqueued
  uint32_t T[kLadderMax];       // their window lengths
};

inline FusedLadder fused_ladder(uint32_t max_shot_hits) {
  FusedLadder l{0, {0, 0}};
  if (max_shot_hits == 0) { l.n = 2; l.T[0] = 4096u; l.T[1] = 8192u; }
  return l;
}

inline FusedArgs make_fused_args(uint32_t T, uint32_t num_sms, Ctrl* ctrl, unsigned long long* tiles, const Params& prm,
                                 const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                                 uint32_t* perm, uint32_t* label, uint64_t max_clusters, const tpx3_clusters_t& out,
                                 uint32_t* n_clusters, void* stage, uint32_t mode, uint32_t lm_wx, uint32_t lm_wy,
                                 const uint32_t* n_dev = nullptr) {
  FusedArgs a;
  a.ctrl = ctrl;
  a.tiles = tiles;
  a.n = prm.n;
  a.P = prm.P;
  a.divP = make_div64(prm.P);
  a.divP32 = make_div32((uint32_t)prm.P);
  a.W = prm.W;
  const FusedSegs sg = fused_segs(prm.n, T, num_sms);
  a.G = sg.G;
  a.nseg = sg.nseg;
  a.maxt = sg.maxt;
  a.num_tiles = sg.nseg * sg.maxt;
  a.num_sms = num_sms;
  a.sensor_w = prm.sensor_w;
  a.sensor_h = prm.sensor_h;
  a.flags = prm.flags;
  a.x = x; a.y = y; a.toa = toa; a.tot = tot;
  a.perm = perm; a.label = label;
  a.max_clusters = max_clusters;
  a.out = out;
  a.n_clusters = n_clusters;
  // staging table: 48 bytes per event position (aliases the general path's sort buffers)
  a.stage_a = reinterpret_cast<uint4*>(stage);
  a.stage_b = a.stage_a + prm.n;
  a.stage_c = reinterpret_cast<uint64_t*>(a.stage_b + prm.n);
  a.stage_d = a.stage_c + prm.n;
  a.mode = mode; a.lm_wx = lm_wx; a.lm_wy = lm_wy;
  a.label_base = nullptr;
  a.head = 0;
  memset(&a.pre, 0, sizeof(a.pre));
  a.seg_kept = nullptr;
  a.labels_only = 0;
  a.n_dev = n_dev;      // then prm.n is the largest count: it sizes the grids and lays out the staging table
  return a;
}

// The fields that depend on the event count (a stream push learns it on the device).
__host__ __device__ inline void fused_set_n(FusedArgs& a, uint64_t n, uint32_t T) {
  a.n = n;
  const FusedSegs sg = fused_segs(n, T, a.num_sms);
  a.G = sg.G; a.nseg = sg.nseg; a.maxt = sg.maxt; a.num_tiles = sg.nseg * sg.maxt;
  a.stage_b = a.stage_a + n;
  a.stage_c = reinterpret_cast<uint64_t*>(a.stage_b + n);
  a.stage_d = a.stage_c + n;
}

// Device side: the next rung, tail-launched by k_fallback_dispatch.
__device__ inline void launch_fused_rung_device(FusedArgs a, uint32_t T) {
  uint32_t ctas, tpc;
  compact_grid(a.num_tiles, a.num_sms, &ctas, &tpc);
#define TPX3_RUNG(T_, THREADS_, MODE_) \
  k_fused_shot_tiles<T_, THREADS_, MODE_><<<a.nseg, THREADS_, FusedSmem<T_>::kBytes, cudaStreamTailLaunch>>>(a)
  if (T == 2048u) {
    if (a.mode == 0u) TPX3_RUNG(2048, 256, 0);
    else if (a.mode == 1u) TPX3_RUNG(2048, 256, 1);
    else if (a.mode == 2u) TPX3_RUNG(2048, 256, 2);
    else TPX3_RUNG(2048, 256, 3);
  } else if (T == 4096u) {
    if (a.mode == 0u) TPX3_RUNG(4096, 512, 0);
    else if (a.mode == 1u) TPX3_RUNG(4096, 512, 1);
    else if (a.mode == 2u) TPX3_RUNG(4096, 512, 2);
    else TPX3_RUNG(4096, 512, 3);
  } else {
    if (a.mode == 0u) TPX3_RUNG(8192, 1024, 0);
    else if (a.mode == 1u) TPX3_RUNG(8192, 1024, 1);
    else if (a.mode == 2u) TPX3_RUNG(8192, 1024, 2);
    else if (a.mode == 3u) TPX3_RUNG(8192, 1024, 3);
    else if (a.mode == 6u) TPX3_RUNG(8192, 1024, 6);
    else TPX3_RUNG(8192, 1024, 5);
  }
#undef TPX3_RUNG
  k_fused_compact<<<ctas, kCompactThreads, 0, cudaStreamTailLaunch>>>(a, tpc, T);
}

// How far the position-indexed arrays of a call sit behind a 16-byte boundary, in elements (FusedArgs::head); -1: they
// are not aligned alike (or not to their element size): no tile kernel. Modes 0, 1, 2, 4 read x, y, tot (2 bytes) and toa
// (8 bytes) by position with 128-bit loads; modes 3 and 5 read perm (4 bytes) that way and gather the events.
__host__ __device__ inline int fused_head_of(uint32_t mode, const void* x, const void* y, const void* toa, const void* tot,
                                             const void* perm) {
  if (mode == 3u || mode == 5u || mode == 6u) return ((uintptr_t)perm & 3u) ? -1 : (int)(((uintptr_t)perm >> 2) & 3u);
  if ((((uintptr_t)x | (uintptr_t)y | (uintptr_t)tot) & 1u) || ((uintptr_t)toa & 7u)) return -1;
  const uint32_t e = (uint32_t)(((uintptr_t)x >> 1) & 7u);
  if ((((uintptr_t)y >> 1) & 7u) != e || (((uintptr_t)tot >> 1) & 7u) != e || (((uintptr_t)toa >> 3) & 1u) != (e & 1u)) return -1;
  return (int)e;
}

// Moves the position-indexed arrays down to the boundary and lets the positions start at `e` (head 0 before the call).
__host__ __device__ inline void fused_apply_head(FusedArgs& a, uint32_t e, uint32_t T) {
  if (a.mode != 3u && a.mode != 5u && a.mode != 6u) { a.x -= e; a.y -= e; a.toa -= e; a.tot -= e; }
  a.perm -= e;
  a.label -= e;
  a.head = e;
  fused_set_n(a, a.n + e, T);
}

// The general route's tile kernel (mode 5) from the arguments of a first attempt in mode 0 / 2 on the same call: back
// to the caller's pointers, then the head that perm's alignment asks for; 8192-event windows.
__host__ __device__ inline void fused_rebase_mode5(FusedArgs& a, uint32_t labels_only, uint32_t new_mode = 5u) {
  const uint32_t e0 = a.head;
  if (a.mode != 3u && a.mode != 5u && a.mode != 6u) { a.x += e0; a.y += e0; a.toa += e0; a.tot += e0; }
  a.perm += e0;
  a.label += e0;
  a.n -= e0;
  a.head = 0;
  a.mode = new_mode;     // 5: connected components, 6: the paper-literal mode
  a.labels_only = labels_only;
  fused_apply_head(a, (uint32_t)(((uintptr_t)a.perm >> 2) & 3u), 8192u);
}

// Host side. Returns TPX3_OK (launched or not applicable; *launched says which) or an error. *args receives the
// arguments of the enqueued rung (the later rungs differ in the segment geometry only).
inline int enqueue_fused(const FusedGeom& g, uint32_t num_sms, uint64_t* launches, Ctrl* ctrl, unsigned long long* tiles,
                         cudaStream_t st, const Params& prm, const uint16_t* x, const uint16_t* y,
                         const uint64_t* toa, const uint16_t* tot, uint32_t* perm, uint32_t* label,
                         uint64_t max_clusters, const tpx3_clusters_t& out, uint32_t* n_clusters, void* stage,
                         bool* launched, FusedArgs* args, uint32_t mode = 0, uint32_t lm_wx = 0, uint32_t lm_wy = 0,
                         const uint32_t* n_dev = nullptr, const uint64_t* label_base = nullptr,
                         const PreArgs* pre = nullptr, const uint32_t* seg_kept = nullptr) {
  *launched = false;
  if (g.variant == 0 || prm.n == 0) return TPX3_OK;
  // the 128-bit load phase needs its arrays on a 16-byte boundary: a chunk of a resident stream that starts at any event
  // is served by moving all of them down to the boundary alike (FusedArgs::head); arrays that are not aligned alike,
  // and the calls whose count lives on the device or that preprocess (library-owned, resp. checked by the caller): not
  const int e = fused_head_of(mode, x, y, toa, tot, perm);
  if (e < 0 || (e > 0 && (n_dev != nullptr || mode == 4u))) return TPX3_OK;
  FusedArgs a = make_fused_args(g.T, num_sms, ctrl, tiles, prm, x, y, toa, tot, perm, label, max_clusters, out,
                                n_clusters, stage, mode, lm_wx, lm_wy, n_dev);
  if (e > 0) fused_apply_head(a, (uint32_t)e, g.T);
  a.label_base = label_base;
  if (pre) { a.pre = *pre; a.seg_kept = seg_kept; }
  if (n_dev) {   // grids that cover every count up to prm.n (fused_segs: a short input is cut into up to `want` segments)
    const uint32_t want = num_sms * (g.T <= 2048u ? 4u : (g.T <= 4096u ? 2u : 1u)) * 8u + 1u;
    if (a.nseg < want) a.nseg = want;
    a.num_tiles = a.nseg * 22u;     // maxt <= 2 * (8 + 2) + 2
  }
  *args = a;
  int rc;
#define TPX3_PICK(MODE_)                                                \
  (g.variant == 3 ? launch_fused<2048, 256, MODE_>(a, st)               \
                  : g.variant == 1 ? launch_fused<4096, 512, MODE_>(a, st) : launch_fused<8192, 1024, MODE_>(a, st))
  if (mode == 0u) rc = TPX3_PICK(0);
  else if (mode == 1u) rc = TPX3_PICK(1);
  else if (mode == 2u) rc = TPX3_PICK(2);
  else if (mode == 4u) rc = TPX3_PICK(4);
  else rc = TPX3_PICK(3);
#undef TPX3_PICK
  if (rc != TPX3_OK) return rc;
  ++*launches;
  uint32_t ctas, tiles_per_cta;
  compact_grid(a.num_tiles, num_sms, &ctas, &tiles_per_cta);
  if (n_dev) ctas = num_sms * 8u;   // the kernel sizes itself from the device's count: the most compact_grid ever asks for
  k_fused_compact<<<ctas, kCompactThreads, 0, st>>>(a, tiles_per_cta, g.T);
  if (cudaGetLastError() != cudaSuccess) return TPX3_ERR_CUDA;
  ++*launches;
  *launched = true;
  return TPX3_OK;
}

}  // namespace tpx3
