// libtpx3 — host side of the C ABI declared in include/tpx3.h: plan, workspace layout, kernel
// launches. All device work is enqueued on the caller's stream; nothing here synchronises
// except tpx3_status and tpx3_process_host (which say so in the header).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "tpx3_centroid.cuh"
#include "tpx3_common.cuh"
#include "tpx3_fused.cuh"
#include "tpx3_link.cuh"
#include "tpx3_localmax.cuh"
#include "tpx3_preprocess.cuh"
#include "tpx3_sort.cuh"
#include "tpx3_stream.cuh"
#include "tpx3_unwrap.cuh"

using namespace tpx3;

struct tpx3_plan_s {
  tpx3_config_t cfg;
  Params prm;               // n filled per call
  size_t workspace_bytes;
  uint64_t launches;
  int num_sms;
  // workspace offsets (bytes from the workspace base), sized for cfg.max_hits
  size_t off_keyA, off_keyB, off_idxA, off_idxB, off_xy, off_tot, off_slab, off_table, off_counts;
  size_t off_slot, off_peak, off_blkcnt, off_tiles, off_segk;
  uint32_t table_mask_max;
  FusedGeom fused;          // which fused variant serves this plan (variant 0: none)
  // optional per-stage timing (tpx3_profile_*)
  bool profiling;
  struct Span { int stage; cudaEvent_t a, b; uint64_t launches0, launches1; };
  std::vector<Span> spans;
  std::vector<cudaEvent_t> free_events;
  uint64_t profiled_calls;
  cudaStream_t copy_in, copy_out;   // copy streams of the pipelined tpx3_process_host (created on first use)
  int host_route;           // last tpx3_process_host: 0 one piece, 1 pipelined, 2 pipelined attempt redone in one piece
  bool device_ready;        // use_device has run for this plan
};

namespace {

inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

__host__ __device__ inline uint32_t table_size_for(uint64_t n) {  // power of two >= 2n, >= 1024
  uint64_t s = 1024;
  while (s < 2 * n) s <<= 1;
  return (uint32_t)s;
}

#define TPX3_LAUNCH(plan, kernel, grid, block, smem, stream, ...)          \
  do {                                                                     \
    kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);            \
    ++(plan)->launches;                                                    \
  } while (0)

inline int cuda_ok(cudaError_t e) { return e == cudaSuccess ? TPX3_OK : TPX3_ERR_CUDA; }

// RAII bracket of one stage: records an event pair on the stream when profiling is enabled.
struct StageTimer {
  tpx3_plan_s* p;
  cudaStream_t st;
  size_t slot;
  bool on;
  static cudaEvent_t take(tpx3_plan_s* p) {
    cudaEvent_t e = nullptr;
    if (!p->free_events.empty()) { e = p->free_events.back(); p->free_events.pop_back(); return e; }
    cudaEventCreate(&e);
    return e;
  }
  StageTimer(tpx3_plan_s* plan, cudaStream_t stream, int stage) : p(plan), st(stream), slot(0), on(plan->profiling) {
    if (!on) return;
    tpx3_plan_s::Span s;
    s.stage = stage; s.a = take(p); s.b = take(p); s.launches0 = p->launches; s.launches1 = p->launches;
    cudaEventRecord(s.a, st);
    slot = p->spans.size();
    p->spans.push_back(s);
  }
  ~StageTimer() {
    if (!on) return;
    cudaEventRecord(p->spans[slot].b, st);
    p->spans[slot].launches1 = p->launches;
  }
};

struct Ws {
  Ctrl* ctrl;
  uint64_t *keyA, *keyB, *slab;
  uint32_t *idxA, *idxB, *xy, *table, *counts, *slot, *blkcnt;
  uint16_t* tot;
  unsigned long long* peak;
  unsigned long long* tiles;
  uint32_t* segk;
};

inline Ws carve(const tpx3_plan_s* p, void* workspace) {
  char* b = (char*)workspace;
  Ws w;
  w.ctrl = (Ctrl*)b;
  w.keyA = (uint64_t*)(b + p->off_keyA);
  w.keyB = (uint64_t*)(b + p->off_keyB);
  w.idxA = (uint32_t*)(b + p->off_idxA);
  w.idxB = (uint32_t*)(b + p->off_idxB);
  w.xy = (uint32_t*)(b + p->off_xy);
  w.tot = (uint16_t*)(b + p->off_tot);
  w.slab = (uint64_t*)(b + p->off_slab);
  w.table = (uint32_t*)(b + p->off_table);
  w.counts = (uint32_t*)(b + p->off_counts);
  w.slot = (uint32_t*)(b + p->off_slot);
  w.peak = (unsigned long long*)(b + p->off_peak);
  w.blkcnt = (uint32_t*)(b + p->off_blkcnt);
  w.tiles = (unsigned long long*)(b + p->off_tiles);
  w.segk = (uint32_t*)(b + p->off_segk);
  return w;
}

// ---- general path: S0-S3 (cluster) and S4-S5 (centroid) ------------------------------------------
// Everything the general kernels need, by value: the same launch sequence is enqueued by the host
// (tpx3_cluster, tpx3_centroid, plans without a fused variant) or, when the fused kernel gave up,
// by k_fallback_dispatch on the device.
struct GenArgs {
  Ws w;
  Params prm;            // n filled in
  SortGeom g;
  uint32_t tsize;        // hash table slots
  uint32_t cent_nblk;
  int sms;
  int general_only;      // centroid kernels: skip when the fused path succeeded
  const uint16_t *x, *y, *tot;
  const uint64_t* toa;
  uint32_t *perm, *label, *n_clusters;
  uint64_t max_clusters;
  tpx3_clusters_t out;
  uint32_t lm_wx, lm_wy;   // paper-literal mode: box half-widths
  uint64_t lm_wt;
  const uint64_t* label_base;   // [dev] or null (stream pushes): added to the label column
  int sorted_tiles;             // the plan has a tile kernel: after the global sort, link through it first (mode 5)
};

// The fields that depend on the event count (a stream push learns it on the device).
__host__ __device__ inline void gen_set_n(GenArgs& a, uint64_t n) {
  a.prm.n = n;
  a.g = sort_geom(n);
  a.tsize = table_size_for(n);
  a.cent_nblk = (uint32_t)((n + kCentTile - 1) / kCentTile);
  if (a.cent_nblk == 0) a.cent_nblk = 1;
}

__host__ __device__ inline uint32_t grid_for_hd(uint64_t n, int threads, int num_sms, int per_sm = 8) {
  uint64_t b = (n + threads - 1) / threads;
  uint64_t cap = (uint64_t)num_sms * per_sm;
  if (b > cap) b = cap;
  return (uint32_t)(b ? b : 1);
}

// GP(stage, kernel, grid, block, args...) is defined by the includer (host launch or device tail launch).
#define TPX3_GENERAL_CLUSTER_SEQUENCE(A)                                                                              \
  do {                                                                                                                \
    TPX3_GENERAL_SORT_SEQUENCE(A);                                                                                    \
    TPX3_GENERAL_LINK_SEQUENCE(A);                                                                                    \
  } while (0)

#define TPX3_GENERAL_SORT_SEQUENCE(A)                                                                                 \
  do {                                                                                                                \
    const uint64_t n_ = (A).prm.n;                                                                                    \
    SortBufs b_;                                                                                                      \
    b_.key[0] = (A).w.keyA; b_.key[1] = (A).w.keyB; b_.idx[0] = (A).w.idxA; b_.idx[1] = (A).w.idxB;                   \
    b_.counts = (A).w.counts;                                                                                         \
    GP(TPX3_STAGE_SORT, k_minmax, grid_for_hd(n_, 256 * 8, (A).sms), 256, (A).w.ctrl, (A).toa, n_);                   \
    GP(TPX3_STAGE_SORT, k_sort_setup, 1, 1, (A).w.ctrl);                                                              \
    /* passes needed for the largest span a ToA can have; the ones past the device-computed npass return at once */  \
    for (int pass_ = 0; pass_ < kMaxPasses; ++pass_) {                                                                \
      GP(TPX3_STAGE_SORT, k_radix_hist, (A).g.nblk, kSortThreads, (A).w.ctrl, pass_, (A).toa, b_, n_, (A).g);         \
      GP(TPX3_STAGE_SORT, k_radix_scan, kRadix / 8, 256, (A).w.ctrl, pass_, (A).w.counts, (A).g.nblk);                 \
      GP(TPX3_STAGE_SORT, k_radix_scatter, (A).g.nblk, kSortThreads, (A).w.ctrl, pass_, (A).toa, b_, (A).perm, n_,    \
         (A).g);                                                                                                      \
      GP(TPX3_STAGE_SORT, k_radix_scatter_packed, (A).g.nblk, kSortThreads, (A).w.ctrl, pass_, (A).toa, b_,           \
         (A).perm, n_, (A).g);                                                                                        \
    }                                                                                                                 \
  } while (0)

#define TPX3_GENERAL_LINK_SEQUENCE(A)                                                                                 \
  do {                                                                                                                \
    const uint64_t n_ = (A).prm.n;                                                                                    \
    GP(TPX3_STAGE_LINK, k_gather, grid_for_hd(n_, 256, (A).sms), 256, (A).w.ctrl, (A).prm, (A).w.keyA, (A).w.keyB,    \
       (A).perm, (A).x, (A).y, (A).tot, (A).w.xy, (A).w.tot, (A).w.slab, (A).label);                                  \
    GP(TPX3_STAGE_LINK, k_fill_u32, grid_for_hd((A).tsize, 256, (A).sms), 256, (A).w.ctrl, 1, (A).w.table,            \
       (uint64_t)(A).tsize, kEmpty);                                                                                  \
    GP(TPX3_STAGE_LINK, k_hash_insert, grid_for_hd(n_, 256, (A).sms), 256, (A).w.ctrl, n_, (A).w.xy, (A).w.slab,      \
       (A).w.table, (A).tsize - 1);                                                                                   \
    GP(TPX3_STAGE_LINK, k_link, grid_for_hd(n_, 256, (A).sms), 256, (A).w.ctrl, (A).prm, (A).w.keyA, (A).w.keyB,      \
       (A).w.xy, (A).w.slab, (A).w.table, (A).tsize - 1, (A).label);                                                  \
    GP(TPX3_STAGE_LINK, k_compress, grid_for_hd(n_, 256, (A).sms), 256, (A).w.ctrl, n_, (A).label, (A).n_clusters);   \
  } while (0)

#define TPX3_GENERAL_CENTROID_SEQUENCE(A)                                                                             \
  do {                                                                                                                \
    const uint64_t n_ = (A).prm.n;                                                                                    \
    GP(TPX3_STAGE_CENTROID, k_root_count, (A).cent_nblk, kCentThreads, (A).w.ctrl, (A).general_only, n_, (A).label,   \
       (A).w.blkcnt);                                                                                                 \
    GP(TPX3_STAGE_CENTROID, k_root_scan, 1, 1024, (A).w.ctrl, (A).general_only, (A).w.blkcnt, (A).cent_nblk,          \
       (A).max_clusters, (A).n_clusters);                                                                             \
    GP(TPX3_STAGE_CENTROID, k_root_slots, (A).cent_nblk, kCentThreads, (A).w.ctrl, (A).general_only, n_, (A).label,   \
       (A).w.blkcnt, (A).w.slot, (A).max_clusters, (A).out, (A).w.peak);                                              \
    GP(TPX3_STAGE_CENTROID, k_accumulate, grid_for_hd(n_, 256, (A).sms), 256, (A).w.ctrl, (A).general_only, n_,       \
       (A).x, (A).y, (A).tot, (A).toa, (A).prm.P, (A).perm, (A).label, (A).w.slot, (A).max_clusters, (A).out,        \
       (A).w.peak);                \
    GP(TPX3_STAGE_CENTROID, k_finalize,                                                                               \
       grid_for_hd((A).max_clusters < n_ ? (A).max_clusters : n_, 256, (A).sms), 256, (A).w.ctrl, (A).general_only,   \
       (A).prm, (A).toa, (A).perm, (A).n_clusters, (A).max_clusters, (A).out, (A).w.peak, (A).label_base);            \
  } while (0)

// Paper-literal mode on the general kernels: the sort stage, then the window walks of tpx3_localmax.cuh. The
// link stage's buffers hold the sorted records (slab: ToA, xy: x | y << 8 | tot << 16); the centroid stage's
// ordinal kernels run on lmax (passed as `label`) in place of the labels.
#define TPX3_LOCALMAX_SEQUENCE(A)                                                                                     \
  do {                                                                                                                \
    TPX3_GENERAL_SORT_SEQUENCE(A);                                                                                    \
    const uint64_t m_ = (A).prm.n;                                                                                    \
    GP(TPX3_STAGE_LINK, k_lm_gather, grid_for_hd(m_, 256, (A).sms), 256, m_, (A).perm, (A).x, (A).y, (A).toa,         \
       (A).tot, (A).w.slab, (A).w.xy);                                                                                \
    GP(TPX3_STAGE_LINK, k_lm_flag, grid_for_hd(m_, 256, (A).sms, 16), 256, m_, (A).prm.P, (A).lm_wx, (A).lm_wy,       \
       (A).lm_wt, (A).w.slab, (A).w.xy, (A).label);                                                                   \
    GP(TPX3_STAGE_CENTROID, k_root_count, (A).cent_nblk, kCentThreads, (A).w.ctrl, 0, m_, (A).label, (A).w.blkcnt);   \
    GP(TPX3_STAGE_CENTROID, k_root_scan, 1, 1024, (A).w.ctrl, 0, (A).w.blkcnt, (A).cent_nblk, (A).max_clusters,       \
       (A).n_clusters);                                                                                               \
    GP(TPX3_STAGE_CENTROID, k_root_slots, (A).cent_nblk, kCentThreads, (A).w.ctrl, 0, m_, (A).label, (A).w.blkcnt,    \
       (A).w.slot, (A).max_clusters, (A).out, (A).w.peak);                                                            \
    GP(TPX3_STAGE_CENTROID, k_lm_emit, grid_for_hd((A).max_clusters < m_ ? (A).max_clusters : m_, 128, (A).sms, 16),  \
       128, (A).w.ctrl, m_, (A).prm.P, (A).lm_wx, (A).lm_wy, (A).lm_wt, (A).w.slab, (A).w.xy, (A).n_clusters,         \
       (A).max_clusters, (A).out);                                                                                    \
  } while (0)

// Device-side fallback: one tiny kernel behind the fused path. If the fused kernel served the call it returns
// at once. Otherwise it enqueues, as tail launches (they run, in order, after this grid and before anything
// the host enqueued later on the stream), either the next rung of the shot-length ladder (plans without a
// hint: the same tile kernel with room for longer shots, then this dispatcher again) or, after the last rung,
// the whole general path. A successful fused call thus pays for one empty launch instead of the 36 early-exit
// launches of the general path. lm != 0: the paper-literal mode.
__global__ void k_general_sorted_tiles(GenArgs a, FusedArgs fa, int what);
__global__ void k_general_slab(GenArgs a, int what);

__global__ void k_fallback_dispatch(GenArgs a, FusedArgs fa, FusedLadder ladder, int rung, int what) {
  Ctrl* c = a.w.ctrl;
  if (c->fused_state == 1u) return;
  if (fa.n_dev) {                       // a stream push: the count is device state
    const uint64_t n = *fa.n_dev;
    if (n == 0) return;
    gen_set_n(a, n);
    fa.n = n;
  }
  if (rung < ladder.n) {
    c->tiles_done = 0; c->fused_fail = 0; c->fused_state = 0; c->tight_tiles = 0; c->tiles_run = 0;
    const FusedSegs sg = fused_segs(fa.n, ladder.T[rung], fa.num_sms);
    fa.G = sg.G; fa.nseg = sg.nseg; fa.maxt = sg.maxt; fa.num_tiles = sg.nseg * sg.maxt;
    launch_fused_rung_device(fa, ladder.T[rung]);
    k_fallback_dispatch<<<1, 1, 0, cudaStreamTailLaunch>>>(a, fa, ladder, rung + 1, what);
    return;
  }
  if (what == 4) {                      // the fused preprocessing call has no second route: the status word says so
    set_error(c, TPX3_ERR_NOT_CONTIGUOUS);
    return;
  }
#define GP(stage, kernel, grid, block, ...) kernel<<<(grid), (block), 0, cudaStreamTailLaunch>>>(__VA_ARGS__)
  if (what == 1 && !a.sorted_tiles) {
    TPX3_LOCALMAX_SEQUENCE(a);
  } else if (what != 3 && a.sorted_tiles) {
    // general route, first choice: the global sort, then the tile kernel on the sorted stream (read through perm)
    TPX3_GENERAL_SORT_SEQUENCE(a);
    k_general_sorted_tiles<<<1, 1, 0, cudaStreamTailLaunch>>>(a, fa, what);
  } else {
    if (what != 3) TPX3_GENERAL_CLUSTER_SEQUENCE(a);
    if (what != 2) TPX3_GENERAL_CENTROID_SEQUENCE(a);
  }
#undef GP
}

// General route, last resort (one shot longer than a tile, P = 0 plans never get here): global sort again (the
// tile attempt's staging table aliases the sort buffers), slab-hash linking, atomic sums.
__global__ void k_general_slab(GenArgs a, int what) {
  Ctrl* c = a.w.ctrl;
  if (c->fused_state == 1u) return;
#define GP(stage, kernel, grid, block, ...) kernel<<<(grid), (block), 0, cudaStreamTailLaunch>>>(__VA_ARGS__)
  if (what == 1) {
    TPX3_LOCALMAX_SEQUENCE(a);
  } else {
    TPX3_GENERAL_CLUSTER_SEQUENCE(a);
    if (what != 2) TPX3_GENERAL_CENTROID_SEQUENCE(a);
  }
#undef GP
}

// General route behind the global sort: perm now IS the (shot, ToA) order of ANY input (shots interleaved in the
// stream, a globally shuffled file), so the tile kernel can finish the call reading the events through perm
// (mode 5, 8192-event windows). Only a shot that does not fit a window sends the call on to k_general_slab.
__global__ void k_general_sorted_tiles(GenArgs a, FusedArgs fa, int what) {
  Ctrl* c = a.w.ctrl;
  c->tiles_done = 0; c->fused_fail = 0; c->fused_state = 0; c->tight_tiles = 0; c->tiles_run = 0;
  fused_rebase_mode5(fa, what == 2 ? 1u : 0u, what == 1 ? 6u : 5u);
  launch_fused_rung_device(fa, 8192u);
  k_general_slab<<<1, 1, 0, cudaStreamTailLaunch>>>(a, what);
}

GenArgs make_gen_args(tpx3_plan_s* p, const Ws& w, int general_only, uint64_t n, const uint16_t* x, const uint16_t* y,
                      const uint64_t* toa, const uint16_t* tot, uint32_t* perm, uint32_t* label, uint64_t max_clusters,
                      const tpx3_clusters_t* out, uint32_t* n_clusters) {
  GenArgs a;
  memset(&a, 0, sizeof(a));
  a.w = w;
  a.prm = p->prm;
  gen_set_n(a, n);
  a.sms = p->num_sms;
  a.general_only = general_only;
  a.x = x; a.y = y; a.tot = tot; a.toa = toa;
  a.perm = perm; a.label = label; a.n_clusters = n_clusters;
  a.max_clusters = max_clusters;
  if (out) a.out = *out;
  return a;
}

// Host-side enqueue with per-stage timing brackets.
struct HostLauncher {
  tpx3_plan_s* p;
  cudaStream_t st;
  int cur;
  bool open;
  size_t slot;
  void enter(int stage) {
    if (!p->profiling || (open && cur == stage)) return;
    leave();
    tpx3_plan_s::Span s;
    s.stage = stage; s.a = StageTimer::take(p); s.b = StageTimer::take(p); s.launches0 = p->launches; s.launches1 = p->launches;
    cudaEventRecord(s.a, st);
    slot = p->spans.size();
    p->spans.push_back(s);
    cur = stage;
    open = true;
  }
  void leave() {
    if (!open) return;
    cudaEventRecord(p->spans[slot].b, st);
    p->spans[slot].launches1 = p->launches;
    open = false;
  }
};

int enqueue_general_cluster(tpx3_plan_s* p, const GenArgs& a, cudaStream_t st) {
  HostLauncher hl{p, st, -1, false, 0};
#define GP(stage, kernel, grid, block, ...)                        \
  do {                                                             \
    hl.enter(stage);                                               \
    kernel<<<(grid), (block), 0, st>>>(__VA_ARGS__);               \
    ++p->launches;                                                 \
  } while (0)
  TPX3_GENERAL_CLUSTER_SEQUENCE(a);
  hl.leave();
  return cuda_ok(cudaGetLastError());
}

int enqueue_general_sort(tpx3_plan_s* p, const GenArgs& a, cudaStream_t st) {
  HostLauncher hl{p, st, -1, false, 0};
  TPX3_GENERAL_SORT_SEQUENCE(a);
  hl.leave();
  return cuda_ok(cudaGetLastError());
}

int enqueue_localmax(tpx3_plan_s* p, const GenArgs& a, cudaStream_t st) {
  HostLauncher hl{p, st, -1, false, 0};
  TPX3_LOCALMAX_SEQUENCE(a);
  hl.leave();
  return cuda_ok(cudaGetLastError());
}

int enqueue_centroid(tpx3_plan_s* p, const GenArgs& a, cudaStream_t st) {
  HostLauncher hl{p, st, -1, false, 0};
  TPX3_GENERAL_CENTROID_SEQUENCE(a);
  hl.leave();
#undef GP
  return cuda_ok(cudaGetLastError());
}

// Every device call starts here: makes the plan's device current and, the first time for a plan, reads its SM
// count and opts the fused kernels in to their dynamic shared memory. The opt-in is per function AND per device,
// so it is tied to the plan (one plan = one device), not to the process; tpx3_plan itself stays host-only.
// Concurrent first calls on one plan are the caller's to serialise (a plan is not thread-safe anyway: it counts
// launches); the work is idempotent.
int use_device(tpx3_plan_s* p) {
  if (cudaSetDevice(p->cfg.device) != cudaSuccess) return TPX3_ERR_CUDA;
  if (!p->device_ready) {
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->cfg.device) != cudaSuccess || sms <= 0)
      return TPX3_ERR_CUDA;
    if (fused_configure_device() != TPX3_OK) return TPX3_ERR_CUDA;
    p->num_sms = sms;
    p->device_ready = true;
  }
  return TPX3_OK;
}

bool clusters_ok(const tpx3_clusters_t* o) {
  return o && o->label && o->size && o->shot && o->sum_tot && o->sum_tot_x && o->sum_tot_y && o->toa_peak && o->cx &&
         o->cy && o->sum_tot_tof && o->ctof;
}

}  // namespace

extern "C" {

int tpx3_plan(const tpx3_config_t* cfg, tpx3_plan_t* out_plan, size_t* workspace_bytes) {
  if (!cfg || !out_plan || !workspace_bytes) return TPX3_ERR_INVALID_ARG;
  if (cfg->struct_size != sizeof(tpx3_config_t)) return TPX3_ERR_INVALID_ARG;
  if (cfg->sensor_w == 0 || cfg->sensor_h == 0 || cfg->sensor_w > 256 || cfg->sensor_h > 256)
    return TPX3_ERR_INVALID_ARG;
  if (cfg->max_hits == 0 || cfg->max_hits > kMaxHits) return TPX3_ERR_INVALID_ARG;
  if (cfg->toa_window_ticks >= (1u << 31)) return TPX3_ERR_INVALID_ARG;
  if (cfg->device < 0 || cfg->reserved != 0) return TPX3_ERR_INVALID_ARG;
  tpx3_plan_s* p = new (std::nothrow) tpx3_plan_s();
  if (!p) return TPX3_ERR_CUDA;
  p->cfg = *cfg;
  p->launches = 0;
  p->profiling = false;
  p->profiled_calls = 0;
  p->copy_in = p->copy_out = nullptr;
  p->host_route = 0;
  p->num_sms = kNumSMs;      // until the first device call reads the device's count (use_device)
  p->device_ready = false;
  Params& prm = p->prm;
  prm.n = 0;
  prm.P = cfg->shot_period_ticks;
  prm.W = cfg->toa_window_ticks;
  prm.sensor_w = cfg->sensor_w;
  prm.sensor_h = cfg->sensor_h;
  prm.flags = cfg->flags;
  prm.slabs_per_shot_p1 = prm.P ? (prm.P + prm.W) / (prm.W + 1ull) + 1ull : 0ull;
  p->fused = fused_geom(prm.P, prm.W, cfg->max_shot_hits);
  const uint64_t N = cfg->max_hits;
  size_t o = 256;  // Ctrl
  // general-path cluster buffers
  p->off_keyA = o; o = align_up(o + 8 * N);
  p->off_keyB = o; o = align_up(o + 8 * N);
  p->off_idxA = o; o = align_up(o + 4 * N);
  p->off_idxB = o; o = align_up(o + 4 * N);
  p->off_xy = o; o = align_up(o + 4 * N);
  p->off_tot = o; o = align_up(o + 2 * N);
  p->off_slab = o; o = align_up(o + 8 * N);
  p->off_table = o; o = align_up(o + 4 * (size_t)table_size_for(N));
  p->off_counts = o; o = align_up(o + 4 * (size_t)kRadix * (kSortMaxBlocks + 1));   // + the digit totals
  // the fused path's staging table (48 bytes per event) aliases keyA .. table
  if (o - p->off_keyA < 48 * (size_t)(N + 8)) o = align_up(p->off_keyA + 48 * (size_t)(N + 8));   // + 8: FusedArgs::head
  // centroid buffers alias the sort buffers (the two steps never run concurrently and the
  // centroid step takes perm/label from the caller, not from the workspace)
  p->off_slot = p->off_keyA;                    // 4N <= 8N
  p->off_peak = p->off_keyB;                    // 8N
  p->off_blkcnt = p->off_idxA;                  // 4 * ceil(N/4096) <= 4N
  p->off_tiles = o; o = align_up(o + 8 * (size_t)(N / 128 + 262144));   // fused path tile status words (fused_segs: nseg * maxt)
  // fused preprocessing call: surviving events in front of every segment (read while the staging table is written,
  // so it may not alias the sort buffers)
  p->off_segk = o; o = align_up(o + 4 * (size_t)(N / 4096 + 16384));
  p->workspace_bytes = o;
  *workspace_bytes = o;
  *out_plan = p;
  return TPX3_OK;
}

// S0-S3 / S4-S5 / S0-S5 share one body: the fused tile kernel in the mode that matches the call (0: everything,
// 2: stop after the labels, 3: start from the caller's perm / label), with the general kernels enqueued from the
// device when it gives up.
static int run_fused_or_general(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                                const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint32_t* perm,
                                uint32_t* label, uint64_t max_clusters, const tpx3_clusters_t* out, uint32_t* n_clusters,
                                uint32_t mode, const tpx3::StreamCtrl* sc = nullptr) {
  // sc != null: a stream push. n is then the LARGEST count the push can emit; the true one (sc->n_work) is
  // device state that every kernel reads for itself, so the host never waits for it.
  const uint32_t* n_dev = sc ? &sc->n_work : nullptr;
  const uint64_t* label_base = sc ? &sc->label_base : nullptr;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  Ws w = carve(p, workspace);
  if (p->profiling) ++p->profiled_calls;
  const bool try_fused = !(p->cfg.flags & TPX3_FLAG_FORCE_GENERAL) && p->fused.variant != 0 && n != 0;
  TPX3_LAUNCH(p, k_ctrl_init, 1, 256, 0, st, w.ctrl, n, w.tiles, 0u, n_clusters, n_dev, sc ? &sc->dead : nullptr);
  if (n == 0) return cuda_ok(cudaGetLastError());
  Params prm = p->prm;
  prm.n = n;
  int rc = TPX3_OK;
  tpx3_clusters_t none;
  memset(&none, 0, sizeof(none));
  GenArgs ga = make_gen_args(p, w, mode == 2u ? 0 : 1, n, x, y, toa, tot, perm, label, max_clusters, out, n_clusters);
  ga.label_base = label_base;
  // the general route links through the tile kernel too, behind its global sort (mode 5), when the plan has one
  ga.sorted_tiles = p->fused.variant != 0 && mode != 3u && ((uintptr_t)perm & 3u) == 0;
  if (sc && !try_fused) {   // general kernels only: launched from the device, which knows the count
    FusedArgs fa = make_fused_args(2048u, (uint32_t)p->num_sms, w.ctrl, w.tiles, prm, x, y, toa, tot, perm, label,
                                   max_clusters, out ? *out : none, n_clusters, (char*)workspace + p->off_keyA, mode, 0u,
                                   0u, n_dev);
    fa.label_base = label_base;
    k_fallback_dispatch<<<1, 1, 0, st>>>(ga, fa, FusedLadder{0, {0, 0}}, 0, (int)mode);
    ++p->launches;
    return cuda_ok(cudaGetLastError());
  }
  if (try_fused) {
    bool launched = false;
    StageTimer timer(p, st, TPX3_STAGE_FUSED);
    FusedArgs fa;
    rc = enqueue_fused(p->fused, (uint32_t)p->num_sms, &p->launches, w.ctrl, w.tiles, st, prm, x, y, toa, tot, perm, label,
                       max_clusters, out ? *out : none, n_clusters, (char*)workspace + p->off_keyA, &launched, &fa, mode,
                       0u, 0u, n_dev, label_base);
    if (rc != TPX3_OK) return rc;
    if (launched) {
      // the next rung or the general path, only if the fused kernel gave up: decided and enqueued on the device
      k_fallback_dispatch<<<1, 1, 0, st>>>(ga, fa, fused_ladder(p->cfg.max_shot_hits), 0, (int)mode);
      ++p->launches;
      return cuda_ok(cudaGetLastError());
    }
  }
  if (ga.sorted_tiles) {
    // global sort, then the tile kernel on the sorted stream (read through perm); the slab-hash kernels only if a
    // shot does not fit a window (decided on the device: k_general_slab)
    rc = enqueue_general_sort(p, ga, st);
    if (rc != TPX3_OK) return rc;
    {
      StageTimer timer(p, st, TPX3_STAGE_FUSED);
      FusedArgs fa = make_fused_args(8192u, (uint32_t)p->num_sms, w.ctrl, w.tiles, prm, x, y, toa, tot, perm, label,
                                     max_clusters, out ? *out : none, n_clusters, (char*)workspace + p->off_keyA, 5u, 0u,
                                     0u, nullptr);
      fa.label_base = label_base;
      fused_rebase_mode5(fa, mode == 2u ? 1u : 0u);
      k_fused_shot_tiles<8192, 1024, 5><<<fa.nseg, 1024, FusedSmem<8192>::kBytes, st>>>(fa);
      uint32_t ctas, tpc;
      compact_grid(fa.num_tiles, (uint32_t)p->num_sms, &ctas, &tpc);
      k_fused_compact<<<ctas, kCompactThreads, 0, st>>>(fa, tpc, 8192u);
      k_general_slab<<<1, 1, 0, st>>>(ga, (int)mode);
      p->launches += 3;
    }
    return cuda_ok(cudaGetLastError());
  }
  if (mode != 3u) {
    rc = enqueue_general_cluster(p, ga, st);
    if (rc != TPX3_OK) return rc;
  }
  return mode != 2u ? enqueue_centroid(p, ga, st) : TPX3_OK;
}

int tpx3_cluster(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x, const uint16_t* y,
                 const uint64_t* toa, const uint16_t* tot, uint32_t* perm, uint32_t* label, uint32_t* n_clusters) {
  if (!p || !workspace || !n_clusters) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot || !perm || !label)) return TPX3_ERR_INVALID_ARG;
  return run_fused_or_general(p, workspace, cuda_stream, n, x, y, toa, tot, perm, label, 0, nullptr, n_clusters, 2u);
}

int tpx3_centroid(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x, const uint16_t* y,
                  const uint64_t* toa, const uint16_t* tot, const uint32_t* perm, const uint32_t* label,
                  uint64_t max_clusters, const tpx3_clusters_t* out, uint32_t* n_clusters) {
  if (!p || !workspace || !n_clusters) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot || !perm || !label)) return TPX3_ERR_INVALID_ARG;
  if (max_clusters && !clusters_ok(out)) return TPX3_ERR_INVALID_ARG;
  if (n && !out) return TPX3_ERR_INVALID_ARG;
  return run_fused_or_general(p, workspace, cuda_stream, n, x, y, toa, tot, const_cast<uint32_t*>(perm),
                              const_cast<uint32_t*>(label), max_clusters, out, n_clusters, 3u);
}

int tpx3_cluster_centroid(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                          const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint32_t* perm, uint32_t* label,
                          uint64_t max_clusters, const tpx3_clusters_t* out, uint32_t* n_clusters) {
  if (!p || !workspace || !n_clusters) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot || !perm || !label || !out)) return TPX3_ERR_INVALID_ARG;
  if (max_clusters && !clusters_ok(out)) return TPX3_ERR_INVALID_ARG;
  return run_fused_or_general(p, workspace, cuda_stream, n, x, y, toa, tot, perm, label, max_clusters, out, n_clusters, 0u);
}

int tpx3_preprocess_cluster_centroid(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                                     const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint64_t n_trig,
                                     const uint64_t* trig, uint64_t cut, const int32_t* table, uint32_t table_len,
                                     uint64_t shot_base, uint32_t* perm, uint32_t* label, uint64_t max_clusters,
                                     const tpx3_clusters_t* out, uint32_t* n_clusters, uint32_t* n_kept) {
  if (!p || !workspace || !n_clusters || !n_kept) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits || (cut >> 63) != 0) return TPX3_ERR_INVALID_ARG;
  if (p->fused.variant == 0 || p->cfg.max_shot_hits == 0) return TPX3_ERR_INVALID_ARG;   // needs a tile kernel and its window
  if (n && (!x || !y || !toa || !tot || !perm || !label || !out)) return TPX3_ERR_INVALID_ARG;
  if ((n_trig && !trig) || (table_len && !table)) return TPX3_ERR_INVALID_ARG;
  if (max_clusters && !clusters_ok(out)) return TPX3_ERR_INVALID_ARG;
  if ((((uintptr_t)x | (uintptr_t)y | (uintptr_t)toa | (uintptr_t)tot) & 15u) != 0) return TPX3_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  Ws w = carve(p, workspace);
  if (p->profiling) ++p->profiled_calls;
  TPX3_LAUNCH(p, k_ctrl_init, 1, 256, 0, st, w.ctrl, n, w.tiles, 0u, n_clusters);
  if (n == 0) {
    if (cudaMemsetAsync(n_kept, 0, sizeof(uint32_t), st) != cudaSuccess) return TPX3_ERR_CUDA;
    return cuda_ok(cudaGetLastError());
  }
  PreArgs pa;
  memset(&pa, 0, sizeof(pa));
  pa.n = n; pa.x = x; pa.y = y; pa.tot = tot; pa.toa = toa; pa.n_trig = n_trig; pa.trig = trig; pa.cut = cut;
  pa.P = p->cfg.shot_period_ticks; pa.shot_base = shot_base; pa.table = table; pa.table_len = table_len;
  Params prm = p->prm;
  prm.n = n;
  StageTimer timer(p, st, TPX3_STAGE_FUSED);
  // pre-pass: surviving events in front of every segment of the tile kernel's grid (same segment length)
  const FusedSegs sg = fused_segs(n, p->fused.T, (uint32_t)p->num_sms);
  TPX3_LAUNCH(p, k_pre_seg_count, sg.nseg, kPreThreads, 0, st, pa, sg.G, w.segk);
  TPX3_LAUNCH(p, k_pre_seg_scan, 1, 1024, 0, st, w.segk, sg.nseg, n_kept);
  GenArgs ga = make_gen_args(p, w, 1, n, x, y, toa, tot, perm, label, max_clusters, out, n_clusters);
  bool launched = false;
  FusedArgs fa;
  int rc = enqueue_fused(p->fused, (uint32_t)p->num_sms, &p->launches, w.ctrl, w.tiles, st, prm, x, y, toa, tot, perm,
                         label, max_clusters, *out, n_clusters, (char*)workspace + p->off_keyA, &launched, &fa, 4u, 0u, 0u,
                         nullptr, nullptr, &pa, w.segk);
  if (rc != TPX3_OK) return rc;
  if (!launched) return TPX3_ERR_INVALID_ARG;
  k_fallback_dispatch<<<1, 1, 0, st>>>(ga, fa, FusedLadder{0, {0, 0}}, 0, 4);
  ++p->launches;
  return cuda_ok(cudaGetLastError());
}

int tpx3_localmax_centroid(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                           const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint32_t wx, uint32_t wy,
                           uint32_t wt, uint32_t* perm, uint32_t* lmax, uint64_t max_clusters,
                           const tpx3_clusters_t* out, uint32_t* n_hits) {
  if (!p || !workspace || !n_hits) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot || !perm || !lmax || !out)) return TPX3_ERR_INVALID_ARG;
  if (max_clusters && !clusters_ok(out)) return TPX3_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  Ws w = carve(p, workspace);
  if (p->profiling) ++p->profiled_calls;
  const bool lm_fused = !(p->cfg.flags & TPX3_FLAG_FORCE_GENERAL) && p->fused.variant != 0 && wt < (1u << 24) && n != 0;
  TPX3_LAUNCH(p, k_ctrl_init, 1, 256, 0, st, w.ctrl, n, w.tiles, 0u, n_hits);
  if (n == 0) return cuda_ok(cudaGetLastError());
  GenArgs ga = make_gen_args(p, w, 0, n, x, y, toa, tot, perm, lmax, max_clusters, out, n_hits);
  ga.lm_wx = wx; ga.lm_wy = wy; ga.lm_wt = wt;
  // the general route runs the tile kernel too, behind its global sort (mode 6), when the plan has one
  ga.sorted_tiles = p->fused.variant != 0 && wt < (1u << 24) && ((uintptr_t)perm & 3u) == 0;
  // shot-contiguous streams: the fused tile kernel in its paper-literal mode (the time window takes the place
  // of the link window in the tile key); anything else: the general kernels, enqueued from the device
  if (lm_fused) {
    Params prm = p->prm;
    prm.n = n;
    prm.W = wt;
    bool launched = false;
    StageTimer timer(p, st, TPX3_STAGE_FUSED);
    FusedArgs fa;
    int rc = enqueue_fused(p->fused, (uint32_t)p->num_sms, &p->launches, w.ctrl, w.tiles, st, prm, x, y, toa, tot, perm, lmax, max_clusters,
                           *out, n_hits, (char*)workspace + p->off_keyA, &launched, &fa, 1u, wx > 255u ? 255u : wx,
                           wy > 255u ? 255u : wy);
    if (rc != TPX3_OK) return rc;
    if (launched) {
      k_fallback_dispatch<<<1, 1, 0, st>>>(ga, fa, fused_ladder(p->cfg.max_shot_hits), 0, 1);
      ++p->launches;
      return cuda_ok(cudaGetLastError());
    }
  }
  if (ga.sorted_tiles) {
    int rc = enqueue_general_sort(p, ga, st);
    if (rc != TPX3_OK) return rc;
    StageTimer timer(p, st, TPX3_STAGE_FUSED);
    Params prm = p->prm;
    prm.n = n;
    prm.W = wt;
    FusedArgs fa = make_fused_args(8192u, (uint32_t)p->num_sms, w.ctrl, w.tiles, prm, x, y, toa, tot, perm, lmax, max_clusters,
                                   *out, n_hits, (char*)workspace + p->off_keyA, 6u, wx > 255u ? 255u : wx,
                                   wy > 255u ? 255u : wy, nullptr);
    fused_rebase_mode5(fa, 0u, 6u);
    k_fused_shot_tiles<8192, 1024, 6><<<fa.nseg, 1024, FusedSmem<8192>::kBytes, st>>>(fa);
    uint32_t ctas, tpc;
    compact_grid(fa.num_tiles, (uint32_t)p->num_sms, &ctas, &tpc);
    k_fused_compact<<<ctas, kCompactThreads, 0, st>>>(fa, tpc, 8192u);
    k_general_slab<<<1, 1, 0, st>>>(ga, 1);     // the window-walk kernels, only if a shot did not fit a window
    p->launches += 3;
    return cuda_ok(cudaGetLastError());
  }
  return enqueue_localmax(p, ga, st);
}

int tpx3_unwrap_toa(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint64_t* raw,
                    uint64_t modulus, uint64_t jump, int64_t wraps_in, int has_prev, uint64_t prev_raw,
                    uint64_t* toa_out, int64_t* wraps_out) {
  if (!p || !workspace || !wraps_out || modulus == 0) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (n && (!raw || !toa_out)) return TPX3_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  Ws w = carve(p, workspace);
  UnwrapArgs a;
  a.n = n; a.raw = raw; a.modulus = modulus; a.jump = jump; a.wraps_in = (long long)wraps_in;
  a.has_prev = has_prev; a.prev_raw = prev_raw; a.out = toa_out; a.wraps_out = (long long*)wraps_out;
  a.blk = w.counts;   // the sort's digit counters: 4 * 256 * 1184 bytes >= 4 * (2^28 / 4096 + 1)
  a.nblk = (uint32_t)((n + kUnwrapTile - 1) / kUnwrapTile);
  if (a.nblk) TPX3_LAUNCH(p, k_unwrap_count, a.nblk, kUnwrapThreads, 0, st, a);
  TPX3_LAUNCH(p, k_unwrap_scan, 1, 1024, 0, st, a);
  if (a.nblk) TPX3_LAUNCH(p, k_unwrap_apply, a.nblk, kUnwrapThreads, 0, st, a);
  return cuda_ok(cudaGetLastError());
}

// ---- tpx3_unwrap_toa without any allocation: scratch in a file-scope device array (tpx3.h) ---------------------
// One 32-bit block count per kUnwrapTile events, for n <= TPX3_STATIC_UNWRAP_MAX. In host code the NAME of the
// array is a host-side stand-in, not a device address: the kernels get the address cudaGetSymbolAddress returns,
// looked up once per device with that device current.
namespace {
constexpr uint32_t kStaticUnwrapBlocks = (uint32_t)(TPX3_STATIC_UNWRAP_MAX / kUnwrapTile);   // 16384 counts = 64 KB
static __device__ __align__(256) uint32_t g_static_unwrap_blk[kStaticUnwrapBlocks];
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
uint32_t* g_static_unwrap_ptr[kStaticMaxDevices];   // device address of the array on device d (null: not looked up yet)
}  // namespace

int tpx3_unwrap_toa_static(int device, void* cuda_stream, uint64_t n, const uint64_t* raw, uint64_t modulus,
                           uint64_t jump, int64_t wraps_in, int has_prev, uint64_t prev_raw, uint64_t* toa_out,
                           int64_t* wraps_out) {
  if (device < 0 || device >= kStaticMaxDevices || !wraps_out || modulus == 0) return TPX3_ERR_INVALID_ARG;
  if (n > TPX3_STATIC_UNWRAP_MAX) return TPX3_ERR_TOO_LARGE;
  if (n && (!raw || !toa_out)) return TPX3_ERR_INVALID_ARG;
  if (cudaSetDevice(device) != cudaSuccess) return TPX3_ERR_CUDA;
  uint32_t* blk = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_unwrap_ptr[device]) {
      void* ptr = nullptr;
      if (cudaGetSymbolAddress(&ptr, g_static_unwrap_blk) != cudaSuccess || !ptr) return TPX3_ERR_CUDA;
      g_static_unwrap_ptr[device] = (uint32_t*)ptr;
    }
    blk = g_static_unwrap_ptr[device];
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  UnwrapArgs a;
  a.n = n; a.raw = raw; a.modulus = modulus; a.jump = jump; a.wraps_in = (long long)wraps_in;
  a.has_prev = has_prev; a.prev_raw = prev_raw; a.out = toa_out; a.wraps_out = (long long*)wraps_out;
  a.blk = blk;
  a.nblk = (uint32_t)((n + kUnwrapTile - 1) / kUnwrapTile);     // <= kStaticUnwrapBlocks
  // every count the scan and the apply kernel read is written by the count kernel of THIS call: nothing to clear
  if (a.nblk) k_unwrap_count<<<a.nblk, kUnwrapThreads, 0, st>>>(a);
  k_unwrap_scan<<<1, 1024, 0, st>>>(a);
  if (a.nblk) k_unwrap_apply<<<a.nblk, kUnwrapThreads, 0, st>>>(a);
  return cuda_ok(cudaGetLastError());
}

int tpx3_timewalk_table(double a, double b, double c, double d, uint32_t length, int32_t* table_host) {
  if (!table_host && length) return TPX3_ERR_INVALID_ARG;
  for (uint32_t tot = 0; tot < length; ++tot) {
    const double base = (double)tot + b;
    const double v = base > 0.0 ? a / std::pow(base, d) + c : c;   // Eq. 1
    const double r = std::floor(std::fabs(v) + 0.5);                // nearest tick, half away from zero
    table_host[tot] = (int32_t)(v >= 0.0 ? r : -r);
  }
  return TPX3_OK;
}

int tpx3_preprocess(tpx3_plan_t p, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                    const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint64_t n_trig,
                    const uint64_t* trig, uint64_t cut, const int32_t* table, uint32_t table_len, uint64_t shot_base,
                    uint16_t* x_out, uint16_t* y_out, uint64_t* toa_out, uint16_t* tot_out, uint32_t* index_out,
                    uint32_t* n_out) {
  if (!p || !workspace || !n_out) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits || p->cfg.shot_period_ticks == 0 || (cut >> 63) != 0) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot || !x_out || !y_out || !toa_out || !tot_out)) return TPX3_ERR_INVALID_ARG;
  if ((n_trig && !trig) || (table_len && !table)) return TPX3_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  Ws w = carve(p, workspace);
  PreArgs a;
  a.n = n; a.x = x; a.y = y; a.tot = tot; a.toa = toa; a.n_trig = n_trig; a.trig = trig; a.cut = cut;
  a.P = p->cfg.shot_period_ticks; a.shot_base = shot_base; a.table = table; a.table_len = table_len;
  a.x_out = x_out; a.y_out = y_out; a.tot_out = tot_out; a.toa_out = toa_out; a.index_out = index_out;
  a.n_out = n_out;
  a.blk = w.counts;     // the sort's digit counters: room for 2^28 / 4096 block counts
  a.nblk = (uint32_t)((n + kPreTile - 1) / kPreTile);
  if (a.nblk) TPX3_LAUNCH(p, k_pre_mark, a.nblk, kPreThreads, 0, st, a);
  TPX3_LAUNCH(p, k_pre_scan, 1, 1024, 0, st, a);
  if (a.nblk) TPX3_LAUNCH(p, k_pre_scatter, a.nblk, kPreThreads, 0, st, a);
  return cuda_ok(cudaGetLastError());
}

// ---- chunked stream (tpx3_stream.cuh) ------------------------------------------------------------
struct tpx3_stream_s {
  tpx3_plan_t plan;
  uint64_t max_chunk, max_carry, disorder;
  int bank;                  // which carry bank holds the carried events
  bool failed;
  bool ended;                // a final push went through: the stream takes no more events
  tpx3::StreamCtrl* ctrl;
  uint16_t *cx[2], *cy[2], *ctot[2];
  uint64_t* ctoa[2];
  uint16_t *wx, *wy, *wtot;
  uint64_t* wtoa;
  uint32_t *wperm, *wlabel, *blk_emit, *blk_keep;
};

namespace {
struct StreamLayout {
  size_t ctrl, cx[2], cy[2], ctot[2], ctoa[2], wx, wy, wtot, wtoa, wperm, wlabel, blk_emit, blk_keep, total;
};
StreamLayout stream_layout(uint64_t max_chunk, uint64_t max_carry) {
  StreamLayout l;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes); return r; };
  const uint64_t m = max_chunk + max_carry;
  l.ctrl = take(sizeof(tpx3::StreamCtrl));
  for (int b = 0; b < 2; ++b) {
    l.cx[b] = take(2 * max_carry); l.cy[b] = take(2 * max_carry); l.ctot[b] = take(2 * max_carry);
    l.ctoa[b] = take(8 * max_carry);
  }
  l.wx = take(2 * m); l.wy = take(2 * m); l.wtot = take(2 * m); l.wtoa = take(8 * m);
  l.wperm = take(4 * m); l.wlabel = take(4 * m);
  const size_t nblk = (size_t)((m + tpx3::kStreamTile - 1) / tpx3::kStreamTile) + 1;
  l.blk_emit = take(4 * nblk); l.blk_keep = take(4 * nblk);
  l.total = o;
  return l;
}
}  // namespace

size_t tpx3_stream_bytes(uint64_t max_chunk, uint64_t max_carry) { return stream_layout(max_chunk, max_carry).total; }

int tpx3_stream_open(tpx3_plan_t p, void* stream_buf, uint64_t max_chunk, uint64_t max_carry, uint64_t disorder_ticks,
                     void* cuda_stream, tpx3_stream_t* out) {
  if (!p || !stream_buf || !out) return TPX3_ERR_INVALID_ARG;
  if (p->cfg.shot_period_ticks == 0 || max_chunk == 0 || max_carry == 0) return TPX3_ERR_INVALID_ARG;
  if (max_chunk + max_carry > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  tpx3_stream_s* s = new (std::nothrow) tpx3_stream_s();
  if (!s) return TPX3_ERR_CUDA;
  const StreamLayout l = stream_layout(max_chunk, max_carry);
  char* b = (char*)stream_buf;
  s->plan = p; s->max_chunk = max_chunk; s->max_carry = max_carry; s->disorder = disorder_ticks;
  s->bank = 0; s->failed = false; s->ended = false;
  s->ctrl = (tpx3::StreamCtrl*)(b + l.ctrl);
  for (int k = 0; k < 2; ++k) {
    s->cx[k] = (uint16_t*)(b + l.cx[k]); s->cy[k] = (uint16_t*)(b + l.cy[k]); s->ctot[k] = (uint16_t*)(b + l.ctot[k]);
    s->ctoa[k] = (uint64_t*)(b + l.ctoa[k]);
  }
  s->wx = (uint16_t*)(b + l.wx); s->wy = (uint16_t*)(b + l.wy); s->wtot = (uint16_t*)(b + l.wtot);
  s->wtoa = (uint64_t*)(b + l.wtoa); s->wperm = (uint32_t*)(b + l.wperm); s->wlabel = (uint32_t*)(b + l.wlabel);
  s->blk_emit = (uint32_t*)(b + l.blk_emit); s->blk_keep = (uint32_t*)(b + l.blk_keep);
  TPX3_LAUNCH(p, tpx3::k_stream_open, 1, 256, 0, (cudaStream_t)cuda_stream, s->ctrl);
  if (cudaGetLastError() != cudaSuccess) { delete s; return TPX3_ERR_CUDA; }
  *out = s;
  return TPX3_OK;
}

int tpx3_stream_push(tpx3_stream_t s, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                     const uint16_t* y, const uint64_t* toa, const uint16_t* tot, int final_push, uint64_t max_clusters,
                     const tpx3_clusters_t* out, uint32_t* n_hits, tpx3_stream_info_t* info) {
  if (!s || !workspace || !out || !n_hits) return TPX3_ERR_INVALID_ARG;
  if (s->failed) return TPX3_ERR_CAPACITY;
  if (s->ended || n > s->max_chunk) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot)) return TPX3_ERR_INVALID_ARG;
  if (max_clusters && !clusters_ok(out)) return TPX3_ERR_INVALID_ARG;
  tpx3_plan_t p = s->plan;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  tpx3::StreamArgs a;
  a.c = s->ctrl; a.n = n; a.carry_cap = (uint32_t)s->max_carry;
  a.x = x; a.y = y; a.tot = tot; a.toa = toa;
  const int in = s->bank, ob = s->bank ^ 1;
  a.cx = s->cx[in]; a.cy = s->cy[in]; a.ctot = s->ctot[in]; a.ctoa = s->ctoa[in];
  a.nx = s->cx[ob]; a.ny = s->cy[ob]; a.ntot = s->ctot[ob]; a.ntoa = s->ctoa[ob];
  a.wx = s->wx; a.wy = s->wy; a.wtot = s->wtot; a.wtoa = s->wtoa;
  a.blk_emit = s->blk_emit; a.blk_keep = s->blk_keep;
  // the number of carried events is device state: the grids cover the largest it can be (blocks past the end
  // of carried ++ chunk count nothing and return)
  a.nblk = (uint32_t)((n + s->max_carry + tpx3::kStreamTile - 1) / tpx3::kStreamTile);
  a.P = p->cfg.shot_period_ticks; a.D = s->disorder; a.final_push = final_push ? 1 : 0;
  TPX3_LAUNCH(p, tpx3::k_stream_cut, n ? 64 : 1, 256, 0, st, a);
  TPX3_LAUNCH(p, tpx3::k_stream_mark, a.nblk, tpx3::kStreamThreads, 0, st, a);
  TPX3_LAUNCH(p, tpx3::k_stream_scan, 1, 1024, 0, st, a);
  TPX3_LAUNCH(p, tpx3::k_stream_scatter, a.nblk, tpx3::kStreamThreads, 0, st, a);
  s->bank = ob;
  // clustering of the emit arrays: enqueued now with grids for the largest emit count; the kernels read the true
  // count (and the label offset) from the stream state
  {
    const int rc = run_fused_or_general(p, workspace, cuda_stream, n + s->max_carry, s->wx, s->wy, s->wtoa, s->wtot,
                                        s->wperm, s->wlabel, max_clusters, out, n_hits, 0u, s->ctrl);
    if (rc != TPX3_OK) return rc;
  }
  if (cudaGetLastError() != cudaSuccess) return TPX3_ERR_CUDA;
  if (final_push) s->ended = true;
  if (!info) return TPX3_OK;            // fully asynchronous: a carry overflow shows in tpx3_status (TPX3_ERR_CAPACITY)
  tpx3::StreamCtrl h;
  if (cudaMemcpyAsync(&h, s->ctrl, sizeof(h), cudaMemcpyDeviceToHost, st) != cudaSuccess) return TPX3_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return TPX3_ERR_CUDA;
  info->n_emitted = h.n_work; info->n_carry = h.n_carry; info->n_late = h.n_late; info->late_total = h.late_total;
  info->label_base = h.label_base; info->shots_emitted = h.final_push ? h.s_emitted : h.s_cut;
  if (h.dead) { s->failed = true; return TPX3_ERR_CAPACITY; }
  return TPX3_OK;
}

int tpx3_stream_close(tpx3_stream_t s) {
  if (!s) return TPX3_ERR_INVALID_ARG;
  delete s;
  return TPX3_OK;
}

// ---- end to end with host buffers ------------------------------------------------------------------
namespace {
// Large calls are pipelined: the input goes up in chunks on a copy stream, every chunk is pushed through the
// stream calls above as soon as it has landed (cut anywhere: open shots are carried), and the hit rows of
// push j go back on a second copy stream while chunk j+1 is still on its way up.
constexpr uint64_t kPipeChunk = 1ull << 22, kPipeCarry = 1ull << 20;
inline bool pipe_sized(uint64_t n) { return n >= 2 * kPipeChunk; }

struct HostIo {
  uint16_t *x, *y, *tot;
  uint64_t* toa;
  uint32_t *perm, *label, *n;
  tpx3_clusters_t d;          // the whole table (monolithic path)
  tpx3_clusters_t bank[2];    // per-push tables (pipelined path)
  uint32_t* bank_n[2];
  void* stream_buf;
  size_t total;
};

struct Carver {
  char* b;
  size_t o;
  char* operator()(size_t bytes) {   // b == nullptr: sizes only
    char* r = b ? b + o : nullptr;
    o = align_up(o + bytes);
    return r;
  }
};

tpx3_clusters_t carve_clusters(Carver& take, uint64_t cap) {
  tpx3_clusters_t d;
  d.label = (uint32_t*)take(4 * cap);
  d.size = (uint32_t*)take(4 * cap);
  d.shot = (uint32_t*)take(4 * cap);
  d.sum_tot = (int64_t*)take(8 * cap);
  d.sum_tot_x = (int64_t*)take(8 * cap);
  d.sum_tot_y = (int64_t*)take(8 * cap);
  d.toa_peak = (uint64_t*)take(8 * cap);
  d.cx = (float*)take(4 * cap);
  d.cy = (float*)take(4 * cap);
  d.sum_tot_tof = (int64_t*)take(8 * cap);
  d.ctof = (float*)take(4 * cap);
  return d;
}

HostIo host_io_layout(char* b, uint64_t n, uint64_t max_clusters) {
  HostIo io;
  Carver take{b, 0};
  io.x = (uint16_t*)take(2 * n);
  io.y = (uint16_t*)take(2 * n);
  io.toa = (uint64_t*)take(8 * n);
  io.tot = (uint16_t*)take(2 * n);
  io.perm = (uint32_t*)take(4 * n);
  io.label = (uint32_t*)take(4 * n);
  io.d = carve_clusters(take, max_clusters);
  io.n = (uint32_t*)take(256);
  io.stream_buf = nullptr;
  if (pipe_sized(n)) {
    for (int k = 0; k < 2; ++k) {
      io.bank[k] = carve_clusters(take, kPipeChunk + kPipeCarry);
      io.bank_n[k] = (uint32_t*)take(256);
    }
    io.stream_buf = take(tpx3_stream_bytes(kPipeChunk, kPipeCarry));
  }
  io.total = take.o;
  return io;
}

// D2H of `cnt` rows of table `d` into the host table `h` at row `at` (columns the caller left NULL are skipped).
cudaError_t copy_rows(const tpx3_clusters_t& h, uint64_t at, const tpx3_clusters_t& d, uint64_t cnt, cudaStream_t st) {
  cudaError_t e = cudaSuccess;
  if (!cnt) return e;
#define TPX3_ROWS(field, bytes)                                                                            \
  if (e == cudaSuccess && h.field)                                                                          \
    e = cudaMemcpyAsync(h.field + at, d.field, (bytes) * cnt, cudaMemcpyDeviceToHost, st);
  TPX3_ROWS(label, 4) TPX3_ROWS(size, 4) TPX3_ROWS(shot, 4) TPX3_ROWS(sum_tot, 8) TPX3_ROWS(sum_tot_x, 8)
  TPX3_ROWS(sum_tot_y, 8) TPX3_ROWS(toa_peak, 8) TPX3_ROWS(cx, 4) TPX3_ROWS(cy, 4) TPX3_ROWS(sum_tot_tof, 8)
  TPX3_ROWS(ctof, 4)
#undef TPX3_ROWS
  return e;
}

// Returns TPX3_OK with *fell_back = false when the pipelined run produced the result; *fell_back = true when
// the stream did not keep its promise (late events, carry overflow): all inputs are on the device by then and
// the caller runs the monolithic call on them.
int process_host_pipelined(tpx3_plan_t p, void* workspace, const HostIo& io, cudaStream_t st, uint64_t n,
                           const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                           uint64_t max_clusters, const tpx3_clusters_t* out_host, uint32_t* n_clusters_host,
                           bool* fell_back) {
  *fell_back = true;
  const uint32_t nchunk = (uint32_t)((n + kPipeChunk - 1) / kPipeChunk);
  std::vector<cudaEvent_t> ev(3 * (size_t)nchunk + 1, nullptr);   // [0] entry, then in / done / out per chunk
  std::vector<uint32_t> nh(nchunk, 0);
  tpx3_stream_t sh = nullptr;
  int rc = TPX3_ERR_CUDA;
  bool ok = (p->copy_in || cudaStreamCreateWithFlags(&p->copy_in, cudaStreamNonBlocking) == cudaSuccess) &&
            (p->copy_out || cudaStreamCreateWithFlags(&p->copy_out, cudaStreamNonBlocking) == cudaSuccess);
  cudaStream_t s_in = p->copy_in, s_out = p->copy_out;
  for (size_t i = 0; ok && i < ev.size(); ++i) ok = cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming) == cudaSuccess;
  auto e_in = [&](uint32_t j) { return ev[1 + 3 * (size_t)j]; };
  auto e_done = [&](uint32_t j) { return ev[2 + 3 * (size_t)j]; };
  auto e_out = [&](uint32_t j) { return ev[3 + 3 * (size_t)j]; };
  uint64_t rows = 0, total = 0;
  bool promise_kept = true;
  if (ok) {
    // the copies may not overtake earlier work of the caller's stream on the same buffers
    ok = cudaEventRecord(ev[0], st) == cudaSuccess && cudaStreamWaitEvent(s_in, ev[0], 0) == cudaSuccess &&
         cudaStreamWaitEvent(s_out, ev[0], 0) == cudaSuccess;
    for (uint32_t j = 0; ok && j < nchunk; ++j) {
      const uint64_t a = (uint64_t)j * kPipeChunk, m = (a + kPipeChunk <= n ? kPipeChunk : n - a);
      ok = cudaMemcpyAsync(io.toa + a, toa + a, 8 * m, cudaMemcpyHostToDevice, s_in) == cudaSuccess &&
           cudaMemcpyAsync(io.x + a, x + a, 2 * m, cudaMemcpyHostToDevice, s_in) == cudaSuccess &&
           cudaMemcpyAsync(io.y + a, y + a, 2 * m, cudaMemcpyHostToDevice, s_in) == cudaSuccess &&
           cudaMemcpyAsync(io.tot + a, tot + a, 2 * m, cudaMemcpyHostToDevice, s_in) == cudaSuccess &&
           cudaEventRecord(e_in(j), s_in) == cudaSuccess;
    }
  }
  if (ok) {
    // D = half a shot period: right for any stream whose pixels arrive less than half a period late; a stream
    // that is worse shows late events and is redone in one piece
    rc = tpx3_stream_open(p, io.stream_buf, kPipeChunk, kPipeCarry, p->cfg.shot_period_ticks / 2, st, &sh);
    ok = rc == TPX3_OK;
  }
  auto rows_back = [&](uint32_t j) {   // after the stream has been synchronised past push j's count
    uint64_t cnt = nh[j];
    total += cnt;
    if (rows + cnt > max_clusters) cnt = max_clusters > rows ? max_clusters - rows : 0;
    bool good = cudaStreamWaitEvent(s_out, e_done(j), 0) == cudaSuccess;
    if (good && out_host) good = copy_rows(*out_host, rows, io.bank[j & 1], cnt, s_out) == cudaSuccess;
    rows += cnt;
    return good && cudaEventRecord(e_out(j), s_out) == cudaSuccess;
  };
  for (uint32_t j = 0; ok && promise_kept && j < nchunk; ++j) {
    const uint64_t a = (uint64_t)j * kPipeChunk, m = (a + kPipeChunk <= n ? kPipeChunk : n - a);
    ok = cudaStreamWaitEvent(st, e_in(j), 0) == cudaSuccess;
    if (ok && j >= 2) ok = cudaStreamWaitEvent(st, e_out(j - 2), 0) == cudaSuccess;   // bank j & 1 is free again
    if (!ok) break;
    tpx3_stream_info_t info;
    rc = tpx3_stream_push(sh, workspace, st, m, io.x + a, io.y + a, io.toa + a, io.tot + a, j + 1 == nchunk,
                          kPipeChunk + kPipeCarry, &io.bank[j & 1], io.bank_n[j & 1], &info);
    if (rc == TPX3_ERR_CAPACITY || (rc == TPX3_OK && info.late_total)) { promise_kept = false; rc = TPX3_OK; break; }
    ok = rc == TPX3_OK;
    if (!ok) break;
    // the push synchronised the stream behind push j-1's clustering: its count is on the host now
    if (j >= 1) ok = rows_back(j - 1);
    ok = ok && cudaMemcpyAsync(&nh[j], io.bank_n[j & 1], 4, cudaMemcpyDeviceToHost, st) == cudaSuccess &&
         cudaEventRecord(e_done(j), st) == cudaSuccess;
  }
  if (ok && promise_kept) {
    ok = cudaStreamSynchronize(st) == cudaSuccess && rows_back(nchunk - 1) && cudaStreamSynchronize(s_out) == cudaSuccess;
    if (ok) {
      *n_clusters_host = (uint32_t)total;
      *fell_back = false;
      rc = total > max_clusters ? TPX3_ERR_CAPACITY : TPX3_OK;
    }
  }
  // leave nothing in flight: the fallback (and the caller) reuse the buffers
  if (s_in) cudaStreamSynchronize(s_in);
  if (s_out) cudaStreamSynchronize(s_out);
  cudaStreamSynchronize(st);
  if (sh) tpx3_stream_close(sh);
  for (auto e : ev) if (e) cudaEventDestroy(e);
  if (!ok) return rc != TPX3_OK ? rc : TPX3_ERR_CUDA;
  return rc;
}
}  // namespace

size_t tpx3_host_io_bytes(uint64_t n, uint64_t max_clusters) { return host_io_layout(nullptr, n, max_clusters).total; }

int tpx3_process_host(tpx3_plan_t p, void* workspace, void* device_io, void* cuda_stream, uint64_t n, const uint16_t* x,
                      const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint32_t* perm, uint32_t* label,
                      uint64_t max_clusters, const tpx3_clusters_t* out_host, uint32_t* n_clusters_host) {
  if (!p || !workspace || !device_io || !n_clusters_host) return TPX3_ERR_INVALID_ARG;
  if (n > p->cfg.max_hits) return TPX3_ERR_INVALID_ARG;
  if (n && (!x || !y || !toa || !tot)) return TPX3_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  const HostIo io = host_io_layout((char*)device_io, n, max_clusters);
  cudaError_t e = cudaSuccess;
  bool resident = false;
  if (pipe_sized(n) && p->cfg.shot_period_ticks && !perm && !label && !(p->cfg.flags & TPX3_FLAG_VALIDATE_INPUT)) {
    bool fell_back = true;
    const int rc = process_host_pipelined(p, workspace, io, st, n, x, y, toa, tot, max_clusters, out_host,
                                          n_clusters_host, &fell_back);
    p->host_route = fell_back ? 2 : 1;
    if (!fell_back || (rc != TPX3_OK && rc != TPX3_ERR_CAPACITY)) return rc;
    resident = true;   // every chunk went up before the stream gave up
  } else {
    p->host_route = 0;
  }
  if (n && !resident) {
    e = cudaMemcpyAsync(io.x, x, 2 * n, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(io.y, y, 2 * n, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(io.toa, toa, 8 * n, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(io.tot, tot, 2 * n, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return TPX3_ERR_CUDA;
  }
  int rc = tpx3_cluster_centroid(p, workspace, cuda_stream, n, io.x, io.y, io.toa, io.tot, io.perm, io.label,
                                 max_clusters, &io.d, io.n);
  if (rc != TPX3_OK) return rc;
  e = cudaMemcpyAsync(n_clusters_host, io.n, 4, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && perm && n) e = cudaMemcpyAsync(perm, io.perm, 4 * n, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && label && n) e = cudaMemcpyAsync(label, io.label, 4 * n, cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return TPX3_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return TPX3_ERR_CUDA;  // the count decides the copy sizes
  uint64_t nc = *n_clusters_host;
  if (nc > max_clusters) nc = max_clusters;
  if (out_host && copy_rows(*out_host, 0, io.d, nc, st) != cudaSuccess) return TPX3_ERR_CUDA;
  tpx3_status_t s;
  rc = tpx3_status(p, workspace, cuda_stream, &s);
  if (rc != TPX3_OK) return rc;
  return s.error ? -(int)s.error : TPX3_OK;
}

int tpx3_host_route(tpx3_plan_t p) { return p ? p->host_route : TPX3_ERR_INVALID_ARG; }

int tpx3_status(tpx3_plan_t p, const void* workspace, void* cuda_stream, tpx3_status_t* out) {
  if (!p || !workspace || !out) return TPX3_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  if (cudaMemcpyAsync(out, workspace, sizeof(tpx3_status_t), cudaMemcpyDeviceToHost, st) != cudaSuccess)
    return TPX3_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return TPX3_ERR_CUDA;
  return TPX3_OK;
}

uint64_t tpx3_launch_count(tpx3_plan_t p) { return p ? p->launches : 0; }

int tpx3_profile_enable(tpx3_plan_t p, int enable) {
  if (!p) return TPX3_ERR_INVALID_ARG;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  p->profiling = enable != 0;
  return TPX3_OK;
}

int tpx3_profile_read(tpx3_plan_t p, tpx3_profile_t* out) {
  if (!p || !out) return TPX3_ERR_INVALID_ARG;
  if (use_device(p) != TPX3_OK) return TPX3_ERR_CUDA;
  memset(out, 0, sizeof(*out));
  int rc = TPX3_OK;
  for (auto& s : p->spans) {
    float ms = 0.f;
    if (cudaEventSynchronize(s.b) != cudaSuccess || cudaEventElapsedTime(&ms, s.a, s.b) != cudaSuccess) rc = TPX3_ERR_CUDA;
    out->ms[s.stage] += ms;
    out->launches[s.stage] += s.launches1 - s.launches0;
    p->free_events.push_back(s.a);
    p->free_events.push_back(s.b);
  }
  p->spans.clear();
  out->calls = p->profiled_calls;
  p->profiled_calls = 0;
  return rc;
}

int tpx3_free(tpx3_plan_t p) {
  if (!p) return TPX3_ERR_INVALID_ARG;
  for (auto& s : p->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
  for (auto e : p->free_events) cudaEventDestroy(e);
  if (p->copy_in) cudaStreamDestroy(p->copy_in);
  if (p->copy_out) cudaStreamDestroy(p->copy_out);
  delete p;
  return TPX3_OK;
}

const char* tpx3_strerror(int err) {
  switch (err) {
    case TPX3_OK: return "ok";
    case TPX3_ERR_INVALID_ARG: return "invalid argument";
    case TPX3_ERR_CAPACITY: return "max_clusters too small";
    case TPX3_ERR_OUT_OF_RANGE: return "event outside the sensor or ToT == 0";
    case TPX3_ERR_CUDA: return "CUDA runtime error";
    case TPX3_ERR_TOO_LARGE: return "n beyond the fixed scratch of the no-allocation entry point (TPX3_STATIC_UNWRAP_MAX)";
    case TPX3_ERR_NOT_CONTIGUOUS: return "stream not shot-contiguous or a shot longer than the window (fused preprocessing call)";
    default: return "unknown error";
  }
}

}  // extern "C"
