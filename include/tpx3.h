/* tpx3.h — C ABI of the B200-native TimePix3 cluster + centroid hot path.
 *
 * What the library computes (arxiv/paper_2603_04942, cited as PAPER.md:<line>):
 *   input   a stream of pixel events (X, Y, ToA, ToT) from a TimePix3 sensor
 *   S0/S1   shot = ToA div P (most recent laser trigger); stable sort of the
 *           events by (shot, ToA) (the stream is "essentially unsorted")
 *   S2      neighbourhood relation A = A^X (.) A^Y (.) A^ToF, |D| <= w inclusive    PAPER.md:117-126, Eq. 4-5
 *           with w_x = w_y = 1 (8-connectivity), w_t = W ticks, same shot only; a particle hit
 *           is a connected component of that relation (BASELINE.json north_star)
 *   S3      label[k] = smallest sorted index in k's component; hit count
 *   S4      per hit: size, sum ToT, sum ToT*X, sum ToT*Y (exact integers); the brightest pixel
 *           (max ToT, ties: the later pixel in the sorted stream wins)
 *   S5      centroid = sum(ToT*X) / sum(ToT), same for Y and for ToF = ToA - shot*P  PAPER.md:156-165, Eq. 8-9
 *           computed as fp32(int64) / fp32(int64), IEEE round-to-nearest divide.
 *
 * Conventions
 *   - Every pointer marked [dev] is device memory on the plan's CUDA device, owned by the
 *     caller (the Python binding passes PyTorch tensors); [host] is host memory. The library
 *     never frees or reallocates caller memory and never writes its inputs.
 *   - `workspace` is a [dev] scratch buffer of at least the `workspace_bytes` reported by
 *     tpx3_plan, 256-byte aligned. Its contents are undefined between calls and need no
 *     initialisation (one word of the control block is a performance hint that is kept from
 *     call to call when the same workspace is reused; it never changes a result).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Device-pointer calls only ENQUEUE work on that stream and return; there is no hidden
 *     synchronisation. Outputs are valid once the stream has reached the end of the call.
 *   - Alignment: every array at the natural alignment of its element type. The fast path reads with 128-bit loads;
 *     x, y, toa, tot that start at the same element offset from a 16-byte boundary - a chunk of a resident
 *     stream cut at any event, arrays offset alike - are served by it all the same (the library reads up to 7
 *     elements in front of the pointers inside the same 16-byte block and ignores them); arrays that are not
 *     offset alike take the general route (same results, slower).
 *   - `perm[k]`  = original (input) index of the event at sorted position k.
 *     `label[k]` = sorted position of the first event of k's hit; indexed by SORTED position.
 *     Clusters are listed in ascending `label` order (exactly one valid output exists).
 *   - Preconditions on the data: x < sensor_w, y < sensor_h, tot >= 1. They are only checked
 *     under TPX3_FLAG_VALIDATE_INPUT (result in tpx3_status).
 *   - Errors: every call returns 0 (TPX3_OK) or a negative tpx3_error_t. Errors that can only
 *     be detected on the device (capacity, validation) are recorded in a device status word
 *     read by tpx3_status. No exceptions, no exit(), no output on stdout, no CPU fallback.
 */
#ifndef TPX3_H_
#define TPX3_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  TPX3_OK = 0,
  TPX3_ERR_INVALID_ARG = -1,   /* null pointer, bad struct_size, n > max_hits, bad config      */
  TPX3_ERR_CAPACITY = -2,      /* max_clusters too small (device-detected; see tpx3_status)     */
  TPX3_ERR_OUT_OF_RANGE = -3,  /* x/y outside the sensor or tot == 0 (under VALIDATE_INPUT)     */
  TPX3_ERR_CUDA = -4,          /* a CUDA runtime call failed                                    */
  TPX3_ERR_NOT_CONTIGUOUS = -5,/* tpx3_preprocess_cluster_centroid only (device-detected): the stream
                                  is not shot-contiguous or a shot does not fit the plan's window;
                                  use tpx3_preprocess followed by tpx3_cluster_centroid            */
  TPX3_ERR_TOO_LARGE = -6      /* tpx3_unwrap_toa_static only: n beyond TPX3_STATIC_UNWRAP_MAX, the
                                  size its fixed scratch array serves; use tpx3_unwrap_toa          */
} tpx3_error_t;

enum {
  TPX3_FLAG_VALIDATE_INPUT = 1u << 0, /* check the data preconditions on the device            */
  TPX3_FLAG_FORCE_GENERAL = 1u << 1   /* never take the shot-contiguous fused path              */
};

typedef struct tpx3_plan_s* tpx3_plan_t;

typedef struct {
  uint32_t struct_size;        /* = sizeof(tpx3_config_t); ABI guard                           */
  uint16_t sensor_w, sensor_h; /* pixels; 1..256 each (TimePix3: 256 x 256)       */
  uint32_t toa_window_ticks;   /* W: |dToA| <= W links, inclusive; < 2^31       */
  uint64_t shot_period_ticks;  /* P: shot = ToA div P; 0 = the whole input is one shot         */
  uint64_t max_hits;           /* largest n of any later call; 1 .. 2^28                       */
  int32_t device;              /* CUDA device ordinal                                          */
  uint32_t flags;              /* TPX3_FLAG_*                                                  */
  uint32_t max_shot_hits;      /* hint: most events one shot can hold; sizes the fused path's
                                  tile windows. <= 1536: 2048-event windows, 4 CTAs per SM;
                                  <= 3584: 4096 events, 2 CTAs per SM; <= 8184: 8192 events;
                                  larger, or a shot that does not fit the window: the general
                                  path runs (same results, slower). 0 = no hint: windows of
                                  2048, then 4096, then 8192 events are tried on the device (a
                                  failed try stops within its first wave of tiles), then the
                                  general path.                                                */
  uint32_t reserved;           /* must be 0                                                    */
} tpx3_config_t;

/* Per-hit (cluster) outputs, structure of arrays, each of capacity max_clusters. [dev] */
typedef struct {
  uint32_t* label;      /* sorted position of the hit's first pixel (ascending)                */
  uint32_t* size;       /* number of pixels                                                    */
  uint32_t* shot;       /* ToA div P of the hit, low 32 bits                                   */
  int64_t* sum_tot;     /* sum ToT                                                             */
  int64_t* sum_tot_x;   /* sum ToT * X                                                         */
  int64_t* sum_tot_y;   /* sum ToT * Y                                                         */
  uint64_t* toa_peak;   /* ToA of the brightest pixel (max (ToT, sorted position))             */
  float* cx;            /* fp32(sum_tot_x) / fp32(sum_tot), Eq. 9                              */
  float* cy;
  int64_t* sum_tot_tof; /* sum ToT * ToF, ToF = ToA - shot * P in ticks (P = 0: ToF = ToA); exact
                           while it stays below 2^63 (always for P <= 2^24)                    */
  float* ctof;          /* fp32(sum_tot_tof) / fp32(sum_tot): the ToF centroid, "identical for
                           X, Y and ToF", PAPER.md:165                                         */
} tpx3_clusters_t;

/* Device status of the most recent call on a workspace (tpx3_status). */
typedef struct {
  uint32_t error;       /* 0 or -(tpx3_error_t) of the first device-detected error             */
  uint32_t path;        /* 1 = fused shot-tile path, 2 = general path (global sort + hash link),
                           3 = paper-literal local-maximum mode                                 */
  uint32_t n_clusters;  /* hits found by the last cluster / centroid call                      */
  uint32_t sort_passes; /* radix passes the general path ran (0 on the fused path)             */
  uint64_t n;           /* events of the last call                                             */
} tpx3_status_t;

/* Validate `cfg`, create a plan (host metadata only) and report the device workspace size the
 * other calls need for up to cfg->max_hits events. Host only; no device memory is allocated. */
int tpx3_plan(const tpx3_config_t* cfg, tpx3_plan_t* out_plan, size_t* workspace_bytes);

/* S0-S3. x, y, tot: uint16[n]; toa: uint64[n] (all [dev], SoA, 14 B/event).
 * Outputs [dev]: perm uint32[n], label uint32[n], n_clusters uint32[1]. n may be 0. Runs where
 * tpx3_cluster_centroid runs (same kernel, stopped after the labels; same decision on the device). */
int tpx3_cluster(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n,
                 const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                 uint32_t* perm, uint32_t* label, uint32_t* n_clusters);

/* S4-S5 for ANY (perm, label) satisfying the post-conditions of tpx3_cluster (perm a
 * permutation; label[k] <= k; label[label[k]] == label[k]). Writes min(n_clusters,
 * max_clusters) entries of `out` and the true count to n_clusters [dev]; if the count exceeds
 * max_clusters the status word records TPX3_ERR_CAPACITY. (perm, label) whose hits each lie inside
 * one shot of a shot-contiguous order - what tpx3_cluster writes - are served by the tile kernel
 * (events read through perm, in the given order: "sorted position" in the tie rule means position in
 * perm); anything else by the general sums. Same results. */
int tpx3_centroid(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n,
                  const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                  const uint32_t* perm, const uint32_t* label, uint64_t max_clusters,
                  const tpx3_clusters_t* out, uint32_t* n_clusters);

/* S0-S5 in one call (same results as tpx3_cluster followed by tpx3_centroid). When the input
 * is shot-contiguous (shot = ToA div P never decreases along the stream, as in a TimePix3
 * readout where disorder is confined to one readout window) and every shot fits one
 * shared-memory tile, the whole path runs as ONE fused kernel; otherwise the general route
 * runs: a global radix sort by ToA, then the same tile kernel on the sorted stream, and only
 * for a shot longer than a tile (or a plan without a shot period) the slab-hash linking and
 * atomic sums. The decision is taken on the device; tpx3_status reports path 1 or 2. */
int tpx3_cluster_centroid(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n,
                          const uint16_t* x, const uint16_t* y, const uint64_t* toa,
                          const uint16_t* tot, uint32_t* perm, uint32_t* label,
                          uint64_t max_clusters, const tpx3_clusters_t* out, uint32_t* n_clusters);

/* Paper-literal mode (section V, Eq. 3-9): a hit is a pixel with no
 * neighbour of greater (ToT, sorted position) inside the box |dX| <= wx, |dY| <= wy, |dToF| <= wt
 * of the same shot (all inclusive; tie: the later pixel wins, :150); its centroid
 * is Eq. 9 over that box (row i of A, A_ii = 1) for X, Y and ToF alike (:165). Uses the plan's
 * shot period; the plan's toa_window_ticks is not used. Shot-contiguous streams run in the fused
 * tile kernel (as tpx3_cluster_centroid), anything else in the general kernels; same results.
 * Outputs [dev]: perm uint32[n]; lmax uint32[n], lmax[k] = k if sorted position k is a hit and
 * 0xFFFFFFFF otherwise; one row of `out` per hit in ascending k (label = k, size = pixels in the
 * box, toa_peak = ToA of the local maximum, sums and centroids over the box); n_hits uint32[1].
 * Capacity and errors as tpx3_centroid. tpx3_status reports path 3. */
int tpx3_localmax_centroid(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n,
                           const uint16_t* x, const uint16_t* y, const uint64_t* toa,
                           const uint16_t* tot, uint32_t wx, uint32_t wy, uint32_t wt, uint32_t* perm,
                           uint32_t* lmax, uint64_t max_clusters, const tpx3_clusters_t* out,
                           uint32_t* n_hits);

/* ToA counter unwrapping (section IV.A, :58-62), for the pixel stream
 * or the trigger (TDC) stream, each on its own. raw uint64[n] [dev]: counter values in
 * [0, modulus) in stream order; modulus: the counter period in the caller's tick (2^42 units of
 * 25/4096 ns for pixels, 2^44 for TDCs); jump: the "20 seconds" threshold in ticks.
 * Event k adds +1 to the wrap counter if raw[k-1] - raw[k] > jump (:60) and -1 if
 * raw[k] - raw[k-1] > jump (a pre-wrap event reported after the wrap, :62); toa_out[k] =
 * raw[k] + wraps_k * modulus (uint64[n] [dev], may not alias raw). wraps_in, has_prev, prev_raw
 * carry the counter and the last raw value of the previous call; wraps_out int64[1] [dev]
 * receives the counter after the last event. Enqueue only. */
int tpx3_unwrap_toa(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n, const uint64_t* raw,
                    uint64_t modulus, uint64_t jump, int64_t wraps_in, int has_prev, uint64_t prev_raw,
                    uint64_t* toa_out, int64_t* wraps_out);

/* The same unwrapping for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): no plan, no workspace. The scratch the three
 * kernels share (one 32-bit count per 4096 events) lives in a file-scope `static __device__` array of the
 * library, 64 KB, which every GPU that loads the library holds until the process exits; it serves
 * n <= TPX3_STATIC_UNWRAP_MAX events, a larger n returns TPX3_ERR_TOO_LARGE before anything is enqueued.
 * The call allocates nothing (no cudaMalloc / cudaFree, no allocating library routine): the array's device
 * address is looked up once per device (cudaGetSymbolAddress, with that device current) and kept.
 * `device` is the CUDA device ordinal of raw / toa_out / wraps_out and of cuda_stream. Arguments, results
 * and rounding are those of tpx3_unwrap_toa. ALL calls on a device share the one array: it keeps the last
 * call's contents (nothing in it has to start at zero: every call overwrites the counts it reads), and
 * two calls that overlap on the GPU (different streams, no ordering between them) race on it - keep them
 * on one stream or order them with events. Enqueue only. */
#define TPX3_STATIC_UNWRAP_MAX (1ull << 26)
int tpx3_unwrap_toa_static(int device, void* cuda_stream, uint64_t n, const uint64_t* raw, uint64_t modulus,
                           uint64_t jump, int64_t wraps_in, int has_prev, uint64_t prev_raw, uint64_t* toa_out,
                           int64_t* wraps_out);

/* Timewalk calibration product (Eq. 1): table_host[ToT] = a / (ToT + b)^d + c for
 * ToT = 0 .. length-1, evaluated in fp64 and rounded to the nearest integer tick (half away from
 * zero; ToT + b <= 0 gives c). a, c in ticks. Host only; table_host int32[length] [host]. */
int tpx3_timewalk_table(double a, double b, double c, double d, uint32_t length, int32_t* table_host);

/* Preprocessing (section IV.B-C, :66-76) of a pixel stream with
 * unwrapped ToA against the list of laser triggers trig uint64[n_trig] [dev], ascending. Per event:
 * s = the most recent trigger (largest s with trig[s] <= ToA; none: dropped), ToF = ToA - trig[s],
 * dropped if ToF > cut ("does not exceed 100 us", :68; cut < 2^63), ToF' = ToF - table[min(ToT, table_len-1)]
 * (int32[table_len] [dev], ticks; table_len = 0: no correction) clamped to [0, P - 1], ToA' =
 * (shot_base + s) * P + ToF' with P = the plan's shot_period_ticks (must be > 0), so that the
 * clustering calls see shot = ToA' div P = shot_base + s. Kept events are written in stream order
 * to x_out, y_out, toa_out, tot_out (capacity n each, [dev], no aliasing of the inputs) and their
 * input positions to index_out uint32[n] (may be NULL); n_out uint32[1] [dev]. Enqueue only. */
int tpx3_preprocess(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                    const uint16_t* y, const uint64_t* toa, const uint16_t* tot, uint64_t n_trig,
                    const uint64_t* trig, uint64_t cut, const int32_t* table, uint32_t table_len,
                    uint64_t shot_base, uint16_t* x_out, uint16_t* y_out, uint64_t* toa_out,
                    uint16_t* tot_out, uint32_t* index_out, uint32_t* n_out);

/* Preprocessing FUSED into the clustering call (SURVEY.md 8f NEXT #3 as worded: "fused into the key-build
 * pass"): same arguments and per-event rules as tpx3_preprocess (trigger assignment, ToF cut, timewalk table,
 * rebase), same hits as tpx3_preprocess followed by tpx3_cluster_centroid on its output, but the
 * intermediate stream is never written: a pre-pass counts the surviving events per segment (reads ToA and the
 * trigger list), and the tile kernel applies the preprocessing in its load phase, before it builds its keys.
 * Outputs [dev]: n_kept uint32[1] = events that survive; perm uint32[n] (first n_kept entries written): perm[k]
 * = INPUT position (into x, y, toa, tot) of the surviving event at sorted position k (the two-call route gives
 * index_out[perm[k]]); label uint32[n] (first n_kept entries), indexed by sorted position among the surviving
 * events; `out` / n_clusters as tpx3_cluster_centroid, with toa_peak and shot in the REBASED time
 * ((shot_base + s) * P + ToF'). Serves shot-contiguous raw streams (the trigger index never decreases along
 * the stream; an event before the first trigger counts to trigger 0 for this purpose) whose shots fit the
 * plan's window (max_shot_hits, counted on the raw stream, must be given); anything else is detected on the
 * device and reported as TPX3_ERR_NOT_CONTIGUOUS by tpx3_status - nothing valid has been written then. The
 * plan's shot period must be > 0 and <= 2^24; x, y, toa, tot must be 16-byte aligned (TPX3_ERR_INVALID_ARG otherwise: this
 * call has no general route to fall back to). Enqueue only. */
int tpx3_preprocess_cluster_centroid(tpx3_plan_t plan, void* workspace, void* cuda_stream, uint64_t n,
                                     const uint16_t* x, const uint16_t* y, const uint64_t* toa,
                                     const uint16_t* tot, uint64_t n_trig, const uint64_t* trig, uint64_t cut,
                                     const int32_t* table, uint32_t table_len, uint64_t shot_base,
                                     uint32_t* perm, uint32_t* label, uint64_t max_clusters,
                                     const tpx3_clusters_t* out, uint32_t* n_clusters, uint32_t* n_kept);

/* End-to-end variant with HOST buffers: copies x, y, toa, tot [host] to the device, runs
 * tpx3_cluster_centroid and copies perm, label (either may be NULL to skip), the first
 * min(n_clusters, max_clusters) entries of every non-NULL array of `out_host` and the count
 * back, then synchronises the stream. `device_io` is a [dev] staging buffer of at least
 * tpx3_host_io_bytes(n, max_clusters) bytes. Returns the device status error, if any.
 * Calls of n >= 2^23 events that ask for neither perm nor label (shot period > 0, no
 * TPX3_FLAG_VALIDATE_INPUT) are pipelined: the input goes up in 2^22-event chunks on a copy stream
 * of the library's own, each chunk is pushed through the stream calls below as it lands (disorder
 * bound: half a shot period), and the hit rows of a push go back on a second copy stream under
 * the next chunk's upload. Same rows as the one-piece route; a stream with late events or more
 * than 2^20 carried events is redone in one piece (tpx3_host_route tells which). */
size_t tpx3_host_io_bytes(uint64_t n, uint64_t max_clusters);
int tpx3_process_host(tpx3_plan_t plan, void* workspace, void* device_io, void* cuda_stream,
                      uint64_t n, const uint16_t* x, const uint16_t* y, const uint64_t* toa,
                      const uint16_t* tot, uint32_t* perm, uint32_t* label, uint64_t max_clusters,
                      const tpx3_clusters_t* out_host, uint32_t* n_clusters_host);

/* Synchronise `cuda_stream` and copy the workspace's status word to *out [host]. */
int tpx3_status(tpx3_plan_t plan, const void* workspace, void* cuda_stream, tpx3_status_t* out);

/* Chunked stream with cuts that are not shot-aligned (last clause; DESIGN.md
 * R24). An endless pixel stream arrives in chunks cut anywhere - inside a shot, inside a hit. Every
 * pixel belongs to "the most recent laser trigger" and no hit crosses a shot, so the
 * stream object holds back the events of shots that may still grow and clusters every shot in one
 * piece: the hit rows of all pushes, in order, are exactly the rows one tpx3_cluster_centroid call
 * on the whole stream would write (labels included: label = position in the (shot, ToA) order of
 * the whole stream, modulo 2^32).
 *   disorder_ticks  D: the stream promises that no event arrives with ToA < (largest ToA so far) - D
 *                   (0 = in ToA order; pixels report out of order, dimmer ones first).
 *   per push        t_max = max(t_max, ToA of the last 65536 events of the chunk); s_cut =
 *                   max(s_emitted, (t_max - D) div P); of the carried events followed by the chunk,
 *                   in stream order: shot < s_emitted: late (dropped, counted); shot < s_cut: emitted
 *                   = clustered now; the rest carried. final != 0 emits everything and ends the
 *                   stream: any later push returns TPX3_ERR_INVALID_ARG.
 *                   (What ONE push emits is not part of the definition: the tail sample is a lower bound of
 *                   the largest ToA, and any lower bound only emits a shot later. The rows of ALL pushes are.)
 * stream_buf [dev]: tpx3_stream_bytes(max_chunk, max_carry) bytes, caller-owned, holds the carried
 * events, the emitted events of the current push and the stream state; max_chunk + max_carry <=
 * the plan's max_hits; the plan's shot period must be > 0. tpx3_stream_open enqueues the reset of the
 * state on cuda_stream. tpx3_stream_push: x, y, toa, tot [dev] of n <= max_chunk events; out,
 * n_hits [dev] as tpx3_cluster_centroid; info [host] (may be NULL). The push SYNCHRONISES cuda_stream
 * once (the number of emitted events sizes the clustering launch); the clustering itself is only
 * enqueued. More than max_carry events to carry: TPX3_ERR_CAPACITY, and the stream is dead. Cluster
 * capacity and input errors are reported as by tpx3_cluster_centroid (tpx3_status). */
typedef struct tpx3_stream_s* tpx3_stream_t;
typedef struct {
  uint64_t n_emitted;     /* events clustered by this push                                  */
  uint64_t n_carry;       /* events held back for the next push                             */
  uint64_t n_late;        /* events of this push whose shot had gone out already (dropped)  */
  uint64_t late_total;    /* the same, since tpx3_stream_open                               */
  uint64_t label_base;    /* events emitted by earlier pushes (added to the label column)   */
  uint64_t shots_emitted; /* every shot below this index is complete and written            */
} tpx3_stream_info_t;
size_t tpx3_stream_bytes(uint64_t max_chunk, uint64_t max_carry);
int tpx3_stream_open(tpx3_plan_t plan, void* stream_buf, uint64_t max_chunk, uint64_t max_carry,
                     uint64_t disorder_ticks, void* cuda_stream, tpx3_stream_t* out);
int tpx3_stream_push(tpx3_stream_t stream, void* workspace, void* cuda_stream, uint64_t n, const uint16_t* x,
                     const uint16_t* y, const uint64_t* toa, const uint16_t* tot, int final_push,
                     uint64_t max_clusters, const tpx3_clusters_t* out, uint32_t* n_hits,
                     tpx3_stream_info_t* info);
int tpx3_stream_close(tpx3_stream_t stream);

/* Which route the last tpx3_process_host call of this plan took: 0 = one piece (copy in, one
 * clustering call, copy out), 1 = pipelined (see tpx3_process_host), 2 = the pipelined attempt met
 * late events or a carry overflow and the call was redone in one piece (same results). */
int tpx3_host_route(tpx3_plan_t plan);

/* Number of kernels the HOST has launched through this plan (for launch accounting). Kernels that the
 * library launches from the device (the next rung of the no-hint ladder, the general path after a fused
 * attempt that gave up: tpx3_status then reports path 2) are not in this count. */
uint64_t tpx3_launch_count(tpx3_plan_t plan);

/* Optional per-stage device timing. While enabled, every call brackets each stage it enqueues
 * with a pair of CUDA events recorded on the call's stream (no synchronisation at call time).
 * tpx3_profile_read waits for the recorded events, writes the summed durations since the last
 * read to *out [host] and recycles the events. Stages: */
enum {
  TPX3_STAGE_FUSED = 0,    /* the fused shot-tile kernel (S0-S5)                                */
  TPX3_STAGE_SORT = 1,     /* general path: min/max, radix passes                               */
  TPX3_STAGE_LINK = 2,     /* general path: gather, hash insert, link, compress                 */
  TPX3_STAGE_CENTROID = 3, /* general path / tpx3_centroid: root ordinals, sums, divide         */
  TPX3_STAGE_COUNT = 4
};
typedef struct {
  double ms[TPX3_STAGE_COUNT];         /* summed device time of the stage, milliseconds        */
  uint64_t launches[TPX3_STAGE_COUNT]; /* kernels launched inside the stage                     */
  uint64_t calls;                      /* API calls profiled                                    */
} tpx3_profile_t;
int tpx3_profile_enable(tpx3_plan_t plan, int enable);
int tpx3_profile_read(tpx3_plan_t plan, tpx3_profile_t* out);

int tpx3_free(tpx3_plan_t plan);
const char* tpx3_strerror(int err);

#ifdef __cplusplus
}
#endif
#endif /* TPX3_H_ */
