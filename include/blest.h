/* include/blest.h -- C ABI of the B200-native BLEST hot path (arXiv 2606.05081).
 *
 * Level-synchronous BFS as an iterated bit-level SpMSpV  x(k+1) = (A x(k)) AND NOT v(k)
 * (Eq. 1) over a Binarized Virtual Slice Set (BVSS), plus the bit-packed
 * multi-source variant (Alg. 5) and closeness centrality.
 * Every step of the path runs in hand-written sm_100a CUDA kernels inside this library; the Python
 * binding (paper_2606_05081_b200/binding.py) only marshals arguments.
 *
 * Conventions
 *  - All functions return an int status: BLEST_OK (0) or a negative BLEST_E* code.  Nothing throws or aborts.
 *    blest_strerror() names a status; blest_last_cuda_error() returns the cudaError_t behind BLEST_ECUDA.
 *  - The caller always speaks ORIGINAL vertex ids, whatever reordering blest_build applied inside.
 *  - Ownership: the library never keeps or frees caller memory.  blest_build copies what it needs; outputs
 *    are caller-allocated.  Output pointers may be DEVICE pointers (e.g. a torch tensor's data_ptr()) or
 *    HOST pointers (pinned or pageable): the library detects which with cudaPointerGetAttributes and, for
 *    host outputs, copies device->host on `cuda_stream` inside the call.
 *  - Asynchrony: traversal calls enqueue on `cuda_stream` (a cudaStream_t cast to void*, NULL = legacy
 *    default stream) and return without waiting for the device; results are valid once the stream is
 *    synchronised.  One handle owns one workspace: calls on the same handle must be stream-ordered.  Host
 *    `srcs` arrays are consumed before return (copied to a handle-owned pinned staging slot; temporaries are
 *    stream-ordered allocations).  Because the calls do not wait, an error that only the device can see (an
 *    internal work-queue overflow) cannot be returned by the call that caused it: it is latched in the handle,
 *    returned by blest_last_status() and by every later traversal call on the handle until it is read there.
 *  - Graph precondition: symmetric (undirected) CSR unless csr.directed, rows sorted ascending, column ids < n,
 *    rowptr[0] = 0, rowptr[n] = nnz < 2^32, 1 <= n <= 2^29 (narrower than uint32 because the kernels pack flags
 *    beside ids: bit 31 of a vertex id in the inline heads / bottom-up lists, 5 bits beside a slice-set id in a
 *    32-bit queue entry; the largest config has n = 2^25).  Self-loops and duplicate entries are legal and have no
 *    effect on the result.  Unsorted rows are always detected
 *    (BLEST_EUNSORTED); symmetry and ranges are checked only when options.validate != 0.
 */
#ifndef BLEST_H
#define BLEST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct blest_graph *blest_handle_t; /* opaque; owns device BVSS, device CSR, perm/iperm, workspace */

enum {
  BLEST_OK = 0,
  BLEST_EINVAL = -1,       /* NULL pointer, src >= n, k = 0, bad option value */
  BLEST_ERANGE = -2,       /* n = 0, n > 2^29, nnz >= 2^32, slice count overflow */
  BLEST_EUNSORTED = -3,    /* a CSR row is not sorted ascending */
  BLEST_ENOTSYM = -4,      /* (validate only) structure is not symmetric / column id out of range */
  BLEST_ENOMEM = -5,       /* host or device allocation failed */
  BLEST_ECUDA = -6,        /* a CUDA call failed; see blest_last_cuda_error() */
  BLEST_EUNSUPPORTED = -7, /* no sm_100 device / cooperative launch unavailable */
  BLEST_EOVERFLOW = -8     /* internal work queue overflow (should not happen with the automatic capacities; latched
                              by the kernels, reported by blest_last_status() and by later calls, never silent) */
};

/* Input graph ("CSC of A").  Symmetric by default, so that one CSR serves as A, A^T and Alg. 4's CSR(G^T);
 * `directed` widens it to the paper's full problem statement. */
typedef struct {
  uint32_t n;             /* vertices */
  uint64_t nnz;           /* directed entries = 2 * undirected edges */
  const uint32_t *rowptr; /* n+1 entries */
  const uint32_t *colidx; /* nnz entries */
  int on_device;          /* 0: host pointers, 1: device pointers (copied to the host for the host builder) */
  int directed;           /* 0: symmetric (undirected) graph.  1: DIRECTED graph: row u lists the
                             out-neighbours of u (the non-zeros of column u of A = the transposed adjacency matrix);
                             levels are hop distances along the edge direction.  The library also keeps the transposed
                             CSR (in-neighbours) for the bottom-up stage (Alg. 4 scans CSR(G^T)).
                             Restrictions: reorder = none | degree (by out-degree); no component pruning; closeness
                             always counts per source; blest_farness_partial is refused (BLEST_EUNSUPPORTED). */
} blest_csr_t;

/* Options.  Zero-initialised == defaults.  reorder/builder/validate are used by blest_build only; the rest
 * can be changed later with blest_configure (so that every path can be forced on one handle: the
 * policy-independence tests and the ablation axes of PAPER.md Tables 4/6). */
typedef struct {
  int reorder;     /* 0 none | 1 RCM | 2 degree-descending (BASELINE.json config 4) |
                      3 JaccardWithWindows (Alg. 1, W = 2^16) applied to the degree order */
  int builder;     /* 0 host (OpenMP over slice sets).  No other builder exists: any other value is BLEST_EINVAL */
  int validate;    /* 0 | 1: O(nnz log d) symmetry + range check */
  int kernel;      /* 0 auto by U_div | 1 eager (Alg. 2) | 2 lazy two-stage (Alg. 3) */
  int switching;   /* 0 auto (per-level cost model; Eq. 6 analogue) | 1 off: slice path only |
                      2 force bottom-up CUDA-core (Alg. 4) on every level >= 2 |
                      3 force top-down CUDA-core (CSR edges) | 4 force slice path | 5 scripted (reserved[0]) */
  int contraction; /* 0 auto | 1 ALU (AND + per-byte test) | 2 mma.sync m8n8k128 b1 and.popc (paper layout, Fig. 3) |
                      3 mma.sync m16n8k32 u8 (bits expanded to bytes) */
  int kappa;       /* multi-source width: 0 -> 64 | 32 | 64 | 128 | 256 (reading R19) */
  int trace;       /* 0 | 1: keep the per-level trace / the multi-source totals of the last call (default) | 2: off (the
                      leader thread then writes no record after a level: about a microsecond per level) */
  float eta;       /* bottom-up switch constant (Eq. 6, eta = 10 on Hopper); 0 -> library default */
  float gamma;     /* scales the slice-path cost in the per-slice-set slice-vs-CSR-edges threshold; 0 -> 1.0 */
  int persist_l2;  /* 0 auto | 1 off.  auto: a single-source traversal of a REORDERED graph whose 4n-byte levels_out
                      fits the device's persisting-L2 carve-out writes levels straight to original ids under a
                      persisting access-policy window of that launch; while such handles exist the library owns
                      cudaLimitPersistingL2CacheSize of the device (the value found is restored by the last
                      blest_destroy).  off: levels go to an internal-id array and one gather pass ends the call. */
  int prune_components; /* 0 on | 1 off.  on: blest_build labels the connected component of the highest-degree vertex
                      (one host BFS, timed as info.component_seconds); a traversal whose source lies in it starts
                      with everything outside marked visited, so no sweep examines vertices it cannot reach.
                      Result-neutral; not part of the paper's method. */
  uint32_t queue_capacity; /* 0 auto (exact bounds) | entries: caps the work queues / chunk list (tests of the
                      overflow report) */
  int tune[4];     /* experiment switches of the kernels, 0 = default: [0] = 1: the balanced top-down phase stages its
                      slice tiles in shared memory with TMA bulk copies (cp.async.bulk + mbarrier, two stages per warp)
                      instead of 128-bit loads into registers -- measured 14 % slower on config 4, hence off by default
                      (DESIGN.md §6); [1] = 1: the multi-source kernel never switches a batch to pull levels;
                      [2] = 1: the lazy kernel always pre-fills levels_out with -1 (no "level guess");
                      [3]: concurrent lanes of the closeness / farness calls (their source batches are split over that
                      many cooperative launches of grid / lanes CTAs on internal streams, forked from and joined into
                      the caller's stream): 0 = 8, k = k (1..16; 1 = one launch on the whole grid) */
  int reserved[6]; /* [0]: switching == 5 ("scripted", tests): level l runs bottom-up iff bit min(l,31) is set;
                      [1..5]: tuning overrides of the switch cost model in 0.01 ps per unit (top-down edge, top-down
                      vertex, bottom-up vertex, bottom-up scanned neighbour, bottom-up bitmap word); 0 = default */
} blest_options_t;

typedef struct {
  uint32_t n;
  uint64_t nnz;
  uint32_t n_slice_sets;   /* N_s = ceil(n / 8) */
  uint32_t n_vss;          /* N_v = sum over slice sets of ceil(slices/128) */
  uint64_t n_slices;       /* real (non-padding) slices */
  uint64_t n_quads;        /* 4-slice groups stored (each slice set padded to a multiple of 4 slices) */
  uint64_t bvss_bytes;     /* device bytes of rowIds + masks + setPtr */
  uint64_t csr_bytes;      /* device bytes of rowptr + colidx */
  uint64_t workspace_bytes;
  double mask_density;     /* nnz / n_slices (rho_c, 1..8) */
  double u_div;            /* update divergence (reading R20) */
  double reorder_seconds, build_seconds, upload_seconds;
  double component_seconds; /* options.prune_components: host BFS labelling the hub's component (0 when off) */
  int kernel_chosen;       /* 1 eager | 2 lazy (after auto dispatch) */
  int reorder, kappa, num_sms, grid_blocks, block_threads;
  uint32_t queue_capacity; /* entries per work queue */
  uint32_t n_sweep_words;  /* 32-vertex words (internal ids) that hold a vertex of non-zero degree: the range the
                              lazy kernel's per-level sweeps cover */
} blest_info_t;

/* One record per BFS level of the most recent blest_bfs call (written by the persistent kernel). */
typedef struct {
  uint32_t level;       /* l (1-based: vertices discovered in this record got level l) */
  uint32_t mode;        /* 0 queue (slice chunks and/or edge chunks) | 1 bottom-up | 2 eager queue */
  uint32_t q_entries;   /* work-queue entries consumed */
  uint32_t new_vertices;
  uint64_t q_bytes;     /* graph bytes the queue entries cover (20 B per quad, 4 B per edge) */
  uint64_t bu_scanned;  /* bottom-up: neighbours scanned */
  uint32_t unvisited;   /* after this level */
  uint32_t reserved;    /* bit 31: this level wrote no levels (levels_out was pre-filled with it: the level guess) */
  uint64_t t_ns;        /* %globaltimer at the end of the level, relative to kernel start */
  uint64_t t_stage1_ns; /* %globaltimer after the Stage-1 barrier of this level (lazy kernel), relative to kernel start */
} blest_level_trace_t;

/* Build: (optional reorder) -> BVSS -> U_div + dispatch -> upload.
 * Synchronous.  opt == NULL => defaults.  Timed separately from traversal; see blest_get_info. */
int blest_build(const blest_csr_t *csr, const blest_options_t *opt, blest_handle_t *out);

/* Host-only pre-processing: the same reorder -> BVSS -> U_div pipeline as blest_build, without touching a device
 * (csr->on_device must be 0).  The handle answers blest_get_info / blest_get_array only; traversal calls return
 * BLEST_EUNSUPPORTED.  Used by the CPU tests of the host logic and for offline inspection. */
int blest_preprocess_host(const blest_csr_t *csr, const blest_options_t *opt, blest_handle_t *out);

/* Change the run-time options (kernel, switching, contraction, kappa, trace, eta, gamma). */
int blest_configure(blest_handle_t h, const blest_options_t *opt);

/* Single-source BFS (Alg. 2/3/4; one persistent cooperative kernel).
 * levels_out: int32[n], device or host; levels_out[v] = hop distance from src, 0 for src, -1 if unreachable. */
int blest_bfs(blest_handle_t h, uint32_t src, int32_t *levels_out, void *cuda_stream);

/* Multi-source BFS (Alg. 5): srcs host uint32[k], k >= 1 (batched by kappa inside; duplicates legal).
 * levels_out: int32[k*n], device or host; row b belongs to srcs[b], original ids, -1 = unreachable. */
int blest_msbfs(blest_handle_t h, const uint32_t *srcs, uint32_t k, int32_t *levels_out, void *cuda_stream);

/* Closeness centrality (Eq. 7-8; readings R13/R14): out[i] = (reach_i - 1) / far_i in fp64, 0.0 when
 * far_i = 0.  srcs host uint32[n_srcs], or NULL = all vertices 0..n-1 (then n_srcs must be n; uses the paper's
 * target-side accumulation).  out: double[n_srcs], device or host. */
int blest_closeness(blest_handle_t h, const uint32_t *srcs, uint64_t n_srcs, double *out, void *cuda_stream);

/* Same traversal as blest_closeness, returning the exact integers: far_out uint64[n_srcs] (sum of hop distances
 * to all reachable vertices), reach_out uint32[n_srcs] (reachable vertices including the source).  Either may be NULL. */
int blest_farness(blest_handle_t h, const uint32_t *srcs, uint64_t n_srcs, uint64_t *far_out, uint32_t *reach_out,
                  void *cuda_stream);

/* Multi-GPU closeness by source partition ("sources partitioned over GPUs, partial sums reduced at the
 * end"): the target-side sums of Eq. 7 over the source range [first, first + count) only.  far_sum uint64[n],
 * reach_sum uint32[n], DEVICE pointers, indexed by ORIGINAL vertex id: far_sum[v] = sum over the sources s of the range
 * of d(s, v), reach_sum[v] = how many of them reach v.  Summing the arrays of disjoint ranges that cover 0..n-1 (one
 * all-reduce) gives the farness / reach of every vertex (the graph is undirected); blest_closeness_from_sums divides. */
int blest_farness_partial(blest_handle_t h, uint32_t first, uint32_t count, uint64_t *far_sum, uint32_t *reach_sum,
                          void *cuda_stream);

/* out[v] = (reach_sum[v] - 1) / far_sum[v] in fp64, 0.0 when far_sum[v] = 0 (Eq. 8, reading R14).  Device pointers. */
int blest_closeness_from_sums(const uint64_t *far_sum, const uint32_t *reach_sum, uint64_t n, double *out,
                              void *cuda_stream);

/* Allocation-free closeness of a source subset, for callers that cannot allocate (CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc).  Same result as blest_closeness(h, srcs, n_srcs, out, stream) (Eq. 7-8 with
 * per-source counts, reading R13), but the call performs NO cudaMalloc / cudaFree / cudaMallocAsync / cudaHostAlloc:
 * its scratch (the kappa-bit state arrays, dirtySets, the per-source sums, a copy of the source ids) lives in ONE
 * file-scope `static __device__` array of about 6.2 MiB that every GPU loading the library holds until the process
 * exits; the work queues and the control block are the handle's (allocated by blest_build).
 *   srcs_dev  DEVICE uint32[n_srcs], original ids (ids >= n are a caller error; they are clamped to n - 1, not checked);
 *   out_dev   DEVICE double[n_srcs].
 * Limits (BLEST_ERANGE beyond them, nothing is truncated; see blest_noalloc_limits): n_srcs <= 4096;
 * ceil(n/8) * 8 * kappa/8 <= 2 MiB, i.e. n <= 262 144 at kappa = 64, 65 536 at kappa = 256; n <= 524 288.
 * The array is shared by ALL calls and handles of the process and keeps the last call's contents; what must start at
 * zero is cleared at the start of each call on `cuda_stream`.  Calls that overlap on the GPU (different streams without
 * ordering) race on it: keep them stream-ordered. */
int blest_closeness_noalloc(blest_handle_t h, const uint32_t *srcs_dev, uint32_t n_srcs, double *out_dev, void *cuda_stream);
int blest_noalloc_limits(uint32_t *max_srcs, uint64_t *max_state_bytes, uint64_t *max_vertices_at_kappa64);

/* Totals of the most recent multi-source launch, for the roofline (needs options.trace): out8[0] work-queue entries
 * (VSS chunks) consumed by Stage 1, [1] quads they hold, [2] slices with a non-zero selection (V_next probed), [3] row words updated
 * by an atomic, [4] dirty slice sets swept by Stage 2, [5] levels (top-down and pull), [6] source batches, [7] neighbours
 * read by the pull levels; totals over the concurrent lanes of the call.  Synchronises the device. */
int blest_get_ms_stats(blest_handle_t h, uint64_t *out8);
/* Where the most recent multi-source launch spent its time (needs options.trace), in nanoseconds of %globaltimer as seen
 * by thread 0 of CTA 0, summed over all batches and levels: out8[0] per-batch init (state clears, source bits, level-0
 * sweep, their barriers), [1] Stage 1 own work, [2] wait at the barrier after Stage 1, [3] Stage 2
 * own work, [4] wait at the barrier after Stage 2, [5] rows a pull level scanned (some live source not
 * there yet), [6] pull levels, [7] 0; a pull level's own work counts under [1], its barrier under [2].  With concurrent
 * lanes the times are those of lane 0 (its share of the batches), the pull counters totals.  Synchronises the device. */
int blest_get_ms_phases(blest_handle_t h, uint64_t *out8);
/* Per-level record of the first levels (at most 60, over consecutive batches) of the most recent multi-source launch
 * (needs options.trace): four words per level -- (level << 32 | work-queue entries consumed), ns of Stage 1 + its
 * barrier, ns of Stage 2 + its barrier, entries enqueued for the next level -- as thread 0 of CTA 0 sees them.
 * `out` has room for 4 * max_levels words; *n_levels = records written.  Synchronises the device. */
int blest_get_ms_level_trace(blest_handle_t h, uint64_t *out, uint32_t max_levels, uint32_t *n_levels);

int blest_get_info(blest_handle_t h, blest_info_t *info);

/* Deferred status of the handle: synchronises the device, returns BLEST_EOVERFLOW if any traversal since the last
 * call of this function overflowed an internal work queue (its results are then incomplete), else BLEST_OK, and
 * clears the latch. */
int blest_last_status(blest_handle_t h);

/* Per-level trace of the last blest_bfs call.  Synchronises the device.  *n_levels = records available
 * (may exceed cap; only min(cap, available) are copied). */
int blest_get_trace(blest_handle_t h, blest_level_trace_t *buf, uint32_t cap, uint32_t *n_levels);

/* Timing of the most recent blest_bfs call on the lazy kernel, from the kernel's own %globaltimer stamps:
 * *init_ns = kernel start -> end of the per-call init (bitmap clears, levels_out = -1), *levels_ns = kernel start ->
 * end of the last level.  Synchronises the device.  Either pointer may be NULL. */
int blest_get_call_stats(blest_handle_t h, uint64_t *init_ns, uint64_t *levels_ns);

/* Copy one internal array to a HOST buffer (tests: BVSS round trip, permutation bijection).  `which`:
 * 0 setPtr uint32[N_s+1] (quad offsets) | 1 rowIds uint32[4*n_quads] | 2 masks uint32[n_quads] |
 * 3 realPtrs uint32[N_s+1] | 4 virtualToReal uint32[N_v] | 5 perm uint32[n] (orig -> internal) |
 * 6 iperm uint32[n] | 7 internal rowptr uint32[n+1] | 8 internal colidx uint32[nnz].
 * bytes must equal the array size exactly. */
int blest_get_array(blest_handle_t h, int which, void *host_dst, uint64_t bytes);

/* getVI(u, rho) = (u mod 8) * rho + floor(u / 8): the multi-source re-indexing, exported for tests. */
uint64_t blest_get_vi(uint64_t u, uint64_t rho);

/* Exhaustive device self-test of one contraction form against (mask & alpha) != 0 over all 2^8 x 2^8 pairs in
 * all four byte positions.  *n_mismatch = differing results (0 = pass). */
int blest_contraction_selftest(int contraction, uint64_t *n_mismatch);

/* Tensor-pipe peak microbenchmark: issues `iters` dependent-free MMA instructions per warp on every SM and
 * reports tera-ops/s (one op = one multiply-accumulate on one bit (b1) or one byte (u8)), 2 ops per MAC not applied.
 * kind: 2 = mma.sync m8n8k128 b1 and.popc | 3 = mma.sync m16n8k32 u8. */
int blest_mma_microbench(int kind, uint32_t iters, double *tera_macs_per_s, double *milliseconds);

/* tcgen05.mma kind::i8 peak (the Blackwell tensor-core form north_star (b) names; operands in shared memory,
 * accumulator in TMEM): `iters` MMAs of shape M = 128, N = n (16..256, multiple of 16), K = 32 per SM, issued by one
 * thread per CTA; tera byte-MACs per second.  The accumulator is read back with tcgen05.ld and checked against
 * 32 * iters for all-ones operands: *n_wrong = accumulator elements that differ (0 = the path works). */
int blest_tcgen05_microbench(uint32_t iters, uint32_t n, double *tera_macs_per_s, uint64_t *n_wrong);

/* L2 bandwidth microbenchmark (roofline denominator of the L2-resident multi-source path): a 16-byte-per-thread copy
 * between two buffers of bytes/2 each, `iters` passes, in the persistent launch configuration; read + write GB/s. */
int blest_l2_microbench(uint64_t bytes, uint32_t iters, double *gb_per_s);

/* Grid-barrier latency microbenchmark: `iters` back-to-back grid barriers in the persistent launch configuration. */
int blest_barrier_microbench(uint32_t iters, double *ns_per_barrier);

/* Thread-block-cluster microbenchmark (the candidate small-frontier mode of DESIGN.md §9): ONE cluster of `cluster_ctas`
 * (1, 2, 4, 8 or -- non-portable -- 16) CTAs of 1 024 threads executes `iters` back-to-back cluster barriers
 * (barrier.cluster arrive.release / wait.acquire) and a chain of `iters` dependent loads from the other CTAs' shared memory
 * (mapa + ld.shared::cluster); nanoseconds per barrier and per load. */
int blest_cluster_microbench(int cluster_ctas, uint32_t iters, double *ns_per_barrier, double *ns_per_dsmem_load);

void blest_destroy(blest_handle_t h);
const char *blest_strerror(int status);
int blest_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BLEST_H */
