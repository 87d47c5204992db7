// bfs_kernels.cuh -- parameter blocks and launch wrappers of the persistent traversal kernels.
#pragma once
#include "device_common.cuh"

namespace blest {

// Tunables of the lazy kernel's top-down stage.
constexpr uint32_t BIG_EDGES = 512;     // longer adjacency lists are deferred to the balanced phase
constexpr uint32_t BIG_QUADS = 128;     // longer slice sets (in quads) are deferred to the balanced phase
constexpr uint32_t CHUNK_EDGES = 256;   // balanced phase: edges per chunk entry
constexpr uint32_t CHUNK_QUADS = 64;    // balanced phase: quads per chunk entry
constexpr uint32_t WL_STAGE = 2048;     // per-CTA shared-memory staging of frontier word ids

struct BfsParams {
  // graph (immutable during traversal)
  uint32_t n, Ns, nwords, qcap;
  uint64_t nnz;
  uint64_t nQuads;         // quads stored (bounds of rowIds / masks; debug asserts)
  uint32_t wlCap;          // capacity of a frontier word list (debug asserts)
  const uint32_t* setPtr;  // Ns+1 quad offsets
  const uint4* rowIds;     // nQuads
  const uint32_t* masks;   // nQuads
  const uint32_t* rowptr;  // internal (reordered) CSR, n+1: OUT-neighbours (the columns of A; top-down edge path)
  const uint32_t* colidx;
  const uint32_t* rowptrIn;  // CSR of the transposed graph: IN-neighbours (Alg. 4's CSR(G^T)); the same
  const uint32_t* colidxIn;  // arrays as rowptr / colidx when the graph is symmetric
  int srcPremarked;          // the source's bit is already set in isoBits (directed graph, source of in-degree 0)
  const uint32_t* perm;    // original -> internal id, or nullptr when no reordering
  const uint32_t* iperm;   // internal -> original id, or nullptr when no reordering
  const uint2* head;       // n: first two IN-neighbours of every vertex (x, y); 0xFFFFFFFF = none; y bit 31 = "has more"
  const uint32_t* deg;     // n: OUT-degrees (read where a discovered vertex is finalised, for the switch counters)
  const uint16_t* popThr;  // nwords: four 4-bit thresholds, one per slice set of the word (slice path iff
                           // popc(frontier byte) >= threshold; 9 = never)
  // lazy kernel state
  uint32_t nSweepWords;    // 32-vertex words covering every vertex of non-zero degree
  uint32_t nIsoInSweep;    // zero-degree vertices inside the sweep range
  const uint32_t* isoBits; // bitmap of zero-degree vertices (padded like V): they start out "visited" so that no
                           // sweep ever examines them; levels_out keeps their -1
  uint32_t* V;             // visited bitmap (single copy)
  uint32_t* F[3];          // frontier bitmaps, rotating: level l reads F[(l-1)%3], writes F[l%3], clears F[(l+1)%3]
  uint32_t* WL[2];         // frontier word lists (ids of non-zero words of the frontier bitmap), level parity
  uint4* chunks;           // balanced-phase chunk entries {start, count, alpha, type}
  uint32_t chunkCap;
  // eager kernel state
  uint2* Q[2];
  int32_t* stamp;  // last level at which a slice set was enqueued
  // levels
  int32_t* out;    // levels in ORIGINAL ids (device)
  int32_t* lvl;    // lazy kernel: where a finalised vertex's level is written: out (index = original id) or, with
                   // `gather`, the internal-id array L
  const uint32_t* ipermW;  // lazy kernel: iperm when lvl is indexed by original ids of a reordered graph, else nullptr
  uint32_t srcLvl;         // index of the source in lvl
  int gather;              // lazy kernel: final pass out[v] = lvl[perm[v]]
  const uint32_t* negBits; // lazy kernel, level guess: bitmap over the indices of lvl of the vertices this traversal cannot
                           // reach (everything outside the source's component), or nullptr = no guess (plain -1 pre-fill)
  int32_t* L;      // levels in internal ids (== out when there is no reordering)
  Ctrl* ctrl;
  unsigned int* hostStatus;  // host-mapped latch of the handle (overflow report), may be nullptr
  blest_level_trace_t* trace;
  uint32_t traceCap;
  uint32_t src;      // internal id
  uint32_t srcOrig;  // original id
  int switching;
  int contraction;
  uint32_t buMask;  // switching == 5: level l runs bottom-up iff bit min(l,31) is set
  float eta, gamma;
  // switch cost model, picoseconds per unit
  float cTdEdge, cTdNew, cTdVertex, cTdWord, cBuVertex, cBuScan, cBuWord;
  int tmaTiles;   // balanced top-down phase: slice tiles staged by TMA bulk copies (options.tune[0])
  int hubFilter;  // top-down marks of low-id vertices are de-duplicated per CTA (degree-sorted graphs)
  float scanExp;  // exponent of nnz/mf in the estimate of neighbours examined per bottom-up vertex
};

struct MsParams {
  uint32_t n, Ns, rho, qcap;
  uint64_t nQuads;  // bounds of rowIds / masks (debug asserts)
  const uint32_t* setPtr;
  const uint4* rowIds;
  const uint32_t* masks;
  const uint32_t* perm;   // original -> internal, or nullptr
  const uint32_t* iperm;  // internal -> original, or nullptr
  uint32_t* F;            // kappa-bit words at getVI index: [rho*8][KW]
  uint32_t* Vc;
  uint32_t* Vn;
  uint8_t* dirty;  // Ns
  uint2* Q[2];
  Ctrl* ctrl;
  unsigned int* hostStatus;  // host-mapped latch of the handle (overflow report), may be nullptr
  const uint32_t* srcs;  // device, original ids; nullptr = identity (source i = vertex srcBase + i)
  uint64_t srcBase;      // first vertex of the source range when srcs == nullptr (multi-GPU partition)
  uint64_t nsrcs;
  unsigned long long* stats;  // optional [16]: totals of the launch for the roofline (queue entries, quads, slices probed,
                              // fresh row updates, dirty slice sets swept, levels, batches), [8..12] phase times of CTA 0
  // outputs (any may be nullptr)
  int32_t* levels;              // [nsrcs][n] original ids
  unsigned long long* farT;     // target-side accumulation, indexed by getVI(internal id) (Eq. 7)
  uint32_t* reachT;
  unsigned long long* farS;     // per-source accumulation [nsrcs]
  uint32_t* reachS;
  int kappa;
  // pull levels (msbfs_kernels.cu ms_pull_level; target-side accumulation only): second frontier array, CSR of the
  // (relabelled) graph, the rotating live-source masks [3][8] and the queue length from which a batch switches
  uint32_t* F2;
  const uint32_t* rowptr;
  const uint32_t* colidx;
  uint32_t* live;
  uint32_t pullMin;  // 0 = never
};
constexpr uint32_t MS_TRACE_LEVELS = 60;     // levels recorded by the multi-source kernel's per-level trace
constexpr size_t MS_STATS_WORDS = 16 + 4 * MS_TRACE_LEVELS;


// persistPtr/persistBytes: optional persisting-L2 access-policy window of this launch (levels_out), nullptr/0 = none
cudaError_t launch_bfs_lazy(const BfsParams& p, int gridBlocks, cudaStream_t st, const void* persistPtr, size_t persistBytes,
                            float hitRatio);
cudaError_t launch_bfs_eager(const BfsParams& p, int gridBlocks, cudaStream_t st);
cudaError_t launch_isolated_source(int32_t* out, uint32_t n, uint32_t src, cudaStream_t st);
cudaError_t launch_add_partial_sums(unsigned long long* far0, uint32_t* reach0, const unsigned long long* far1,
                                    const uint32_t* reach1, uint64_t count, cudaStream_t st);
cudaError_t launch_msbfs(const MsParams& p, int gridBlocks, cudaStream_t st);
cudaError_t launch_closeness_finalize(uint32_t n, uint32_t rho, const uint32_t* perm, const unsigned long long* farT,
                                      const uint32_t* reachT, const unsigned long long* farS, const uint32_t* reachS,
                                      uint64_t nsrcs, double* cc, unsigned long long* farOut, uint32_t* reachOut,
                                      cudaStream_t st);
int max_coop_blocks_lazy();
int max_coop_blocks_eager();
int max_coop_blocks_msbfs();

// ---- allocation-free closeness of a source subset (blest_closeness_noalloc; msbfs_kernels.cu) ----------------------
constexpr uint32_t NOALLOC_MAX_SRCS = 4096;             // sources per call
constexpr uint64_t NOALLOC_MAX_STATE_BYTES = 2u << 20;  // bytes of ONE kappa-bit state array: ceil(n/8) * 8 * kappa/8
constexpr uint64_t NOALLOC_MAX_SETS = 1u << 16;         // slice sets (one dirty byte each): n <= 524 288
// p: everything but F / Vc / Vn / dirty / srcs / farS / reachS / stats, which are placed in the file-scope scratch
// array here.  srcsDev: device uint32[nsrcs] (ids >= n are clamped to n - 1 instead of faulting).  out: device fp64[nsrcs].
cudaError_t launch_closeness_noalloc(MsParams p, const uint32_t* srcsDev, uint32_t nsrcs, int gridBlocks, double* out,
                                     cudaStream_t st);

}  // namespace blest
