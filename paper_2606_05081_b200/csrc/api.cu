// api.cu -- the C ABI of include/blest.h: handle lifetime, device memory, launches.  No traversal arithmetic here.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <vector>

#include "bfs_kernels.cuh"
#include "host_graph.h"

namespace blest {
cudaError_t run_contraction_selftest(int contraction, unsigned long long* dMismatch);
cudaError_t run_mma_peak(int kind, uint32_t iters, int blocks, int* dSink, double* macsPerLaunch);
cudaError_t run_barrier_bench(unsigned int* dBar, uint32_t iters, int blocks, unsigned long long* dNs);
cudaError_t run_cluster_bench(int clusterCtas, uint32_t iters, unsigned long long* dOut);
cudaError_t run_l2_copy(const uint4* src, uint4* dst, uint64_t n16, uint32_t iters, int blocks);
cudaError_t run_tcgen05_peak(uint32_t iters, uint32_t n, int blocks, unsigned int* dBad, double* macsPerLaunch);
}  // namespace blest

using namespace blest;

static thread_local int g_lastCuda = 0;

#define CK(call)                                  \
  do {                                            \
    cudaError_t e__ = (call);                     \
    if (e__ != cudaSuccess) {                     \
      g_lastCuda = (int)e__;                      \
      cudaGetLastError();                         \
      return e__ == cudaErrorMemoryAllocation ? BLEST_ENOMEM : BLEST_ECUDA; \
    }                                             \
  } while (0)

static constexpr uint32_t TRACE_CAP = 1u << 17;
static constexpr double UDIV_THRESHOLD = 25000.0;
// switch cost model defaults, picoseconds per unit
static constexpr float COST_TD_EDGE = 4.6f, COST_TD_NEW = 16.5f, COST_TD_VERTEX = 40.0f, COST_TD_WORD = 30.0f;
static constexpr float COST_BU_VERTEX = 4.0f, COST_BU_SCAN = 4.5f, COST_BU_WORD = 20.0f;

struct blest_graph {
  uint32_t n = 0, Ns = 0, Nv = 0, nwords = 0, rho = 0, qcap = 0;
  uint64_t nnz = 0, nSlices = 0, nQuads = 0;
  blest_options_t opt{};
  blest_info_t info{};
  bool hasPerm = false;
  bool directed = false;  // rows are out-neighbours of a directed graph; the transposed CSR is kept for Alg. 4
  bool hubby = false;     // degree-sorted AND scale-free-like: the first 1 % of the vertices own >= 20 % of the edge endpoints
  bool hostOnly = false;  // blest_preprocess_host: no device arrays, traversal calls are refused
  HostBvss hb;            // kept only when hostOnly
  HostCsr hcsr;           // kept only when hostOnly
  std::vector<uint32_t> perm, iperm, realPtrs, virtualToReal;
  int gridLazy = 0, gridEager = 0, gridMs = 0;
  // device graph
  uint32_t *dSetPtr = nullptr, *dRowIds = nullptr, *dMasks = nullptr, *dRowptr = nullptr, *dColidx = nullptr;
  uint32_t *dPerm = nullptr, *dIperm = nullptr;
  uint32_t *dRowptrIn = nullptr, *dColidxIn = nullptr;  // transposed CSR (== dRowptr / dColidx for a symmetric graph)
  // single-source workspace
  uint32_t nSweepWords = 0, nIsoInSweep = 0, chunkCap = 0;
  std::vector<uint32_t> setQuads;  // per slice set: quads stored          (popThr is rebuilt when gamma changes)
  std::vector<uint64_t> setDeg;    // per slice set: degree sum of its 8 columns
  uint2* dHead = nullptr;
  uint32_t* dDeg = nullptr;
  uint32_t* dIso = nullptr;
  uint16_t* dPopThr = nullptr;
  std::vector<uint32_t> isoBits;  // host bitmap of the vertices nothing can discover (in-degree 0; internal ids)
  std::vector<uint32_t> deadSrc;  // host bitmap of the vertices of out-degree 0: such a source reaches nothing
  std::vector<uint32_t> hubComp;  // host bitmap of the connected component of the highest-degree vertex
  uint32_t* dOutside = nullptr;   // device bitmap: NOT in that component (zero-degree vertices included)
  uint32_t* dOutsideOrig = nullptr;  // the same bitmap indexed by ORIGINAL vertex id (reordered graphs; level guess)
  uint32_t nOutsideInSweep = 0;
  uint32_t *dV = nullptr, *dF[3] = {nullptr, nullptr, nullptr}, *dWL[2] = {nullptr, nullptr};
  uint4* dChunks = nullptr;
  uint2* dQ[2] = {nullptr, nullptr};
  Ctrl* dCtrl = nullptr;      // eager / multi-source kernels: zeroed by a memset node before every launch
  Ctrl* dCtrlLazy = nullptr;  // lazy kernel: zeroed once here, self-resetting afterwards (no memset per call)
  Ctrl* lastCtrl = nullptr;   // control block of the most recent traversal (blest_get_trace / blest_get_call_stats)
  unsigned int* hStatus = nullptr;  // host-mapped latch: a kernel that overflows a work queue stores 1 here
  int device = 0;
  bool persistRef = false;    // this handle holds a reference on the device's persisting-L2 state
  blest_level_trace_t* dTrace = nullptr;
  int32_t *dL = nullptr, *dStamp = nullptr, *dOut = nullptr;
  // multi-source workspace: grow-only (sized for the widest kappa used so far; a wider kappa frees and re-allocates)
  uint64_t msWords = 0;
  uint32_t *dMsF = nullptr, *dMsVc = nullptr, *dMsVn = nullptr, *dMsF2 = nullptr, *dMsLive = nullptr;
  // pinned staging slots for host `srcs` arrays (consumed before the call returns; recycled once their copy has run)
  struct StageSlot { void* host = nullptr; size_t cap = 0; cudaEvent_t ev = nullptr; };
  std::vector<StageSlot> stage;
  // concurrent lanes of the multi-source calls (launch_ms_lanes): lane 0 is the workspace above on the caller's stream,
  // lanes 1.. own a stream, an event and a second copy of every per-launch array
  struct MsLane {
    cudaStream_t st = nullptr;
    cudaEvent_t done = nullptr;
    uint64_t words = 0;  // size of the state arrays (grow-only with kappa, as lane 0)
    uint32_t *F = nullptr, *F2 = nullptr, *Vc = nullptr, *Vn = nullptr, *live = nullptr;
    uint8_t* dirty = nullptr;
    uint2* Q[2] = {nullptr, nullptr};
    Ctrl* ctrl = nullptr;
    unsigned long long* farT = nullptr;
    uint32_t* reachT = nullptr;
    unsigned long long* stats = nullptr;
  };
  std::vector<MsLane> msLanes;   // lanes 1..
  cudaEvent_t msFork = nullptr;
  int msLanesUsed = 1;           // lanes of the most recent multi-source launch (blest_get_ms_stats sums over them)
  uint8_t* dDirty = nullptr;
  unsigned long long* dFarT = nullptr;
  uint32_t* dReachT = nullptr;
  unsigned long long* dMsStats = nullptr;  // [16] totals of the last multi-source launch (blest_get_ms_stats) + phase times
                                           // of CTA 0 in [8..15] (blest_get_ms_phases)
  uint64_t wsBytes = 0;
  std::vector<void*> allocs;
};

template <class T>
static int dev_alloc(blest_graph* g, T** p, uint64_t count, bool zero = false) {
  uint64_t bytes = std::max<uint64_t>(count * sizeof(T), 16);
  bytes = (bytes + 15) & ~15ull;
  CK(cudaMalloc((void**)p, bytes));
  g->allocs.push_back((void*)*p);
  g->wsBytes += bytes;
  if (zero) CK(cudaMemset(*p, 0, bytes));
  return BLEST_OK;
}

static bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, p);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

static double now_s() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

static void normalise_options(blest_options_t& o) {
  if (o.kappa == 0) o.kappa = 64;
  if (o.eta <= 0.f) o.eta = 10.f;
  if (o.gamma <= 0.f) o.gamma = 1.0f;
}

static int check_options(const blest_options_t& o) {
  if (o.reorder < 0 || o.reorder > 3 || o.builder != 0) return BLEST_EINVAL;
  if (o.persist_l2 < 0 || o.persist_l2 > 1 || o.prune_components < 0 || o.prune_components > 1) return BLEST_EINVAL;
  if (o.kernel < 0 || o.kernel > 2 || o.switching < 0 || o.switching > 5) return BLEST_EINVAL;
  if (o.contraction < 0 || o.contraction > 3) return BLEST_EINVAL;
  if (o.kappa != 0 && o.kappa != 32 && o.kappa != 64 && o.kappa != 128 && o.kappa != 256) return BLEST_EINVAL;
  return BLEST_OK;
}

// Per slice set: the smallest number k of frontier columns from which the slice path is expected to be cheaper than
// the CSR edges of those columns.  Costs in byte equivalents; a bitmap probe / mark counts as MARK
// bytes (one 32-byte L2 sector request).  Slices: 20 B per quad + one mark per slice that hits,
// P(hit) = 1 - (1 - k/8)^rho with rho = edges per slice; edges: (k/8) of the set's edges, 4 B + one mark each.
static void build_pop_thresholds(const blest_graph* g, float gamma, std::vector<uint16_t>& thr) {
  constexpr double MARK = 32.0;
  thr.assign(g->nwords, 0x9999u);
#pragma omp parallel for schedule(static)
  for (int64_t w = 0; w < (int64_t)g->nwords; ++w) {
    uint32_t packed = 0;
    for (uint32_t q = 0; q < 4; ++q) {
      const uint64_t s = (uint64_t)w * 4 + q;
      uint32_t t = 9;
      if (s < g->Ns && g->setQuads[s] > 0 && g->setDeg[s] > 0) {
        const double nq = g->setQuads[s], D = (double)g->setDeg[s];
        const double S = 4.0 * nq, rho = std::max(1.0, D / S);
        for (uint32_t k = 1; k <= 8; ++k) {
          const double cs = 20.0 * nq + S * MARK * (1.0 - std::pow(1.0 - k / 8.0, rho));
          const double ce = (k / 8.0) * D * (4.0 + MARK) + 8.0 * k;
          if (cs * gamma <= ce) { t = k; break; }
        }
      }
      packed |= t << (4 * q);
    }
    thr[w] = (uint16_t)packed;
  }
}

static int upload_pop_thresholds(blest_graph* g) {
  std::vector<uint16_t> thr;
  build_pop_thresholds(g, g->opt.gamma, thr);
  CK(cudaMemcpy(g->dPopThr, thr.data(), thr.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
  return BLEST_OK;
}

// Persisting-L2 set-aside.  cudaLimitPersistingL2CacheSize is a DEVICE-wide limit, so it is managed per device, under a
// lock, and only while handles that use it exist (options.persist_l2 = auto on a reordered graph): the first such handle
// records the limit it found, the last blest_destroy restores it.  While the library owns it, the set-aside is switched on
// for the lazy single-source traversals that put a window over levels_out and off for every other path (an unused
// set-aside just shrinks the L2 for everything else: measured 3x slower bottom-up levels).
struct PersistState {
  int refs = 0;
  size_t original = 0, current = 0;
  int maxPersist = -1, maxWindow = -1;
};
static std::mutex g_persistMutex;
static std::map<int, PersistState> g_persist;

static PersistState& persist_state_locked(int dev) {
  PersistState& ps = g_persist[dev];
  if (ps.maxPersist < 0) {
    if (cudaDeviceGetAttribute(&ps.maxPersist, cudaDevAttrMaxPersistingL2CacheSize, dev) != cudaSuccess) ps.maxPersist = 0;
    if (cudaDeviceGetAttribute(&ps.maxWindow, cudaDevAttrMaxAccessPolicyWindowSize, dev) != cudaSuccess) ps.maxWindow = 0;
    cudaGetLastError();
  }
  return ps;
}
static void persist_acquire(blest_graph* g) {
  std::lock_guard<std::mutex> lk(g_persistMutex);
  PersistState& ps = persist_state_locked(g->device);
  if (ps.refs++ == 0) {
    if (cudaDeviceGetLimit(&ps.original, cudaLimitPersistingL2CacheSize) != cudaSuccess) ps.original = 0;
    cudaGetLastError();
    ps.current = ps.original;
  }
  g->persistRef = true;
}
static void persist_set_locked(PersistState& ps, size_t bytes) {
  if (bytes == ps.current) return;
  if (bytes == 0) cudaCtxResetPersistingL2Cache();
  cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, bytes);
  cudaGetLastError();
  ps.current = bytes;
}
static void persist_release(blest_graph* g) {
  if (!g->persistRef) return;
  std::lock_guard<std::mutex> lk(g_persistMutex);
  PersistState& ps = persist_state_locked(g->device);
  if (--ps.refs == 0) persist_set_locked(ps, ps.original);
  g->persistRef = false;
}
// Called by every traversal of a handle that holds a reference: bytes > 0 switches the set-aside on (capped at the
// device maximum), 0 switches it off.  Returns the bytes in force.
static size_t persist_use(blest_graph* g, size_t bytes) {
  if (!g->persistRef) return 0;
  std::lock_guard<std::mutex> lk(g_persistMutex);
  PersistState& ps = persist_state_locked(g->device);
  persist_set_locked(ps, bytes ? (size_t)ps.maxPersist : 0);
  return ps.current;
}
static bool persist_fits(blest_graph* g, size_t bytes) {
  std::lock_guard<std::mutex> lk(g_persistMutex);
  PersistState& ps = persist_state_locked(g->device);
  return bytes <= (size_t)ps.maxPersist && bytes <= (size_t)ps.maxWindow;
}
static size_t persist_max(blest_graph* g) {
  std::lock_guard<std::mutex> lk(g_persistMutex);
  return (size_t)persist_state_locked(g->device).maxPersist;
}

extern "C" {

const char* blest_strerror(int status) {
  switch (status) {
    case BLEST_OK: return "ok";
    case BLEST_EINVAL: return "invalid argument";
    case BLEST_ERANGE: return "size out of range";
    case BLEST_EUNSORTED: return "CSR rows are not sorted";
    case BLEST_ENOTSYM: return "CSR is not structurally symmetric or has out-of-range column ids";
    case BLEST_ENOMEM: return "out of memory";
    case BLEST_ECUDA: return "CUDA error";
    case BLEST_EUNSUPPORTED: return "unsupported device or option";
    case BLEST_EOVERFLOW: return "internal work queue overflow";
    default: return "unknown status";
  }
}

int blest_last_cuda_error(void) { return g_lastCuda; }

uint64_t blest_get_vi(uint64_t u, uint64_t rho) { return (u % SIGMA) * rho + u / SIGMA; }

void blest_destroy(blest_handle_t h) {
  if (!h) return;
  if (!h->hostOnly) {
    cudaDeviceSynchronize();  // enqueued work may still use the workspace
    cudaGetLastError();
    persist_release(h);
  }
  for (void* p : h->allocs) cudaFree(p);
  for (auto& ln : h->msLanes) {
    if (ln.done) cudaEventDestroy(ln.done);
    if (ln.st) cudaStreamDestroy(ln.st);
  }
  if (h->msFork) cudaEventDestroy(h->msFork);
  for (auto& sl : h->stage) {
    if (sl.ev) cudaEventDestroy(sl.ev);
    if (sl.host) cudaFreeHost(sl.host);
  }
  if (h->hStatus) cudaFreeHost(h->hStatus);
  delete h;
}

static int build_impl(const blest_csr_t* csr, const blest_options_t* optIn, blest_handle_t* out, bool hostOnly) {
  if (!csr || !out || !csr->rowptr || (!csr->colidx && csr->nnz)) return BLEST_EINVAL;
  *out = nullptr;
  blest_options_t opt{};
  if (optIn) opt = *optIn;
  int rc = check_options(opt);
  if (rc) return rc;
  normalise_options(opt);
  if (csr->n == 0 || csr->n > (1u << 29) || csr->nnz > 0xFFFFFFFFull) return BLEST_ERANGE;
  if (hostOnly && csr->on_device) return BLEST_EINVAL;

  int sms = 0, dev = 0;
  if (!hostOnly) {
    int major = 0, coop = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10 || !coop) return BLEST_EUNSUPPORTED;
  }

  blest_graph* g = new (std::nothrow) blest_graph();
  if (!g) return BLEST_ENOMEM;
  g->hostOnly = hostOnly;
  g->device = dev;
  struct Guard { blest_graph* g; ~Guard() { if (g) blest_destroy(g); } } guard{g};

  try {
    HostCsr in;
    in.n = csr->n;
    in.nnz = csr->nnz;
    in.rowptr.resize((size_t)csr->n + 1);
    in.colidx.resize((size_t)csr->nnz);
    if (csr->on_device) {
      CK(cudaMemcpy(in.rowptr.data(), csr->rowptr, in.rowptr.size() * 4, cudaMemcpyDeviceToHost));
      if (csr->nnz) CK(cudaMemcpy(in.colidx.data(), csr->colidx, in.colidx.size() * 4, cudaMemcpyDeviceToHost));
    } else {
      std::memcpy(in.rowptr.data(), csr->rowptr, in.rowptr.size() * 4);
      if (csr->nnz) std::memcpy(in.colidx.data(), csr->colidx, in.colidx.size() * 4);
    }
    const bool directed = csr->directed != 0;
    if (directed && (opt.reorder == 1 || opt.reorder == 3)) return BLEST_EUNSUPPORTED;  // RCM / Jaccard: symmetric input only
    rc = check_csr(in, opt.validate != 0 && !directed);
    if (rc) return rc;
    g->directed = directed;

    // A1 reorder (timed separately, Table 7)
    double t0 = now_s();
    HostCsr work;
    HostCsr* gcsr = &in;
    if (opt.reorder) {
      make_permutation(in, opt.reorder, g->perm);
      g->iperm.resize(in.n);
      for (uint32_t i = 0; i < in.n; ++i) g->iperm[g->perm[i]] = i;
      relabel_csr(in, g->perm, work);
      std::vector<uint32_t>().swap(in.colidx);
      std::vector<uint32_t>().swap(in.rowptr);
      gcsr = &work;
      g->hasPerm = true;
    }
    g->info.reorder_seconds = now_s() - t0;

    // A2 BVSS build + A3 statistics
    t0 = now_s();
    HostBvss b;
    rc = build_bvss(*gcsr, b);
    if (rc) return rc;
    g->info.build_seconds = now_s() - t0;

    g->n = gcsr->n;
    g->nnz = gcsr->nnz;
    g->Ns = b.Ns;
    g->Nv = b.Nv;
    g->rho = b.Ns;  // rho = ceil(n / sigma)
    g->nSlices = b.nSlices;
    g->nQuads = b.nQuads;
    g->nwords = (g->n + 31) / 32;
    // Directed graph: A = the transposed adjacency matrix, so the rows given are the COLUMNS of A (the
    // BVSS builder reads them as such), and Alg. 4 scans IN-neighbours: the transposed CSR, by a counting sort.
    HostCsr gin;
    if (directed) {
      gin.n = gcsr->n;
      gin.nnz = gcsr->nnz;
      gin.rowptr.assign((size_t)gin.n + 1, 0);
      gin.colidx.resize(gin.nnz);
      for (uint64_t e = 0; e < gcsr->nnz; ++e) ++gin.rowptr[gcsr->colidx[e] + 1];
      for (uint32_t i = 0; i < gin.n; ++i) gin.rowptr[i + 1] += gin.rowptr[i];
      std::vector<uint32_t> fill(gin.rowptr.begin(), gin.rowptr.end() - 1);
      for (uint32_t u = 0; u < gcsr->n; ++u)  // ascending u: every in-list comes out sorted
        for (uint32_t e = gcsr->rowptr[u]; e < gcsr->rowptr[u + 1]; ++e) gin.colidx[fill[gcsr->colidx[e]]++] = u;
    }
    const HostCsr* gcsrIn = directed ? &gin : gcsr;
    {  // sweep range of the lazy kernel: the 32-vertex words that hold a vertex with an edge; vertices nothing can
       // discover (in-degree 0) start out visited
      g->isoBits.assign(g->nwords, 0u);
      g->deadSrc.assign(g->nwords, 0u);
      uint32_t last = 0;
      bool any = false;
      for (uint32_t u = 0; u < g->n; ++u) {
        const bool noIn = gcsrIn->rowptr[u + 1] == gcsrIn->rowptr[u], noOut = gcsr->rowptr[u + 1] == gcsr->rowptr[u];
        if (noIn) g->isoBits[u >> 5] |= 1u << (u & 31u);
        if (noOut) g->deadSrc[u >> 5] |= 1u << (u & 31u);
        if (!noIn || !noOut) { last = u; any = true; }
      }
      g->nSweepWords = any ? last / 32u + 1u : 0u;
      uint32_t iso = 0;
      for (uint32_t w = 0; w < g->nSweepWords; ++w) iso += (uint32_t)__builtin_popcount(g->isoBits[w]);
      g->nIsoInSweep = iso;
      // Connected component of the highest-degree vertex (level-synchronous host BFS, OpenMP over the frontier).  A
      // traversal from a source inside it can never leave it, so the lazy kernel starts with everything outside marked
      // visited: no sweep ever examines those vertices, and the traversal ends as soon as the component is exhausted.
      if (!hostOnly && any && opt.prune_components == 0 && !directed) {
        const double tc0 = now_s();
        uint32_t hub = 0, best = 0;
        for (uint32_t u = 0; u < g->n; ++u) {
          const uint32_t d = gcsr->rowptr[u + 1] - gcsr->rowptr[u];
          if (d > best) { best = d; hub = u; }
        }
        g->hubComp.assign(g->nwords, 0u);
        std::vector<uint32_t> frontier{hub}, next;
        g->hubComp[hub >> 5] |= 1u << (hub & 31u);
        while (!frontier.empty()) {
          next.clear();
#pragma omp parallel
          {
            std::vector<uint32_t> mine;
#pragma omp for schedule(dynamic, 256) nowait
            for (int64_t i = 0; i < (int64_t)frontier.size(); ++i) {
              const uint32_t u = frontier[i];
              for (uint32_t e = gcsr->rowptr[u]; e < gcsr->rowptr[u + 1]; ++e) {
                const uint32_t v = gcsr->colidx[e], bit = 1u << (v & 31u);
                if (g->hubComp[v >> 5] & bit) continue;
                const uint32_t old = __atomic_fetch_or(&g->hubComp[v >> 5], bit, __ATOMIC_RELAXED);
                if (!(old & bit)) mine.push_back(v);
              }
            }
#pragma omp critical
            next.insert(next.end(), mine.begin(), mine.end());
          }
          frontier.swap(next);
        }
        uint32_t outside = 0;
        for (uint32_t w = 0; w < g->nSweepWords; ++w) {
          const uint32_t valid = (w == g->nwords - 1 && (g->n & 31u)) ? ((1u << (g->n & 31u)) - 1u) : 0xFFFFFFFFu;
          outside += (uint32_t)__builtin_popcount(~g->hubComp[w] & valid);
        }
        g->nOutsideInSweep = outside;
        g->info.component_seconds = now_s() - tc0;
      }
    }
    // scale-free-like test in the spirit of PAPER.md:199 (fn. 2: the top 1 % of the vertices hold a large share of the
    // degree); only meaningful after the degree sort, where the top vertices are the first ones
    g->hubby = (opt.reorder == 2 || opt.reorder == 3) && g->nnz > 0 &&
               (double)gcsr->rowptr[std::max<uint32_t>(g->n / 100u, 1u)] >= 0.20 * (double)g->nnz;
    g->realPtrs.swap(b.realPtrs);
    g->virtualToReal.swap(b.virtualToReal);
    g->opt = opt;
    const double uDiv = b.uDiv;

    if (hostOnly) {
      g->info.bvss_bytes = ((uint64_t)g->Ns + 1) * 4 + g->nQuads * 20;
      g->info.csr_bytes = ((uint64_t)g->n + 1) * 4 + g->nnz * 4;
      g->hb = std::move(b);
      g->hcsr = std::move(*gcsr);
    } else {
      // upload
      t0 = now_s();
      uint64_t before = g->wsBytes;
      if ((rc = dev_alloc(g, &g->dSetPtr, (uint64_t)g->Ns + 1))) return rc;
      if ((rc = dev_alloc(g, &g->dRowIds, g->nQuads * 4))) return rc;
      if ((rc = dev_alloc(g, &g->dMasks, g->nQuads))) return rc;
      g->info.bvss_bytes = g->wsBytes - before;
      before = g->wsBytes;
      if ((rc = dev_alloc(g, &g->dRowptr, (uint64_t)g->n + 1))) return rc;
      if ((rc = dev_alloc(g, &g->dColidx, g->nnz))) return rc;
      g->info.csr_bytes = g->wsBytes - before;
      CK(cudaMemcpy(g->dSetPtr, b.setPtr.data(), ((size_t)g->Ns + 1) * 4, cudaMemcpyHostToDevice));
      if (g->nQuads) {
        CK(cudaMemcpy(g->dRowIds, b.rowIds.data(), (size_t)g->nQuads * 16, cudaMemcpyHostToDevice));
        CK(cudaMemcpy(g->dMasks, b.masks.data(), (size_t)g->nQuads * 4, cudaMemcpyHostToDevice));
      }
      CK(cudaMemcpy(g->dRowptr, gcsr->rowptr.data(), ((size_t)g->n + 1) * 4, cudaMemcpyHostToDevice));
      if (g->nnz) CK(cudaMemcpy(g->dColidx, gcsr->colidx.data(), (size_t)g->nnz * 4, cudaMemcpyHostToDevice));
      g->dRowptrIn = g->dRowptr;
      g->dColidxIn = g->dColidx;
      if (directed) {
        if ((rc = dev_alloc(g, &g->dRowptrIn, (uint64_t)g->n + 1))) return rc;
        if ((rc = dev_alloc(g, &g->dColidxIn, g->nnz))) return rc;
        g->info.csr_bytes += ((uint64_t)g->n + 1 + g->nnz) * 4;
        CK(cudaMemcpy(g->dRowptrIn, gin.rowptr.data(), ((size_t)g->n + 1) * 4, cudaMemcpyHostToDevice));
        if (g->nnz) CK(cudaMemcpy(g->dColidxIn, gin.colidx.data(), (size_t)g->nnz * 4, cudaMemcpyHostToDevice));
      }
      if (g->hasPerm) {
        if ((rc = dev_alloc(g, &g->dPerm, g->n))) return rc;
        if ((rc = dev_alloc(g, &g->dIperm, g->n))) return rc;
        CK(cudaMemcpy(g->dPerm, g->perm.data(), (size_t)g->n * 4, cudaMemcpyHostToDevice));
        CK(cudaMemcpy(g->dIperm, g->iperm.data(), (size_t)g->n * 4, cudaMemcpyHostToDevice));
      }
      {  // auxiliary arrays of the CUDA-core paths: inline heads (first two neighbours), capped degrees, per-set
         // degree sums for the slice/edge thresholds
        std::vector<uint2> head(g->n);
        std::vector<uint32_t> deg(g->n);
#pragma omp parallel for schedule(static)
        for (int64_t u = 0; u < (int64_t)g->n; ++u) {
          const uint32_t b0 = gcsrIn->rowptr[u], d = gcsrIn->rowptr[u + 1] - b0;  // in-neighbours (Alg. 4)
          uint2 hd = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
          if (d >= 1) hd.x = gcsrIn->colidx[b0];
          if (d >= 2) hd.y = gcsrIn->colidx[b0 + 1] | (d > 2 ? 0x80000000u : 0u);
          head[u] = hd;
          deg[u] = gcsr->rowptr[u + 1] - gcsr->rowptr[u];  // out-degree: what a frontier vertex expands
        }
        g->setQuads.resize(g->Ns);
        g->setDeg.resize(g->Ns);
#pragma omp parallel for schedule(static)
        for (int64_t s = 0; s < (int64_t)g->Ns; ++s) {
          g->setQuads[s] = b.setPtr[s + 1] - b.setPtr[s];
          const uint64_t u0 = (uint64_t)s * SIGMA, u1 = std::min<uint64_t>(u0 + SIGMA, g->n);
          g->setDeg[s] = gcsr->rowptr[u1] - gcsr->rowptr[u0];
        }
        if ((rc = dev_alloc(g, &g->dHead, g->n))) return rc;
        if ((rc = dev_alloc(g, &g->dDeg, g->n))) return rc;
        if ((rc = dev_alloc(g, &g->dIso, (uint64_t)g->nwords + 16, true))) return rc;
        CK(cudaMemcpy(g->dIso, g->isoBits.data(), (size_t)g->nwords * 4, cudaMemcpyHostToDevice));
        if (!g->hubComp.empty()) {
          std::vector<uint32_t> outside(g->nwords);
          for (uint32_t w = 0; w < g->nwords; ++w) {
            const uint32_t valid = (w == g->nwords - 1 && (g->n & 31u)) ? ((1u << (g->n & 31u)) - 1u) : 0xFFFFFFFFu;
            outside[w] = ~g->hubComp[w] & valid;
          }
          if ((rc = dev_alloc(g, &g->dOutside, (uint64_t)g->nwords + 16, true))) return rc;
          CK(cudaMemcpy(g->dOutside, outside.data(), (size_t)g->nwords * 4, cudaMemcpyHostToDevice));
          if (g->hasPerm) {  // by original id: what the pre-fill of levels_out reads (bfs_lazy.cu "level guess")
            std::vector<uint32_t> oo(g->nwords, 0u);
            for (uint32_t v = 0; v < g->n; ++v) {
              const uint32_t u = g->perm[v];
              if ((outside[u >> 5] >> (u & 31u)) & 1u) oo[v >> 5] |= 1u << (v & 31u);
            }
            if ((rc = dev_alloc(g, &g->dOutsideOrig, (uint64_t)g->nwords + 16, true))) return rc;
            CK(cudaMemcpy(g->dOutsideOrig, oo.data(), (size_t)g->nwords * 4, cudaMemcpyHostToDevice));
          }
        }
        if ((rc = dev_alloc(g, &g->dPopThr, (uint64_t)g->nwords + 16))) return rc;
        CK(cudaMemcpy(g->dHead, head.data(), (size_t)g->n * sizeof(uint2), cudaMemcpyHostToDevice));
        CK(cudaMemcpy(g->dDeg, deg.data(), (size_t)g->n * 4, cudaMemcpyHostToDevice));
        g->info.csr_bytes += (uint64_t)g->n * 12 + (uint64_t)g->nwords * 2;
        if ((rc = upload_pop_thresholds(g))) return rc;
      }
      g->info.upload_seconds = now_s() - t0;
      { HostBvss drop; std::swap(drop, b); }  // release the host copy

      // workspace
      const uint64_t qcap64 = (uint64_t)g->Nv + g->n + g->nnz / TD_CHUNK + 1024;
      if (qcap64 > 0xFFFFFFF0ull) return BLEST_ERANGE;
      g->qcap = (uint32_t)qcap64;
      if (opt.queue_capacity) g->qcap = std::min(g->qcap, std::max(opt.queue_capacity, 1u));
      if ((rc = dev_alloc(g, &g->dV, (uint64_t)g->nwords + 16, true))) return rc;
      for (int k = 0; k < 3; ++k)
        if ((rc = dev_alloc(g, &g->dF[k], (uint64_t)g->nwords + 16, true))) return rc;
      for (int k = 0; k < 2; ++k)
        if ((rc = dev_alloc(g, &g->dWL[k], (uint64_t)g->nSweepWords + 16384))) return rc;
      // every deferred segment owns more than BIG_EDGES edges / BIG_QUADS quads of its own => exact capacity bounds
      // (with one word per warp the thresholds are lower, but then there are at most 36 segments per warp of the grid)
      g->chunkCap = (uint32_t)(g->nnz / CHUNK_EDGES + g->nQuads / CHUNK_QUADS + g->nnz / BIG_EDGES + g->nQuads / BIG_QUADS + 16 +
                               36ull * 32ull * 1024ull);
      if (opt.queue_capacity) g->chunkCap = std::min(g->chunkCap, std::max(opt.queue_capacity, 1u));
      // the lists are zeroed: after an overflow (options.queue_capacity) a consumer may read an entry that was never
      // written, and an all-zero entry is an empty / in-range work item
      if ((rc = dev_alloc(g, &g->dChunks, g->chunkCap, true))) return rc;
      if ((rc = dev_alloc(g, &g->dQ[0], g->qcap, true))) return rc;
      if ((rc = dev_alloc(g, &g->dQ[1], g->qcap, true))) return rc;
      if ((rc = dev_alloc(g, &g->dCtrl, 1, true))) return rc;
      if ((rc = dev_alloc(g, &g->dCtrlLazy, 1, true))) return rc;
      CK(cudaHostAlloc((void**)&g->hStatus, sizeof(unsigned int), cudaHostAllocMapped));
      *g->hStatus = 0;
      if (g->hasPerm && opt.persist_l2 == 0) persist_acquire(g);
      if ((rc = dev_alloc(g, &g->dTrace, TRACE_CAP, true))) return rc;
      if ((rc = dev_alloc(g, &g->dStamp, g->Ns))) return rc;
      if ((rc = dev_alloc(g, &g->dOut, g->n))) return rc;
      if (g->hasPerm && (rc = dev_alloc(g, &g->dL, g->n))) return rc;

      g->gridLazy = max_coop_blocks_lazy();
      g->gridEager = max_coop_blocks_eager();
      g->gridMs = max_coop_blocks_msbfs();
      if (g->gridLazy <= 0 || g->gridEager <= 0 || g->gridMs <= 0) return BLEST_EUNSUPPORTED;
    }

    blest_info_t& I = g->info;
    I.n = g->n;
    I.nnz = g->nnz;
    I.n_slice_sets = g->Ns;
    I.n_vss = g->Nv;
    I.n_slices = g->nSlices;
    I.n_quads = g->nQuads;
    I.mask_density = g->nSlices ? (double)g->nnz / (double)g->nSlices : 0.0;
    I.u_div = uDiv;
    I.reorder = opt.reorder;
    I.num_sms = sms;
    I.grid_blocks = g->gridLazy;
    I.block_threads = BLOCK_THREADS;
    I.queue_capacity = g->qcap;
    I.n_sweep_words = g->nSweepWords;
  } catch (const std::bad_alloc&) {
    return BLEST_ENOMEM;
  }
  guard.g = nullptr;
  *out = g;
  return BLEST_OK;
}

int blest_build(const blest_csr_t* csr, const blest_options_t* opt, blest_handle_t* out) {
  return build_impl(csr, opt, out, false);
}

int blest_preprocess_host(const blest_csr_t* csr, const blest_options_t* opt, blest_handle_t* out) {
  return build_impl(csr, opt, out, true);
}

int blest_configure(blest_handle_t h, const blest_options_t* optIn) {
  if (!h || !optIn) return BLEST_EINVAL;
  blest_options_t o = *optIn;
  o.reorder = h->opt.reorder;
  o.builder = h->opt.builder;
  o.validate = h->opt.validate;
  o.prune_components = h->opt.prune_components;
  o.queue_capacity = h->opt.queue_capacity;
  int rc = check_options(o);
  if (rc) return rc;
  normalise_options(o);
  const bool gammaChanged = o.gamma != h->opt.gamma;
  h->opt = o;
  if (!h->hostOnly && h->hasPerm) {
    if (o.persist_l2 == 0 && !h->persistRef) persist_acquire(h);
    if (o.persist_l2 == 1 && h->persistRef) persist_release(h);
  }
  if (gammaChanged && !h->hostOnly) return upload_pop_thresholds(h);
  return BLEST_OK;
}

static int resolved_kernel(const blest_graph* g) {
  if (g->opt.kernel) return g->opt.kernel;
  return g->info.u_div > UDIV_THRESHOLD ? 2 : 1;
}

int blest_get_info(blest_handle_t h, blest_info_t* info) {
  if (!h || !info) return BLEST_EINVAL;
  h->info.kernel_chosen = resolved_kernel(h);
  h->info.kappa = h->opt.kappa;
  h->info.workspace_bytes = h->hostOnly ? 0 : h->wsBytes - h->info.bvss_bytes - h->info.csr_bytes;
  *info = h->info;
  return BLEST_OK;
}

// Deferred device-side errors (include/blest.h "Asynchrony"): latched by the kernels in a host-mapped word.
static int pending_status(blest_graph* h) {
  return (h->hStatus && *(volatile unsigned int*)h->hStatus) ? BLEST_EOVERFLOW : BLEST_OK;
}

int blest_last_status(blest_handle_t h) {
  if (!h) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_OK;
  CK(cudaDeviceSynchronize());
  const int rc = pending_status(h);
  *(volatile unsigned int*)h->hStatus = 0;
  return rc;
}

int blest_bfs(blest_handle_t h, uint32_t src, int32_t* levels_out, void* cuda_stream) {
  if (!h || !levels_out) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  if (src >= h->n) return BLEST_EINVAL;
  if (int rc = pending_status(h)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool devOut = is_device_ptr(levels_out);
  BfsParams p{};
  p.n = h->n; p.Ns = h->Ns; p.nwords = h->nwords; p.qcap = h->qcap; p.nnz = h->nnz;
  p.nQuads = h->nQuads; p.wlCap = h->nSweepWords + 16384u;
  p.setPtr = h->dSetPtr; p.rowIds = reinterpret_cast<const uint4*>(h->dRowIds); p.masks = h->dMasks;
  p.rowptr = h->dRowptr; p.colidx = h->dColidx;
  p.rowptrIn = h->dRowptrIn; p.colidxIn = h->dColidxIn;
  p.perm = h->hasPerm ? h->dPerm : nullptr;
  p.iperm = h->hasPerm ? h->dIperm : nullptr;
  p.nSweepWords = h->nSweepWords; p.nIsoInSweep = h->nIsoInSweep; p.isoBits = h->dIso;
  {  // source inside the hub's component: everything outside starts out visited (zero-degree vertices are outside too)
    const uint32_t is = h->hasPerm ? h->perm[src] : src;
    if (h->dOutside && ((h->hubComp[is >> 5] >> (is & 31u)) & 1u)) {
      p.isoBits = h->dOutside;
      p.nIsoInSweep = h->nOutsideInSweep;
    }
  }
  p.V = h->dV; p.F[0] = h->dF[0]; p.F[1] = h->dF[1]; p.F[2] = h->dF[2];
  p.WL[0] = h->dWL[0]; p.WL[1] = h->dWL[1];
  p.chunks = h->dChunks; p.chunkCap = h->chunkCap;
  p.head = h->dHead; p.deg = h->dDeg; p.popThr = h->dPopThr;
  p.Q[0] = h->dQ[0]; p.Q[1] = h->dQ[1];
  p.out = devOut ? levels_out : h->dOut;
  p.L = h->hasPerm ? h->dL : p.out;
  p.stamp = h->dStamp;
  p.hostStatus = h->hStatus;
  p.trace = h->opt.trace != 2 ? h->dTrace : nullptr;
  p.traceCap = TRACE_CAP;
  p.src = h->hasPerm ? h->perm[src] : src;
  p.srcOrig = src;
  {  // switch cost model, ps per unit (fitted to per-level traces on the B200); reserved[1..5] override (x0.01)
    const float dflt[5] = {COST_TD_EDGE, COST_TD_VERTEX, COST_BU_VERTEX, COST_BU_SCAN, COST_BU_WORD};
    float* dst[5] = {&p.cTdEdge, &p.cTdVertex, &p.cBuVertex, &p.cBuScan, &p.cBuWord};
    for (int k = 0; k < 5; ++k) *dst[k] = h->opt.reserved[1 + k] > 0 ? 0.01f * (float)h->opt.reserved[1 + k] : dflt[k];
    p.cTdWord = COST_TD_WORD;
    p.cTdNew = COST_TD_NEW;
    p.scanExp = h->hubby ? 0.5f : 1.0f;
    p.hubFilter = h->hubby ? 1 : 0;
  }
  p.switching = h->opt.switching;
  p.contraction = h->opt.contraction ? h->opt.contraction : 1;  // auto -> ALU (measured fastest)
  p.buMask = (uint32_t)h->opt.reserved[0];
  p.tmaTiles = h->opt.tune[0] == 1;
  p.eta = h->opt.eta;
  p.gamma = h->opt.gamma;
  p.srcPremarked = (p.isoBits == h->dIso) ? (int)((h->isoBits[p.src >> 5] >> (p.src & 31u)) & 1u) : 0;
  if ((h->deadSrc[p.src >> 5] >> (p.src & 31u)) & 1u) {
    h->lastCtrl = nullptr;
    CK(launch_isolated_source(p.out, h->n, src, st));  // nothing to traverse
  } else if (resolved_kernel(h) == 1) {
    persist_use(h, 0);
    p.ctrl = h->dCtrl;
    h->lastCtrl = h->dCtrl;
    CK(cudaMemsetAsync(h->dCtrl, 0, sizeof(Ctrl), st));
    CK(launch_bfs_eager(p, h->gridEager, st));
  } else {
    // levels_out is written once per discovered vertex at a scattered (original-id) position when the graph was
    // reordered: keep its lines in L2 for the duration of the call (persisting access-policy window of the launch),
    // so that those 4-byte writes merge there instead of each costing DRAM a sector.  Measured on C4: -5..10 % per BFS.
    const size_t bytes = (size_t)h->n * 4;
    const bool usePersist = h->persistRef && persist_fits(h, bytes);
    // reordered graph: levels scattered straight into levels_out when L2 can hold it, else internal array + gather pass
    p.gather = h->hasPerm && !usePersist;
    p.lvl = p.gather ? h->dL : p.out;
    p.ipermW = (h->hasPerm && !p.gather) ? h->dIperm : nullptr;
    p.srcLvl = p.gather ? p.src : src;
    // level guess: only when everything the traversal cannot reach is known (source inside the labelled component), as
    // a bitmap over the indices of p.lvl; options.tune[2] = 1 switches it off
    p.negBits = nullptr;
    if (p.isoBits == h->dOutside && h->dOutside && h->opt.tune[2] != 1)
      p.negBits = (h->hasPerm && !p.gather) ? h->dOutsideOrig : h->dOutside;
    p.ctrl = h->dCtrlLazy;  // self-resetting: no memset node before the launch
    h->lastCtrl = h->dCtrlLazy;
    persist_use(h, usePersist ? bytes : 0);
    const cudaError_t le = launch_bfs_lazy(p, h->gridLazy, st, usePersist ? (const void*)p.out : nullptr, usePersist ? bytes : 0,
                                           usePersist ? (float)std::min(1.0, (double)persist_max(h) / (double)bytes) : 0.f);
    CK(le);
  }
  if (!devOut) CK(cudaMemcpyAsync(levels_out, h->dOut, (size_t)h->n * 4, cudaMemcpyDeviceToHost, st));
  return BLEST_OK;
}

int blest_get_trace(blest_handle_t h, blest_level_trace_t* buf, uint32_t cap, uint32_t* n_levels) {
  if (!h || !n_levels) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  CK(cudaDeviceSynchronize());
  Ctrl c{};
  if (h->lastCtrl) CK(cudaMemcpy(&c, h->lastCtrl, sizeof(Ctrl), cudaMemcpyDeviceToHost));
  *n_levels = c.nlevels;
  const uint32_t k = std::min(std::min(cap, c.nlevels), TRACE_CAP);
  if (buf && k) CK(cudaMemcpy(buf, h->dTrace, (size_t)k * sizeof(blest_level_trace_t), cudaMemcpyDeviceToHost));
  return (c.error & 1u) ? BLEST_EOVERFLOW : BLEST_OK;
}

int blest_get_call_stats(blest_handle_t h, uint64_t* init_ns, uint64_t* levels_ns) {
  if (!h) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  CK(cudaDeviceSynchronize());
  Ctrl c{};
  if (h->lastCtrl) CK(cudaMemcpy(&c, h->lastCtrl, sizeof(Ctrl), cudaMemcpyDeviceToHost));
  if (init_ns) *init_ns = c.tInit;
  if (levels_ns) {
    *levels_ns = 0;
    if (c.nlevels) {
      blest_level_trace_t last;
      CK(cudaMemcpy(&last, h->dTrace + std::min(c.nlevels, TRACE_CAP) - 1, sizeof(last), cudaMemcpyDeviceToHost));
      *levels_ns = last.t_ns;
    }
  }
  return BLEST_OK;
}

static int ensure_ms_workspace(blest_graph* g) {
  persist_use(g, 0);  // the multi-source state wants the whole L2
  const uint64_t words = (uint64_t)g->rho * 8u * (g->opt.kappa / 32) + 4;
  int rc;
  if (words > g->msWords) {
    // grow-only: a wider kappa than any used before replaces the three state arrays (the old ones may still be in use
    // by enqueued work, hence the synchronisation -- this happens at most three times in a handle's life)
    if (g->dMsF) {
      CK(cudaDeviceSynchronize());
      for (uint32_t* old : {g->dMsF, g->dMsVc, g->dMsVn, g->dMsF2}) {
        auto it = std::find(g->allocs.begin(), g->allocs.end(), (void*)old);
        if (it != g->allocs.end()) g->allocs.erase(it);
        cudaFree(old);
      }
      g->wsBytes -= 4 * ((g->msWords * 4 + 15) & ~15ull);
      g->dMsF = g->dMsVc = g->dMsVn = g->dMsF2 = nullptr;
      g->msWords = 0;
    }
    if ((rc = dev_alloc(g, &g->dMsF, words, true))) return rc;
    if ((rc = dev_alloc(g, &g->dMsVc, words, true))) return rc;
    if ((rc = dev_alloc(g, &g->dMsVn, words, true))) return rc;
    if ((rc = dev_alloc(g, &g->dMsF2, words, true))) return rc;
    g->msWords = words;
  }
  if (!g->dDirty && (rc = dev_alloc(g, &g->dDirty, (uint64_t)g->Ns + 16, true))) return rc;
  if (!g->dFarT && (rc = dev_alloc(g, &g->dFarT, (uint64_t)g->rho * 8u, true))) return rc;
  if (!g->dReachT && (rc = dev_alloc(g, &g->dReachT, (uint64_t)g->rho * 8u, true))) return rc;
  if (!g->dMsStats && (rc = dev_alloc(g, &g->dMsStats, MS_STATS_WORDS, true))) return rc;
  if (!g->dMsLive && (rc = dev_alloc(g, &g->dMsLive, 24, true))) return rc;
  return BLEST_OK;
}

static void fill_ms_params(blest_graph* h, MsParams& p) {
  p.n = h->n; p.Ns = h->Ns; p.rho = h->rho; p.qcap = h->qcap; p.nQuads = h->nQuads;
  p.setPtr = h->dSetPtr; p.rowIds = reinterpret_cast<const uint4*>(h->dRowIds); p.masks = h->dMasks;
  p.perm = h->hasPerm ? h->dPerm : nullptr;
  p.iperm = h->hasPerm ? h->dIperm : nullptr;
  p.F = h->dMsF; p.Vc = h->dMsVc; p.Vn = h->dMsVn; p.dirty = h->dDirty;
  p.Q[0] = h->dQ[0]; p.Q[1] = h->dQ[1];
  p.ctrl = h->dCtrl;
  p.hostStatus = h->hStatus;
  p.kappa = h->opt.kappa;
  p.stats = h->opt.trace != 2 ? h->dMsStats : nullptr;
  // pull levels (target-side accumulation on a symmetric graph only; the kernel checks the rest): a batch switches when a
  // level's queue holds at least half of all VSSs, i.e. the frontier touches most slice sets; options.tune[1] = 1: never
  p.F2 = h->dMsF2; p.rowptr = h->dRowptr; p.colidx = h->dColidx; p.live = h->dMsLive;
  p.pullMin = (h->opt.tune[1] == 1 || h->directed) ? 0u : std::max(1u, h->Nv / 2u);
}

// ---- concurrent lanes -------------------------------------------------------------------------------------------------
// Source batches are independent (PAPER.md:678 partitions them over GPUs); on ONE GPU the persistent kernel does not need
// the whole grid either: measured on config 5 (kappa = 64), the same launch on 74 of the 148 SMs is only 1.30 x slower and
// on 37 SMs 1.88 x (57 % of the warp samples of the full-grid launch wait at a grid barrier: small levels, stragglers).
// Closeness / farness calls therefore split their batches over up to `lanes` cooperative launches of gridMs / lanes CTAs
// each, on separate streams forked from and joined into the caller's stream by events: while one lane sits in a barrier
// or a small level, the SMs of the others are busy.  Every lane has its own per-launch arrays; the target-side sums of
// lanes 1.. are added to lane 0's afterwards.  Cooperative grids are scheduled whole, so the lanes cannot deadlock on each
// other's barriers.  options.tune[3]: 0 = 8 lanes, k = k lanes (1..16; 1 = the single full-grid launch).
static int ms_lane_count(const blest_graph* h, uint64_t batches) {
  int want = h->opt.tune[3] > 0 ? h->opt.tune[3] : 8;
  want = std::max(1, std::min(want, 16));
  want = (int)std::min<uint64_t>((uint64_t)want, std::max<uint64_t>(batches, 1));
  want = std::min(want, std::max(1, h->gridMs));
  // per-lane workspace: two work queues + four state arrays; keep the extra lanes below 4 GiB in total
  const uint64_t perLane = (uint64_t)h->qcap * 16u + 4u * h->msWords * 4u + (uint64_t)h->rho * 8u * 12u;
  while (want > 1 && perLane * (uint64_t)(want - 1) > (4ull << 30)) --want;
  return want;
}

static int ensure_ms_lanes(blest_graph* g, int lanes) {
  int rc;
  if (!g->msFork) CK(cudaEventCreateWithFlags(&g->msFork, cudaEventDisableTiming));
  if ((int)g->msLanes.size() < lanes - 1) g->msLanes.resize((size_t)lanes - 1);
  for (int i = 0; i < lanes - 1; ++i) {
    blest_graph::MsLane& ln = g->msLanes[(size_t)i];
    if (!ln.st) CK(cudaStreamCreateWithFlags(&ln.st, cudaStreamNonBlocking));
    if (!ln.done) CK(cudaEventCreateWithFlags(&ln.done, cudaEventDisableTiming));
    if (ln.words < g->msWords) {  // (a wider kappa: ensure_ms_workspace has synchronised the device already)
      for (uint32_t** a : {&ln.F, &ln.F2, &ln.Vc, &ln.Vn}) {
        if (*a) {
          auto it = std::find(g->allocs.begin(), g->allocs.end(), (void*)*a);
          if (it != g->allocs.end()) g->allocs.erase(it);
          cudaFree(*a);
          g->wsBytes -= (ln.words * 4 + 15) & ~15ull;
          *a = nullptr;
        }
        if ((rc = dev_alloc(g, a, g->msWords, true))) return rc;
      }
      ln.words = g->msWords;
    }
    if (!ln.dirty && (rc = dev_alloc(g, &ln.dirty, (uint64_t)g->Ns + 16, true))) return rc;
    if (!ln.live && (rc = dev_alloc(g, &ln.live, 24, true))) return rc;
    for (int q = 0; q < 2; ++q)
      if (!ln.Q[q] && (rc = dev_alloc(g, &ln.Q[q], (uint64_t)g->qcap))) return rc;
    if (!ln.ctrl && (rc = dev_alloc(g, &ln.ctrl, 1, true))) return rc;
    if (!ln.farT && (rc = dev_alloc(g, &ln.farT, (uint64_t)g->rho * 8u, true))) return rc;
    if (!ln.reachT && (rc = dev_alloc(g, &ln.reachT, (uint64_t)g->rho * 8u, true))) return rc;
    if (!ln.stats && (rc = dev_alloc(g, &ln.stats, MS_STATS_WORDS, true))) return rc;
  }
  return BLEST_OK;
}

// The multi-source kernel over p.nsrcs sources (p = lane 0's arrays, outputs and source range), split over lanes.
// Enqueues only.  The caller has cleared p.farT / p.reachT / p.farS / p.reachS on `st`.
static cudaError_t launch_ms_lanes(blest_graph* h, const MsParams& p, cudaStream_t st) {
  const uint64_t kappa = (uint64_t)p.kappa, batches = (p.nsrcs + kappa - 1) / kappa;
  int lanes = ms_lane_count(h, batches);
  if (lanes > 1 && ensure_ms_lanes(h, lanes) != BLEST_OK) {
    cudaGetLastError();
    lanes = 1;  // no memory for a second workspace: the single full-grid launch
  }
  h->msLanesUsed = lanes;
  cudaError_t e = cudaSuccess;
  if (lanes > 1) e = cudaEventRecord(h->msFork, st);
  const int grid = std::max(1, h->gridMs / lanes);
  for (int i = 0; i < lanes && e == cudaSuccess; ++i) {
    const uint64_t b0 = batches * (uint64_t)i / (uint64_t)lanes, b1 = batches * (uint64_t)(i + 1) / (uint64_t)lanes;
    const uint64_t first = b0 * kappa, end = std::min<uint64_t>(p.nsrcs, b1 * kappa);
    MsParams q = p;
    q.srcBase = p.srcBase + first;
    q.nsrcs = end - first;
    if (p.srcs) q.srcs = p.srcs + first;
    if (p.farS) q.farS = p.farS + first;
    if (p.reachS) q.reachS = p.reachS + first;
    cudaStream_t s = st;
    if (i > 0) {
      blest_graph::MsLane& ln = h->msLanes[(size_t)i - 1];
      s = ln.st;
      q.F = ln.F; q.F2 = ln.F2; q.Vc = ln.Vc; q.Vn = ln.Vn; q.live = ln.live; q.dirty = ln.dirty;
      q.Q[0] = ln.Q[0]; q.Q[1] = ln.Q[1];
      q.ctrl = ln.ctrl;
      if (p.stats) q.stats = ln.stats;
      if (p.farT) q.farT = ln.farT;
      if (p.reachT) q.reachT = ln.reachT;
      e = cudaStreamWaitEvent(s, h->msFork, 0);
      if (e == cudaSuccess && p.farT) e = cudaMemsetAsync(ln.farT, 0, (size_t)h->rho * 8u * 8u, s);
      if (e == cudaSuccess && p.reachT) e = cudaMemsetAsync(ln.reachT, 0, (size_t)h->rho * 8u * 4u, s);
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(q.ctrl, 0, sizeof(Ctrl), s);
    if (e == cudaSuccess) e = cudaMemsetAsync(i > 0 ? h->msLanes[(size_t)i - 1].stats : h->dMsStats, 0,
                                              MS_STATS_WORDS * sizeof(unsigned long long), s);
    if (e == cudaSuccess && q.nsrcs) e = launch_msbfs(q, i == 0 && lanes == 1 ? h->gridMs : grid, s);
    if (e == cudaSuccess && i > 0) e = cudaEventRecord(h->msLanes[(size_t)i - 1].done, s);
  }
  for (int i = 1; i < lanes && e == cudaSuccess; ++i) {
    blest_graph::MsLane& ln = h->msLanes[(size_t)i - 1];
    e = cudaStreamWaitEvent(st, ln.done, 0);
    if (e == cudaSuccess && (p.farT || p.reachT))
      e = launch_add_partial_sums(p.farT, p.reachT, p.farT ? ln.farT : nullptr, p.reachT ? ln.reachT : nullptr,
                                  (uint64_t)h->rho * 8u, st);
  }
  return e;
}

// Stream-ordered temporaries of one multi-source call: device buffers from the stream's memory pool
// (cudaMallocAsync / cudaFreeAsync: no host block), the caller's `srcs` copied through a pinned staging slot.
struct MsTemps {
  cudaStream_t st;
  std::vector<void*> dev;
  cudaError_t alloc(void** p, size_t bytes) {
    cudaError_t e = cudaMallocAsync(p, std::max<size_t>(bytes, 16), st);
    if (e == cudaSuccess) dev.push_back(*p);
    return e;
  }
  void release() {
    for (void* p : dev) cudaFreeAsync(p, st);
    dev.clear();
  }
};

// Copy `count` source ids to the device without blocking: host -> pinned slot (now), pinned -> device (on the stream).
// A slot is reused once the copy that read it has executed (event query); a new one is made when none is free.
static cudaError_t stage_srcs(blest_graph* h, const uint32_t* srcs, uint64_t count, uint32_t* dDst, cudaStream_t st) {
  const size_t bytes = (size_t)count * 4;
  blest_graph::StageSlot* slot = nullptr;
  for (auto& sl : h->stage)
    if (sl.cap >= bytes && cudaEventQuery(sl.ev) == cudaSuccess) { slot = &sl; break; }
  cudaGetLastError();  // cudaErrorNotReady of a busy slot is not an error
  if (!slot) {
    if (h->stage.size() >= 16) {  // bounded: wait for the oldest copy instead of growing without limit
      blest_graph::StageSlot old = h->stage.front();
      h->stage.erase(h->stage.begin());
      cudaEventSynchronize(old.ev);
      cudaEventDestroy(old.ev);
      cudaFreeHost(old.host);
    }
    blest_graph::StageSlot sl;
    sl.cap = std::max<size_t>(bytes, 4096);
    cudaError_t e = cudaHostAlloc(&sl.host, sl.cap, cudaHostAllocDefault);
    if (e != cudaSuccess) return e;
    e = cudaEventCreateWithFlags(&sl.ev, cudaEventDisableTiming);
    if (e != cudaSuccess) { cudaFreeHost(sl.host); return e; }
    h->stage.push_back(sl);
    slot = &h->stage.back();
  }
  std::memcpy(slot->host, srcs, bytes);
  cudaError_t e = cudaMemcpyAsync(dDst, slot->host, bytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaEventRecord(slot->ev, st);
  return e;
}

static int ms_fail(cudaError_t e) {
  g_lastCuda = (int)e;
  cudaGetLastError();
  return e == cudaErrorMemoryAllocation ? BLEST_ENOMEM : BLEST_ECUDA;
}

int blest_msbfs(blest_handle_t h, const uint32_t* srcs, uint32_t k, int32_t* levels_out, void* cuda_stream) {
  if (!h || !srcs || !levels_out || k == 0) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  for (uint32_t i = 0; i < k; ++i)
    if (srcs[i] >= h->n) return BLEST_EINVAL;
  if (int rc = pending_status(h)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_ms_workspace(h);
  if (rc) return rc;
  const bool devOut = is_device_ptr(levels_out);
  MsTemps tmp{st, {}};
  uint32_t* dSrcs = nullptr;
  int32_t* dLevels = nullptr;
  cudaError_t e = tmp.alloc((void**)&dSrcs, (size_t)k * 4);
  if (e == cudaSuccess && !devOut) e = tmp.alloc((void**)&dLevels, (size_t)k * h->n * 4);
  if (e == cudaSuccess) e = stage_srcs(h, srcs, k, dSrcs, st);
  MsParams p{};
  fill_ms_params(h, p);
  p.srcs = dSrcs;
  p.nsrcs = k;
  p.levels = devOut ? levels_out : dLevels;
  h->lastCtrl = h->dCtrl;
  if (e == cudaSuccess) e = cudaMemsetAsync(h->dCtrl, 0, sizeof(Ctrl), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->dMsStats, 0, MS_STATS_WORDS * sizeof(unsigned long long), st);
  h->msLanesUsed = 1;
  if (e == cudaSuccess) e = launch_msbfs(p, h->gridMs, st);
  if (e == cudaSuccess && !devOut)
    e = cudaMemcpyAsync(levels_out, dLevels, (size_t)k * h->n * 4, cudaMemcpyDeviceToHost, st);
  tmp.release();  // stream-ordered: the buffers live until the work enqueued above has run
  if (e != cudaSuccess) return ms_fail(e);
  return BLEST_OK;
}

static int closeness_impl(blest_handle_t h, const uint32_t* srcs, uint64_t n_srcs, double* cc, uint64_t* farOut,
                          uint32_t* reachOut, void* cuda_stream) {
  if (!h || n_srcs == 0) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  if (!cc && !farOut && !reachOut) return BLEST_EINVAL;
  if (!srcs && n_srcs != h->n) return BLEST_EINVAL;
  if (srcs)
    for (uint64_t i = 0; i < n_srcs; ++i)
      if (srcs[i] >= h->n) return BLEST_EINVAL;
  if (int rc = pending_status(h)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_ms_workspace(h);
  if (rc) return rc;
  uint32_t* dSrcs = nullptr;
  unsigned long long *dFarS = nullptr, *dFarO = nullptr;
  uint32_t *dReachS = nullptr, *dReachO = nullptr;
  double* dCc = nullptr;
  MsTemps tmp{st, {}};
  cudaError_t e = cudaSuccess;
  const bool ccDev = cc && is_device_ptr(cc), farDev = farOut && is_device_ptr(farOut), reachDev = reachOut && is_device_ptr(reachOut);
  MsParams p{};
  fill_ms_params(h, p);
  p.nsrcs = n_srcs;
  if (srcs || h->directed) {
    // arbitrary subset: per-source counts (reading R13).  Also every run on a DIRECTED graph: the target-side sums of
    // Eq. 7 are the farness of the reached vertex only when d(s, u) = d(u, s).
    if (srcs) e = tmp.alloc((void**)&dSrcs, n_srcs * 4);
    if (e == cudaSuccess) e = tmp.alloc((void**)&dFarS, n_srcs * 8);
    if (e == cudaSuccess) e = tmp.alloc((void**)&dReachS, n_srcs * 4);
    if (e == cudaSuccess && srcs) e = stage_srcs(h, srcs, n_srcs, dSrcs, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(dFarS, 0, n_srcs * 8, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(dReachS, 0, n_srcs * 4, st);
    p.srcs = dSrcs;
    p.farS = dFarS;
    p.reachS = dReachS;
  } else {  // all vertices: the paper's target-side accumulation (Eq. 7)
    e = cudaMemsetAsync(h->dFarT, 0, (size_t)h->rho * 8u * 8u, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->dReachT, 0, (size_t)h->rho * 8u * 4u, st);
    p.farT = h->dFarT;
    p.reachT = h->dReachT;
  }
  if (e == cudaSuccess && cc && !ccDev) e = tmp.alloc((void**)&dCc, n_srcs * 8);
  if (e == cudaSuccess && farOut && !farDev) e = tmp.alloc((void**)&dFarO, n_srcs * 8);
  if (e == cudaSuccess && reachOut && !reachDev) e = tmp.alloc((void**)&dReachO, n_srcs * 4);
  h->lastCtrl = h->dCtrl;
  if (e == cudaSuccess) e = launch_ms_lanes(h, p, st);
  if (e == cudaSuccess)
    e = launch_closeness_finalize(h->n, h->rho, h->hasPerm ? h->dPerm : nullptr, p.farT, p.reachT, p.farS, p.reachS, n_srcs,
                                  cc ? (ccDev ? cc : dCc) : nullptr,
                                  farOut ? (farDev ? (unsigned long long*)farOut : dFarO) : nullptr,
                                  reachOut ? (reachDev ? reachOut : dReachO) : nullptr, st);
  if (e == cudaSuccess && cc && !ccDev) e = cudaMemcpyAsync(cc, dCc, n_srcs * 8, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && farOut && !farDev) e = cudaMemcpyAsync(farOut, dFarO, n_srcs * 8, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && reachOut && !reachDev) e = cudaMemcpyAsync(reachOut, dReachO, n_srcs * 4, cudaMemcpyDeviceToHost, st);
  tmp.release();  // stream-ordered
  if (e != cudaSuccess) return ms_fail(e);
  return BLEST_OK;
}

int blest_farness_partial(blest_handle_t h, uint32_t first, uint32_t count, uint64_t* far_sum, uint32_t* reach_sum,
                          void* cuda_stream) {
  if (!h || !far_sum || !reach_sum || count == 0) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  if ((uint64_t)first + count > h->n) return BLEST_EINVAL;
  if (h->directed) return BLEST_EUNSUPPORTED;  // target-side sums need d(s, u) = d(u, s)
  if (!is_device_ptr(far_sum) || !is_device_ptr(reach_sum)) return BLEST_EINVAL;
  if (int rc = pending_status(h)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_ms_workspace(h);
  if (rc) return rc;
  MsParams p{};
  fill_ms_params(h, p);
  p.srcBase = first;
  p.nsrcs = count;
  p.farT = h->dFarT;
  p.reachT = h->dReachT;
  h->lastCtrl = h->dCtrl;
  cudaError_t e = cudaMemsetAsync(h->dFarT, 0, (size_t)h->rho * 8u * 8u, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->dReachT, 0, (size_t)h->rho * 8u * 4u, st);
  if (e == cudaSuccess) e = launch_ms_lanes(h, p, st);
  // target-side sums in ORIGINAL vertex ids (the finalize kernel maps id -> getVI(perm[id]))
  if (e == cudaSuccess)
    e = launch_closeness_finalize(h->n, h->rho, h->hasPerm ? h->dPerm : nullptr, p.farT, p.reachT, nullptr, nullptr, h->n,
                                  nullptr, (unsigned long long*)far_sum, reach_sum, st);
  if (e != cudaSuccess) return ms_fail(e);
  return BLEST_OK;
}

int blest_closeness_from_sums(const uint64_t* far_sum, const uint32_t* reach_sum, uint64_t n, double* out, void* cuda_stream) {
  if (!far_sum || !reach_sum || !out || n == 0) return BLEST_EINVAL;
  if (!is_device_ptr(far_sum) || !is_device_ptr(reach_sum) || !is_device_ptr(out)) return BLEST_EINVAL;
  cudaError_t e = launch_closeness_finalize((uint32_t)std::min<uint64_t>(n, 0xFFFFFFFFull), 0, nullptr, nullptr, nullptr,
                                            (const unsigned long long*)far_sum, reach_sum, n, out, nullptr, nullptr,
                                            (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return ms_fail(e);
  return BLEST_OK;
}

int blest_closeness_noalloc(blest_handle_t h, const uint32_t* srcs_dev, uint32_t n_srcs, double* out_dev, void* cuda_stream) {
  if (!h || !srcs_dev || !out_dev || n_srcs == 0) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  // limits of the file-scope scratch (msbfs_kernels.cu): rejected, never truncated
  const uint64_t stateBytes = (uint64_t)h->rho * 8u * (uint64_t)(h->opt.kappa / 32) * 4u;  // exactly what the kernel touches
  if (n_srcs > NOALLOC_MAX_SRCS || stateBytes > NOALLOC_MAX_STATE_BYTES || h->Ns > NOALLOC_MAX_SETS) return BLEST_ERANGE;
  if (!is_device_ptr(srcs_dev) || !is_device_ptr(out_dev)) return BLEST_EINVAL;
  if (int rc = pending_status(h)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  persist_use(h, 0);  // (a device limit, not an allocation; only handles that hold a reference touch it)
  MsParams p{};
  fill_ms_params(h, p);  // graph arrays, work queues and control block of the handle: allocated by blest_build
  h->lastCtrl = h->dCtrl;
  cudaError_t e = cudaMemsetAsync(h->dCtrl, 0, sizeof(Ctrl), st);
  h->msLanesUsed = 1;
  if (e == cudaSuccess) e = launch_closeness_noalloc(p, srcs_dev, n_srcs, h->gridMs, out_dev, st);
  if (e != cudaSuccess) return ms_fail(e);
  return BLEST_OK;
}

int blest_noalloc_limits(uint32_t* max_srcs, uint64_t* max_state_bytes, uint64_t* max_vertices_at_kappa64) {
  if (max_srcs) *max_srcs = NOALLOC_MAX_SRCS;
  if (max_state_bytes) *max_state_bytes = NOALLOC_MAX_STATE_BYTES;
  if (max_vertices_at_kappa64) *max_vertices_at_kappa64 = NOALLOC_MAX_STATE_BYTES / 8u;
  return BLEST_OK;
}

int blest_get_ms_stats(blest_handle_t h, uint64_t* out8) {
  if (!h || !out8) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  for (int k = 0; k < 8; ++k) out8[k] = 0;
  if (!h->dMsStats) return BLEST_OK;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(out8, h->dMsStats, 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  for (int i = 1; i < h->msLanesUsed && (size_t)i - 1 < h->msLanes.size(); ++i) {  // totals over the lanes of the launch
    uint64_t t[8];
    CK(cudaMemcpy(t, h->msLanes[(size_t)i - 1].stats, 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
    for (int k = 0; k < 8; ++k) out8[k] += t[k];
  }
  return BLEST_OK;
}

int blest_get_ms_phases(blest_handle_t h, uint64_t* out8) {
  if (!h || !out8) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  for (int k = 0; k < 8; ++k) out8[k] = 0;
  if (!h->dMsStats) return BLEST_OK;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(out8, h->dMsStats + 8, 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  for (int i = 1; i < h->msLanesUsed && (size_t)i - 1 < h->msLanes.size(); ++i) {  // times: lane 0's; pull counters: totals
    uint64_t t[8];
    CK(cudaMemcpy(t, h->msLanes[(size_t)i - 1].stats + 8, 8 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
    out8[5] += t[5];
    out8[6] += t[6];
  }
  return BLEST_OK;
}

int blest_get_ms_level_trace(blest_handle_t h, uint64_t* out, uint32_t max_levels, uint32_t* n_levels) {
  if (!h || !out || !n_levels) return BLEST_EINVAL;
  if (h->hostOnly) return BLEST_EUNSUPPORTED;
  *n_levels = 0;
  if (!h->dMsStats) return BLEST_OK;
  CK(cudaDeviceSynchronize());
  std::vector<uint64_t> buf(MS_STATS_WORDS);
  CK(cudaMemcpy(buf.data(), h->dMsStats, MS_STATS_WORDS * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  const uint32_t have = (uint32_t)std::min<uint64_t>(buf[5], MS_TRACE_LEVELS), k = std::min(have, max_levels);
  for (uint32_t i = 0; i < 4 * k; ++i) out[i] = buf[16 + i];
  *n_levels = k;
  return BLEST_OK;
}

int blest_closeness(blest_handle_t h, const uint32_t* srcs, uint64_t n_srcs, double* out, void* cuda_stream) {
  if (!out) return BLEST_EINVAL;
  return closeness_impl(h, srcs, n_srcs, out, nullptr, nullptr, cuda_stream);
}

int blest_farness(blest_handle_t h, const uint32_t* srcs, uint64_t n_srcs, uint64_t* far_out, uint32_t* reach_out,
                  void* cuda_stream) {
  return closeness_impl(h, srcs, n_srcs, nullptr, far_out, reach_out, cuda_stream);
}

int blest_get_array(blest_handle_t h, int which, void* host_dst, uint64_t bytes) {
  if (!h || !host_dst) return BLEST_EINVAL;
  const void* src = nullptr;
  uint64_t want = 0;
  bool onHost = false;
  switch (which) {
    case 0: src = h->dSetPtr; want = ((uint64_t)h->Ns + 1) * 4; break;
    case 1: src = h->dRowIds; want = h->nQuads * 16; break;
    case 2: src = h->dMasks; want = h->nQuads * 4; break;
    case 3: src = h->realPtrs.data(); want = ((uint64_t)h->Ns + 1) * 4; onHost = true; break;
    case 4: src = h->virtualToReal.data(); want = (uint64_t)h->Nv * 4; onHost = true; break;
    case 5: if (!h->hasPerm) return BLEST_EINVAL; src = h->perm.data(); want = (uint64_t)h->n * 4; onHost = true; break;
    case 6: if (!h->hasPerm) return BLEST_EINVAL; src = h->iperm.data(); want = (uint64_t)h->n * 4; onHost = true; break;
    case 7: src = h->dRowptr; want = ((uint64_t)h->n + 1) * 4; break;
    case 8: src = h->dColidx; want = h->nnz * 4; break;
    default: return BLEST_EINVAL;
  }
  if (h->hostOnly) {
    onHost = true;
    switch (which) {
      case 0: src = h->hb.setPtr.data(); break;
      case 1: src = h->hb.rowIds.data(); break;
      case 2: src = h->hb.masks.data(); break;
      case 7: src = h->hcsr.rowptr.data(); break;
      case 8: src = h->hcsr.colidx.data(); break;
      default: break;
    }
  }
  if (bytes != want) return BLEST_EINVAL;
  if (want == 0) return BLEST_OK;
  if (onHost) std::memcpy(host_dst, src, want);
  else CK(cudaMemcpy(host_dst, src, want, cudaMemcpyDeviceToHost));
  return BLEST_OK;
}

int blest_contraction_selftest(int contraction, uint64_t* n_mismatch) {
  if (!n_mismatch || contraction < 1 || contraction > 3) return BLEST_EINVAL;
  unsigned long long* d = nullptr;
  CK(cudaMalloc((void**)&d, 8));
  cudaError_t e = cudaMemset(d, 0, 8);
  if (e == cudaSuccess) e = run_contraction_selftest(contraction, d);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  unsigned long long v = 0;
  if (e == cudaSuccess) e = cudaMemcpy(&v, d, 8, cudaMemcpyDeviceToHost);
  cudaFree(d);
  CK(e);
  *n_mismatch = v;
  return BLEST_OK;
}

int blest_tcgen05_microbench(uint32_t iters, uint32_t n, double* tera_macs_per_s, uint64_t* n_wrong) {
  if (!tera_macs_per_s || !n_wrong || iters == 0 || n < 16 || n > 256 || (n & 15u)) return BLEST_EINVAL;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  unsigned int* dBad = nullptr;
  CK(cudaMalloc((void**)&dBad, 4));
  cudaError_t e = cudaMemset(dBad, 0, 4);
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  double macs = 0;
  if (e == cudaSuccess) e = run_tcgen05_peak(iters, n, sms, dBad, &macs);  // warm-up (and the correctness check)
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  float best = 1e30f;
  for (int rep = 0; rep < 5 && e == cudaSuccess; ++rep) {
    cudaEventRecord(a);
    e = run_tcgen05_peak(iters, n, sms, dBad, &macs);
    cudaEventRecord(b);
    if (e == cudaSuccess) e = cudaEventSynchronize(b);
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    best = std::min(best, ms);
  }
  unsigned int bad = 0;
  if (e == cudaSuccess) e = cudaMemcpy(&bad, dBad, 4, cudaMemcpyDeviceToHost);
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(dBad);
  CK(e);
  *tera_macs_per_s = macs / (best * 1e-3) / 1e12;
  *n_wrong = bad;
  return BLEST_OK;
}

int blest_mma_microbench(int kind, uint32_t iters, double* tera_macs_per_s, double* milliseconds) {
  if (!tera_macs_per_s || (kind != 2 && kind != 3) || iters == 0) return BLEST_EINVAL;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  int* dSink = nullptr;
  CK(cudaMalloc((void**)&dSink, 4));
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  double macs = 0;
  cudaError_t e = run_mma_peak(kind, iters, sms, dSink, &macs);  // warm-up
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  float best = 1e30f;
  for (int rep = 0; rep < 5 && e == cudaSuccess; ++rep) {
    cudaEventRecord(a);
    e = run_mma_peak(kind, iters, sms, dSink, &macs);
    cudaEventRecord(b);
    if (e == cudaSuccess) e = cudaEventSynchronize(b);
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    best = std::min(best, ms);
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(dSink);
  CK(e);
  *tera_macs_per_s = macs / (best * 1e-3) / 1e12;
  if (milliseconds) *milliseconds = best;
  return BLEST_OK;
}

int blest_l2_microbench(uint64_t bytes, uint32_t iters, double* gb_per_s) {
  if (!gb_per_s || iters == 0 || bytes < 4096) return BLEST_EINVAL;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const uint64_t n16 = bytes / 32;  // half the footprint is read, half written
  uint4 *a = nullptr, *b = nullptr;
  CK(cudaMalloc((void**)&a, n16 * 16));
  cudaError_t e = cudaMalloc((void**)&b, n16 * 16);
  if (e == cudaSuccess) e = cudaMemset(a, 1, n16 * 16);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  if (e == cudaSuccess) e = run_l2_copy(a, b, n16, 2, sms);  // warm-up: both buffers become L2-resident
  float best = 1e30f;
  for (int rep = 0; rep < 5 && e == cudaSuccess; ++rep) {
    cudaEventRecord(e0);
    e = run_l2_copy(a, b, n16, iters, sms);
    cudaEventRecord(e1);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    best = std::min(best, ms);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(a);
  if (b) cudaFree(b);
  CK(e);
  *gb_per_s = (double)n16 * 32.0 * iters / (best * 1e-3) / 1e9;
  return BLEST_OK;
}

int blest_cluster_microbench(int cluster_ctas, uint32_t iters, double* ns_per_barrier, double* ns_per_dsmem_load) {
  if (!ns_per_barrier || !ns_per_dsmem_load || iters == 0 || cluster_ctas < 1 || cluster_ctas > 16 ||
      (cluster_ctas & (cluster_ctas - 1)))
    return BLEST_EINVAL;
  unsigned long long* dOut = nullptr;
  CK(cudaMalloc((void**)&dOut, 24));
  cudaError_t e = cudaMemset(dOut, 0, 24);
  if (e == cudaSuccess) e = run_cluster_bench(cluster_ctas, iters, dOut);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  unsigned long long v[3] = {0, 0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(v, dOut, 24, cudaMemcpyDeviceToHost);
  cudaFree(dOut);
  CK(e);
  *ns_per_barrier = (double)v[0] / iters;
  *ns_per_dsmem_load = (double)v[1] / iters;
  return BLEST_OK;
}

int blest_barrier_microbench(uint32_t iters, double* ns_per_barrier) {
  if (!ns_per_barrier || iters == 0) return BLEST_EINVAL;
  int dev = 0, sms = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  unsigned int* dBar = nullptr;
  unsigned long long* dNs = nullptr;
  CK(cudaMalloc((void**)&dBar, 16));
  cudaError_t e = cudaMalloc((void**)&dNs, 8);
  if (e == cudaSuccess) e = cudaMemset(dBar, 0, 16);
  if (e == cudaSuccess) e = run_barrier_bench(dBar, iters, sms, dNs);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  unsigned long long ns = 0;
  if (e == cudaSuccess) e = cudaMemcpy(&ns, dNs, 8, cudaMemcpyDeviceToHost);
  cudaFree(dBar);
  if (dNs) cudaFree(dNs);
  CK(e);
  *ns_per_barrier = (double)ns / iters;
  return BLEST_OK;
}

}  // extern "C"
