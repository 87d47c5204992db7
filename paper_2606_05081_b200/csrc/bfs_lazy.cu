// bfs_lazy.cu -- single-source BLEST traversal with lazy vertex updates (Alg. 3, :345-455) and the
// per-level switch to CUDA-core paths (§5.3, Eq. 6, Alg. 4), as ONE persistent cooperative kernel per call
// (PAPER.md:464, :496).  DESIGN.md §5.2 explains every deviation from the listing; in short:
//
//   state     one visited bitmap V and three rotating frontier bitmaps (level l reads F[(l-1)%3], marks F[l%3] and
//             clears F[(l+1)%3]); the paper's V_next XOR V_curr is F[l%3] AND NOT V.
//   top-down  Stage 1 consumes the list of non-zero frontier WORDS produced by the previous finalisation, 32 words per
//             warp step.  Every newly active slice set takes either the slice path -- the pull
//             contraction over the set's BVSS quads -- or the CSR edges of its frontier vertices
//             (the CUDA-core top-down path of north_star (e)).  The segments of the 32 words are flattened with a warp
//             scan, so that all lanes work whatever the degrees are, and every lane keeps several independent
//             loads / bitmap probes in flight.  Hub segments are cut into equal chunks and spread over the grid in a
//             second, balanced phase.  Marks are filtered no-return atomic ORs.  Stage 2 is the
//             finalisation sweep: level written once per discovered vertex, counters, next word list.
//   bottom-up Alg. 4 fused with its finalisation: the warp that owns word w of the visited bitmap
//             decides all 32 bits, so V, F_next, levels and the counters are written in the same sweep (one grid
//             barrier per level).  The first two neighbours of every vertex are kept inline (`head`), so most
//             unvisited vertices are resolved by one coalesced 8-byte load and one or two bitmap probes.
//   switch    start of each level: estimated cost of the two directions from the counters of the previous
//             finalisation (#unvisited as in Eq. 6, plus degree sums), scaled by eta.
//   output    levels_out is pre-filled with -1 ("infinity", reading R1) and the level of a vertex is
//             written to levels_out[original id] at the moment it is finalised (A10 fused into A6 / Alg. 4) -- when
//             the array fits the persisting-L2 window; otherwise levels go to an internal-id array and a final
//             gather pass moves them (scattered writes that miss L2 cost DRAM a read-modify-write each).
#include <cstddef>
#include "bfs_kernels.cuh"

namespace blest {

namespace {

constexpr uint32_t FULL = 0xffffffffu;
constexpr uint32_t NONE = 0xffffffffu;

constexpr uint32_t BU_LIST = 512;   // per-warp list of unvisited vertices (sparse bottom-up groups)
constexpr uint32_t BU_BATCH = 256;  // vertices per bottom-up batch: 8 per lane in flight
constexpr uint32_t DLIST_CAP = 1024;  // finalisation: dense words a CTA pools before its warps share them
constexpr uint32_t TILE_QUADS = 64;  // balanced top-down phase: quads per TMA-staged slice tile (1 KB of row ids + 256 B of masks)
constexpr uint32_t HUB_BITS = 1u << 17;  // top-down: marks of the first 2^17 vertices are de-duplicated per CTA in shared memory

struct LazyShared {
  unsigned long long acc[6];
  unsigned long long ctl[4];  // control words of the level, read by one thread and broadcast
  uint32_t wlCnt;
  uint32_t wlBase;
  uint32_t buDecision;  // direction of the level, evaluated by the thread that read the control words
  unsigned long long tStage1;     // (leader) %globaltimer after the level's Stage-1 barrier
  unsigned int epoch;             // (thread 0) grid barriers executed on this control block
  unsigned long long degVisited;  // (thread 0) degree sum of the vertices visited so far: the switch's `mu`
  uint32_t guess;       // the level levels_out is pre-filled with (0 = none; see the kernel)
  uint32_t guessSlot;   // degree class of the source
  uint32_t bestLevel;   // (thread 0) the level that discovered the most vertices so far, and how many
  unsigned long long bestCount;
  // The two directions never run at the same time: the bottom-up lists share their memory with the slice tiles that
  // the balanced top-down phase stages by TMA bulk copies (td_phase_b).
  union {
    struct {
      uint32_t buFound[WARPS_PER_BLOCK][32];
      uint32_t buSlotU[WARPS_PER_BLOCK][32];
      uint32_t buSlotTag[WARPS_PER_BLOCK][32];
      uint32_t buList[WARPS_PER_BLOCK][BU_LIST];
    };
    struct {
      alignas(128) uint4 tileRows[WARPS_PER_BLOCK][2][TILE_QUADS];       // row ids of a tile: 4 slices per quad
      alignas(16) uint32_t tileMasks[WARPS_PER_BLOCK][2][TILE_QUADS + 8];  // its masks (+ alignment slack of the copy)
    };
  };
  unsigned long long tileBar[WARPS_PER_BLOCK][2];  // mbarriers of the two tile stages of every warp (never overlaid)
  uint32_t tilePhase[WARPS_PER_BLOCK];             // their parities, kept across levels (bit s = stage s)
  uint32_t wl[WL_STAGE];
  uint32_t dcount, dvalid;      // finalisation: dense words shared by the CTA's warps
  uint2 dlist[DLIST_CAP];       // (word id, new-frontier bits)
  uint32_t hub[HUB_BITS / 32];  // top-down Stage 1: low-id vertices this CTA has already marked in this level
};

// Per-LANE counters of one level: 32 bits each (a lane's share of a level is far below 2^32 vertices, edge endpoints or
// bytes; nnz < 2^32 bounds the degree sum), widened when the warp's values are added up -- five 64-bit counters per thread
// cost the persistent kernel ten of its 64 registers.  `unv` is signed: discoveries are subtracted from it.
struct Counters {
  uint32_t nnew = 0;
  int32_t unv = 0;
  uint32_t mf = 0, scanned = 0, qbytes = 0;
};

// warp shuffle reduce -> shared atomics -> one global atomic per block and counter
__device__ __forceinline__ void block_accumulate(LazyShared& sh, const Counters& c, Ctrl* ctrl, uint32_t ci) {
  unsigned long long v[5] = {c.nnew, (unsigned long long)(long long)c.unv, c.mf, c.scanned, c.qbytes};
#pragma unroll
  for (int k = 0; k < 5; ++k) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v[k] += __shfl_down_sync(FULL, v[k], d);
  }
  if ((threadIdx.x & 31) == 0) {
#pragma unroll
    for (int k = 0; k < 5; ++k)
      if (v[k]) atomicAdd(&sh.acc[k], v[k]);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (sh.acc[0]) atomicAdd(&ctrl->newcount[ci], sh.acc[0]);
    if (sh.acc[1]) atomicAdd(&ctrl->unvisited[ci], sh.acc[1]);
    if (sh.acc[2]) atomicAdd(&ctrl->mf[ci], sh.acc[2]);
    if (sh.acc[3]) atomicAdd(&ctrl->buScanned[ci], sh.acc[3]);
    if (sh.acc[4]) atomicAdd(&ctrl->qbytes[ci], sh.acc[4]);
#pragma unroll
    for (int k = 0; k < 5; ++k) sh.acc[k] = 0;
  }
  __syncthreads();
}

// ---- frontier word list: per-CTA staging in shared memory, one global atomic per flush -------------------------
__device__ __forceinline__ void wl_flush(LazyShared& sh, uint32_t* WLn, unsigned int* wlc) {
  __syncthreads();
  const uint32_t cnt = min(sh.wlCnt, WL_STAGE);
  if (threadIdx.x == 0) sh.wlBase = cnt ? atomicAdd(wlc, cnt) : 0u;
  __syncthreads();
  const uint32_t base = sh.wlBase;
  for (uint32_t i = threadIdx.x; i < cnt; i += blockDim.x) WLn[base + i] = sh.wl[i];
  __syncthreads();
  if (threadIdx.x == 0) sh.wlCnt = 0;
  __syncthreads();
}
// Reserve cnt slots (called by one lane).  Returns the first slot of the CTA's staging area, or 0x80000000 | slot of
// the global list once the area is full; the unusable tail of the area is filled with a sentinel the consumer skips.
__device__ __forceinline__ uint32_t wl_reserve(LazyShared& sh, unsigned int* wlc, uint32_t cnt) {
  const uint32_t pos = atomicAdd(&sh.wlCnt, cnt);
  if (pos + cnt <= WL_STAGE) return pos;
  for (uint32_t i = pos; i < WL_STAGE; ++i) sh.wl[i] = NONE;
  return 0x80000000u | atomicAdd(wlc, cnt);
}
__device__ __forceinline__ void wl_store(LazyShared& sh, uint32_t* WLn, uint32_t slot, uint32_t w) {
  BLEST_ASSERT((slot & 0x80000000u) || slot < WL_STAGE);
  if (slot & 0x80000000u) WLn[slot & 0x7FFFFFFFu] = w;
  else sh.wl[slot] = w;
}
// Warp-level append of the non-zero words among the lanes' (word id, flag) pairs.
__device__ __forceinline__ void wl_append(LazyShared& sh, uint32_t* WLn, unsigned int* wlc, uint32_t word, bool nonzero,
                                          uint32_t lane) {
  const uint32_t nz = __ballot_sync(FULL, nonzero);
  if (!nz) return;
  uint32_t base = 0;
  if (lane == 0) base = wl_reserve(sh, wlc, (uint32_t)__popc(nz));
  base = __shfl_sync(FULL, base, 0);
  if (nonzero) wl_store(sh, WLn, base + __popc(nz & ((1u << lane) - 1u)), word);
}

__device__ __forceinline__ uint32_t valid_mask(const BfsParams& p, uint32_t w) {
  return (w == p.nwords - 1 && (p.n & 31u)) ? ((1u << (p.n & 31u)) - 1u) : FULL;
}

__device__ __forceinline__ void prefetch_l2(const void* ptr) { asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr)); }

// ---- lazy marks ----------------------------------------------------------------------------------
// U candidate vertices per lane: filtered no-return atomic ORs into the next frontier.  The probes of the U
// candidates are issued together (V first: it does not change during Stage 1, so L1 may serve it; then F_next at L2).
// probeFn: also read F_next before the atomic.  It pays when a level has many more edges than unvisited vertices
// (most marks would repeat an earlier one, and repeated atomics on a hot word serialise in L2); otherwise it is one
// more scattered access per edge for nothing, so the level decides (mf > 4 nu).
// hub: per-CTA shared bitmap over the first HUB_BITS vertex ids.  After the degree sort those are the hubs, the targets
// of most edges: a shared-memory atomic drops the repeats before they cost a scattered probe and an L2 atomic on a hot
// word (each CTA sends at most one mark per hub and level).
struct Marks {
  const uint32_t* V;
  uint32_t* Fn;
  bool probeFn;
  uint32_t* hub;
  uint32_t hubLimit;  // HUB_BITS, or 0 = filter off (graphs that are not degree-sorted: low ids are no hubs there)
  uint32_t nBits;     // vertices (bound of every mark; debug asserts)
};
template <int U>
__device__ __forceinline__ void mark_batch(const Marks& mk, const uint32_t (&v)[U], uint32_t valid) {
  const uint32_t* V = mk.V;
  uint32_t* Fn = mk.Fn;
#pragma unroll
  for (int j = 0; j < U; ++j) BLEST_ASSERT(!((valid >> j) & 1u) || v[j] < mk.nBits);
#pragma unroll
  for (int j = 0; j < U; ++j)
    if (((valid >> j) & 1u) && v[j] < mk.hubLimit) {
      const uint32_t bit = 1u << (v[j] & 31u);
      if (atomicOr(&mk.hub[v[j] >> 5], bit) & bit) valid &= ~(1u << j);
    }
  uint32_t vw[U];
#pragma unroll
  for (int j = 0; j < U; ++j) vw[j] = ((valid >> j) & 1u) ? V[v[j] >> 5] : FULL;
  uint32_t need = 0;
#pragma unroll
  for (int j = 0; j < U; ++j)
    if (!((vw[j] >> (v[j] & 31u)) & 1u)) need |= 1u << j;
  if (!mk.probeFn) {
#pragma unroll
    for (int j = 0; j < U; ++j)
      if ((need >> j) & 1u) atomicOr(&Fn[v[j] >> 5], 1u << (v[j] & 31u));
    return;
  }
  uint32_t fw[U];
#pragma unroll
  for (int j = 0; j < U; ++j) fw[j] = ((need >> j) & 1u) ? __ldcg(&Fn[v[j] >> 5]) : FULL;
#pragma unroll
  for (int j = 0; j < U; ++j)
    if (((need >> j) & 1u) && !((fw[j] >> (v[j] & 31u)) & 1u)) atomicOr(&Fn[v[j] >> 5], 1u << (v[j] & 31u));
}

// Smallest lane whose inclusive prefix exceeds idx (idx < total); all 32 lanes must call.
__device__ __forceinline__ uint32_t find_owner(uint32_t incl, uint32_t idx) {
  uint32_t lo = 0;
#pragma unroll
  for (int step = 16; step > 0; step >>= 1) {
    const uint32_t probe = __shfl_sync(FULL, incl, lo + step - 1);
    if (probe <= idx) lo += step;
  }
  return lo;
}

// CUDA-core top-down: each lane owns one adjacency segment [r0, r0+deg); the warp walks the concatenation.
__device__ __forceinline__ void expand_edges(const BfsParams& p, const Marks& Fn, uint32_t r0, uint32_t deg, uint32_t lane) {
  const uint32_t incl = warp_incl_scan(deg, lane);
  const uint32_t total = __shfl_sync(FULL, incl, 31);
  const uint32_t basePtr = r0 - (incl - deg);
  for (uint32_t base = 0; base < total; base += 128u) {
    uint32_t v[4], valid = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint32_t idx = base + 32u * j + lane;
      const uint32_t own = find_owner(incl, idx);
      const uint32_t bp = __shfl_sync(FULL, basePtr, own);
      v[j] = 0;
      if (idx < total) {
        BLEST_ASSERT((uint64_t)bp + idx < p.nnz);
        v[j] = __ldcs(p.colidx + (bp + idx));
        valid |= 1u << j;
      }
    }
    mark_batch<4>(Fn, v, valid);
  }
}

// One contiguous run of edges handled by the whole warp (balanced phase, long adjacency lists).
__device__ __forceinline__ void warp_edges(const BfsParams& p, const Marks& Fn, uint32_t e0, uint32_t e1, uint32_t lane) {
  for (uint32_t base = e0; base < e1; base += 128u) {
    uint32_t v[4], valid = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint32_t idx = base + 32u * j + lane;
      v[j] = 0;
      if (idx < e1) {
        BLEST_ASSERT(idx < p.nnz);
        v[j] = __ldcs(p.colidx + idx);
        valid |= 1u << j;
      }
    }
    mark_batch<4>(Fn, v, valid);
  }
}

__device__ __forceinline__ void mark_quad(const BfsParams& p, const Marks& Fn, const uint4& r, uint32_t hits) {
  const uint32_t v[4] = {r.x, r.y, r.z, r.w};
  mark_batch<4>(Fn, v, hits);
}

// Pull contraction over quads [a, a+nq) of ONE slice set with frontier word alpha: per lane a
// 128-bit row-id load and a 32-bit mask load, four quads in flight.  alpha is warp-uniform, all 32 lanes take part
// (the MMA forms of the contraction need both).
template <int CONTR>
__device__ __forceinline__ void warp_slices(const BfsParams& p, const Marks& Fn, uint32_t a, uint32_t nq, uint32_t alpha,
                                            uint32_t lane) {
  for (uint32_t base = 0; base < nq; base += 128u) {
    uint4 r[4];
    uint32_t m[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t idx = base + 32u * k + lane;
      r[k] = make_uint4(0, 0, 0, 0);
      m[k] = 0;
      if (idx < nq) {
        BLEST_ASSERT((uint64_t)a + idx < p.nQuads);
        r[k] = __ldcs(p.rowIds + a + idx);
        m[k] = __ldcs(p.masks + a + idx);
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (base + 32u * k < nq) {  // warp-uniform
        const uint32_t hits = contract<CONTR>(m[k], alpha, lane);
        mark_quad(p, Fn, r[k], hits);
      }
    }
  }
}

// Slice path, flattened: each lane owns the quads [a, a+nq) of one slice set with its own frontier word alpha; the
// warp walks the concatenation, two quads per lane in flight (ALU contraction: it needs no warp-uniform alpha).
__device__ __forceinline__ void expand_slices(const BfsParams& p, const Marks& Fn, uint32_t a, uint32_t nq, uint32_t alpha,
                                              uint32_t lane) {
  const uint32_t incl = warp_incl_scan(nq, lane);
  const uint32_t total = __shfl_sync(FULL, incl, 31);
  const uint32_t basePtr = a - (incl - nq);
  for (uint32_t base = 0; base < total; base += 64u) {
    uint4 r[2];
    uint32_t m[2], al[2];
    bool ok[2];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const uint32_t idx = base + 32u * j + lane;
      const uint32_t own = find_owner(incl, idx);
      const uint32_t bp = __shfl_sync(FULL, basePtr, own);
      al[j] = __shfl_sync(FULL, alpha, own);
      ok[j] = idx < total;
      r[j] = make_uint4(0, 0, 0, 0);
      m[j] = 0;
      if (ok[j]) {
        BLEST_ASSERT((uint64_t)bp + idx < p.nQuads);
        r[j] = __ldcs(p.rowIds + (bp + idx));
        m[j] = __ldcs(p.masks + (bp + idx));
      }
    }
#pragma unroll
    for (int j = 0; j < 2; ++j)
      if (__any_sync(FULL, ok[j])) mark_quad(p, Fn, r[j], contract_alu(m[j], al[j]));
  }
}

// A hub segment (long adjacency list / big slice set) is cut into equal chunks by the warp that found it; the chunks
// are consumed by the whole grid in the balanced phase.
__device__ __forceinline__ void emit_chunks(const BfsParams& p, Ctrl* ctrl, uint32_t ci, uint32_t type, uint32_t start,
                                            uint32_t count, uint32_t alpha, uint32_t lane, bool coarse) {
  // fine chunks when the frontier is short (a few hubs must still spread over all warps), four times coarser when it
  // is long (enough chunks anyway; a full 128-quad / 512-edge step per lane batch)
  const uint32_t per = (type ? CHUNK_EDGES : CHUNK_QUADS) * (coarse ? 4u : 1u);
  const uint32_t nent = (count + per - 1) / per;
  uint32_t pos = 0;
  if (lane == 0) {
    pos = atomicAdd(&ctrl->qc[ci], nent);
    atomicAdd(&ctrl->nBig[ci], 1u);
  }
  pos = __shfl_sync(FULL, pos, 0);
  if ((uint64_t)pos + nent > p.chunkCap) {
    if (lane == 0) report_overflow(ctrl, p.hostStatus);
    return;
  }
  BLEST_ASSERT((uint64_t)pos + nent <= p.chunkCap);
  for (uint32_t i = lane; i < nent; i += 32) p.chunks[pos + i] = make_uint4(start + i * per, min(per, count - i * per), alpha, type);
}

// Stage 1, top-down, phase A: 32 non-zero frontier words per warp step (lane = word).
template <int CONTR>
__device__ __forceinline__ void td_phase_a(const BfsParams& p, LazyShared& sh, const uint32_t* WLc, uint32_t wlCount,
                                           const uint32_t* Fp, const Marks& Fn, Ctrl* ctrl, uint32_t ci) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  const int sw = p.switching;
  // words per warp step: 32 when the list is long; fewer when it is short, so that a small frontier still spreads
  // over the grid (one word per warp below nwarps words)
  const uint32_t W = min(32u, max(1u, (wlCount + nwarps - 1) / nwarps));
  const bool coarse = wlCount >= nwarps;
  // one word per warp (tiny frontier): segments beyond one batch of a lane set go to the balanced phase, so that no
  // single warp walks thousands of edges while the grid waits
  const uint32_t bigEdges = W == 1u ? 128u : BIG_EDGES, bigQuads = W == 1u ? 32u : BIG_QUADS;
  Counters c;
  for (uint32_t i0 = gwarp * W; i0 < wlCount; i0 += nwarps * W) {
    const uint32_t i = i0 + lane;
    uint32_t t = NONE, fw = 0, thr = 0x9999u;
    if (lane < W && i < wlCount) t = __ldcg(&WLc[i]);
    if (t != NONE) {  // NONE: staging sentinel (wl_reserve)
      BLEST_ASSERT(t < p.nSweepWords);
      fw = Fp[t];
      if (sw == 0 || sw == 5) thr = __ldg(&p.popThr[t]);
    }
    // which of the word's four slice sets take the slice path: forced, or by the build-time threshold on the number
    // of frontier columns
    uint32_t smask = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t byte = (fw >> (8 * k)) & 0xFFu;
      bool use = false;
      if (byte) {
        if (sw == 1 || sw == 4) use = true;
        else if (sw == 3) use = false;
        else use = (uint32_t)__popc(byte) >= ((thr >> (4 * k)) & 15u);
      }
      if (use) smask |= 1u << k;
    }
    uint32_t ebits = fw;
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if ((smask >> k) & 1u) ebits &= ~(0xFFu << (8 * k));
    // ---- slice path
    if (__any_sync(FULL, smask != 0)) {
      uint32_t a[4], nq[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        a[k] = nq[k] = 0;
        if ((smask >> k) & 1u) {
          const uint32_t s = t * 4u + k;
          a[k] = __ldg(&p.setPtr[s]);
          nq[k] = __ldg(&p.setPtr[s + 1]) - a[k];
          c.qbytes += 20u * nq[k] + 8u;
        }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (!__any_sync(FULL, nq[k] != 0)) continue;
        const uint32_t alpha = (fw >> (8 * k)) & 0xFFu;
        // hub sets -> balanced phase; with an MMA contraction every set is walked by the whole warp (uniform alpha)
        uint32_t big = __ballot_sync(FULL, nq[k] > (CONTR == 1 ? bigQuads : 0u));
        while (big) {
          const int src = __ffs(big) - 1;
          big &= big - 1;
          const uint32_t A = __shfl_sync(FULL, a[k], src), NQ = __shfl_sync(FULL, nq[k], src), AL = __shfl_sync(FULL, alpha, src);
          if (NQ > bigQuads) emit_chunks(p, ctrl, ci, 0u, A, NQ, AL, lane, coarse);
          else warp_slices<CONTR>(p, Fn, A, NQ, AL, lane);
        }
        if (CONTR == 1) expand_slices(p, Fn, a[k], nq[k] > bigQuads ? 0u : nq[k], alpha, lane);
      }
    }
    // ---- CUDA-core edge path: up to four frontier vertices per lane and round
    while (__any_sync(FULL, ebits != 0)) {
      uint32_t r0[4], deg[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        r0[q] = deg[q] = 0;
        if (ebits) {
          const uint32_t u = t * 32u + (uint32_t)(__ffs(ebits) - 1);
          ebits &= ebits - 1;
          r0[q] = __ldg(&p.rowptr[u]);
          deg[q] = __ldg(&p.rowptr[u + 1]) - r0[q];
          c.qbytes += 8u;
        }
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (!__any_sync(FULL, deg[q] != 0)) continue;
        c.qbytes += 4u * deg[q];
        uint32_t big = __ballot_sync(FULL, deg[q] > bigEdges);
        while (big) {
          const int src = __ffs(big) - 1;
          big &= big - 1;
          emit_chunks(p, ctrl, ci, 1u, __shfl_sync(FULL, r0[q], src), __shfl_sync(FULL, deg[q], src), 0u, lane, coarse);
        }
        expand_edges(p, Fn, r0[q], deg[q] > bigEdges ? 0u : deg[q], lane);
      }
    }
  }
  block_accumulate(sh, c, ctrl, ci);
}

// Phase B: one warp per chunk, round-robin: every warp gets the same share of the hubs' bytes.
// With options.tune[0] (ALU contraction only): the slice chunks are cut into tiles of TILE_QUADS quads and STAGED IN SHARED MEMORY BY TMA BULK COPIES
// (cp.async.bulk + mbarrier, two stages per warp): while the warp contracts and marks tile t, the row ids and masks of
// tile t+1 are already travelling, without occupying registers or load/store-unit slots (north_star (b); the paper's
// profile has 39 % of Alg. 3's time waiting on these loads).  The masks of a tile start at a 4-byte
// granularity, a bulk copy at 16 bytes: the copy starts at the aligned word below and the lanes index past the slack.
template <int CONTR>
__device__ __forceinline__ void td_phase_b(const BfsParams& p, LazyShared& sh, uint32_t nChunks, const Marks& Fn) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  if (CONTR != 1 || !p.tmaTiles) {  // default (measured faster) and the MMA forms: 128-bit loads into registers
    for (uint32_t i = gwarp; i < nChunks; i += nwarps) {
      BLEST_ASSERT(i < p.chunkCap);
      const uint4 e = __ldcg(&p.chunks[i]);
      if (e.w) warp_edges(p, Fn, e.x, e.x + e.y, lane);
      else warp_slices<CONTR>(p, Fn, e.x, e.y, e.z, lane);
    }
    return;
  }
  // pass 1: the edge chunks (CSR segments of hub vertices)
  bool anySlices = false;
  for (uint32_t i = gwarp; i < nChunks; i += nwarps) {
    BLEST_ASSERT(i < p.chunkCap);
    const uint4 e = __ldcg(&p.chunks[i]);
    if (e.w) warp_edges(p, Fn, e.x, e.x + e.y, lane);
    else anySlices = true;
  }
  if (!anySlices) return;
  // pass 2: the slice chunks, tile by tile through the two-stage ring
  uint4 (*rows)[TILE_QUADS] = sh.tileRows[warp];
  uint32_t (*masks)[TILE_QUADS + 8] = sh.tileMasks[warp];
  uint64_t* bar = reinterpret_cast<uint64_t*>(sh.tileBar[warp]);
  uint32_t phase = sh.tilePhase[warp];
  uint32_t ci = gwarp, off = 0;
  uint4 ce = make_uint4(0, 0, 0, 1);
  bool have = false;
  uint32_t tStart[2], tCnt[2], tAlpha[2];
  // next tile of this warp's slice chunks -> stage `st`; false when there is none (warp-uniform)
  auto stage_next = [&](uint32_t st) -> bool {
    for (;;) {
      if (!have) {
        if (ci >= nChunks) return false;
        ce = __ldcg(&p.chunks[ci]);
        have = true;
        off = 0;
      }
      if (ce.w || off >= ce.y) { have = false; ci += nwarps; continue; }
      break;
    }
    tStart[st] = ce.x + off;
    tCnt[st] = min(TILE_QUADS, ce.y - off);
    tAlpha[st] = ce.z;
    off += TILE_QUADS;
    if (lane == 0) {
      const uint32_t m0 = tStart[st] & ~3u, m1 = (tStart[st] + tCnt[st] + 3u) & ~3u;
      BLEST_ASSERT((uint64_t)tStart[st] + tCnt[st] <= p.nQuads && m1 - m0 <= TILE_QUADS + 8u);
      mbar_arrive_expect_tx(&bar[st], tCnt[st] * 16u + (m1 - m0) * 4u);
      bulk_g2s(rows[st], p.rowIds + tStart[st], tCnt[st] * 16u, &bar[st]);
      bulk_g2s(masks[st], p.masks + m0, (m1 - m0) * 4u, &bar[st]);
    }
    return true;
  };
  bool live[2];
  live[0] = stage_next(0);
  live[1] = live[0] && stage_next(1);
  for (uint32_t st = 0; live[st]; st ^= 1u) {
    mbar_wait(&bar[st], (phase >> st) & 1u);
    phase ^= 1u << st;
    uint4 r[2];
    uint32_t m[2];
    const uint32_t cnt = tCnt[st], alpha = tAlpha[st], slack = tStart[st] & 3u;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const uint32_t idx = 32u * k + lane;
      r[k] = make_uint4(0, 0, 0, 0);
      m[k] = 0;
      if (idx < cnt) {
        r[k] = rows[st][idx];
        m[k] = masks[st][slack + idx];
      }
    }
    __syncwarp();  // every lane has its quads in registers: the stage may be refilled
    live[st] = stage_next(st);
#pragma unroll
    for (int k = 0; k < 2; ++k)
      if (32u * k < cnt) mark_quad(p, Fn, r[k], contract_alu(m[k], alpha));  // (warp-uniform condition)
  }
  if (lane == 0) sh.tilePhase[warp] = phase;
}

// levels_out[original id of u] = level, for the set bits of up to eight words at a time (lane = bit: coalesced
// iperm / degree loads); also the degree sum of the new frontier for the switch.
// `store` = false on the level the pre-fill already wrote ("level guess", see the kernel): only the degree sum remains.
__device__ __forceinline__ void write_levels_dense(const BfsParams& p, uint32_t wordBase, uint32_t fm, uint32_t sel,
                                                   int32_t level, uint32_t lane, Counters& c, bool store) {
  while (sel) {
    uint32_t u[8], on = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      u[q] = 0;
      if (sel) {
        const int src = __ffs(sel) - 1;
        sel &= sel - 1;
        const uint32_t f = __shfl_sync(FULL, fm, src);
        on |= ((f >> lane) & 1u) << q;
        u[q] = (wordBase + src) * 32u + lane;
      }
    }
    uint32_t o[8], dg[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) o[q] = (store && ((on >> q) & 1u)) ? (p.ipermW ? __ldg(&p.ipermW[u[q]]) : u[q]) : 0u;
#pragma unroll
    for (int q = 0; q < 8; ++q) dg[q] = ((on >> q) & 1u) ? __ldg(&p.deg[u[q]]) : 0u;
#pragma unroll
    for (int q = 0; q < 8; ++q) c.mf += dg[q];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      BLEST_ASSERT(!((on >> q) & 1u) || (o[q] < p.n && u[q] < p.n));
      if (store && ((on >> q) & 1u)) p.lvl[o[q]] = level;
    }
  }
}
// Same for a lane's own sparse word (a few bits): four vertices in flight.
__device__ __forceinline__ void write_levels_sparse(const BfsParams& p, uint32_t t, uint32_t bits, int32_t level, Counters& c,
                                                    bool store) {
  while (bits) {
    uint32_t u[4], o[4];
    bool on[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      on[q] = bits != 0;
      u[q] = 0;
      if (bits) {
        u[q] = t * 32u + (uint32_t)(__ffs(bits) - 1);
        bits &= bits - 1;
      }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) o[q] = (store && on[q]) ? (p.ipermW ? __ldg(&p.ipermW[u[q]]) : u[q]) : 0u;
    uint32_t dg[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) dg[q] = on[q] ? __ldg(&p.deg[u[q]]) : 0u;
#pragma unroll
    for (int q = 0; q < 4; ++q) c.mf += dg[q];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      BLEST_ASSERT(!on[q] || (o[q] < p.n && u[q] < p.n));
      if (store && on[q]) p.lvl[o[q]] = level;
    }
  }
}

// Levels of up to eight (word, bits) entries of the CTA's dense list at a time (lane = bit).
__device__ __forceinline__ void write_levels_list(const BfsParams& p, const uint2* ent, uint32_t cnt, int32_t level,
                                                  uint32_t lane, Counters& c, bool store) {
  uint32_t u[8], on = 0;
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    u[q] = 0;
    if ((uint32_t)q < cnt) {
      const uint2 e = ent[q];  // same address in all lanes: a broadcast
      on |= ((e.y >> lane) & 1u) << q;
      u[q] = e.x * 32u + lane;
    }
  }
  uint32_t o[8], dg[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) o[q] = (store && ((on >> q) & 1u)) ? (p.ipermW ? __ldg(&p.ipermW[u[q]]) : u[q]) : 0u;
#pragma unroll
  for (int q = 0; q < 8; ++q) dg[q] = ((on >> q) & 1u) ? __ldg(&p.deg[u[q]]) : 0u;
  uint32_t sum = 0;
#pragma unroll
  for (int q = 0; q < 8; ++q) sum += dg[q];
  c.mf += sum;
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    BLEST_ASSERT(!((on >> q) & 1u) || (o[q] < p.n && u[q] < p.n));
    if (store && ((on >> q) & 1u)) p.lvl[o[q]] = level;
  }
}

// Stage 2 after a top-down Stage 1: frontier finalisation (readings R9/R10).
__device__ __forceinline__ void td_finalize(const BfsParams& p, LazyShared& sh, uint32_t level, uint32_t* Fn, uint32_t* Fs,
                                            uint32_t* WLn, Ctrl* ctrl, uint32_t ci, bool store) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  // Consecutive 32-word batches go to warps of DIFFERENT CTAs (odd multiplier, coprime to the warp count), and the
  // dense words a CTA finds are pooled and shared by its 32 warps: after a degree sort the discoveries of an early
  // level sit in a few thousand consecutive words, which would otherwise be 1 024 level writes each for ~170 warps
  // (4 x 4.5 us of dependent rounds) while 4 500 warps wait.
  const uint32_t mult = (nwarps % 149u) ? 149u : 1u;
  const uint32_t first = (uint32_t)(((uint64_t)gwarp * mult) % nwarps);
  if (threadIdx.x == 0) { sh.dcount = 0; sh.dvalid = 0; }
  __syncthreads();
  Counters c;
  for (uint32_t wb = first * 32u; wb < p.nSweepWords; wb += nwarps * 32u) {
    const uint32_t t = wb + lane;
    uint32_t fm = 0;
    if (t < p.nSweepWords) {
      const uint32_t fn = __ldcg(&Fn[t]), v = __ldcg(&p.V[t]);
      fm = fn & ~v;  // "diff" of PAPER.md:404: marked in this level and not visited before
      Fs[t] = 0;     // the frontier of two levels ago becomes the clean F_next of the next level
      if (fn != fm) Fn[t] = fm;
      if (fm) p.V[t] = v | fm;
      c.unv += __popc(~(v | fm) & valid_mask(p, t));
      c.nnew += __popc(fm);
    }
    if (!__any_sync(FULL, fm != 0)) continue;
    // next level's work list (PAPER.md:420-440 enqueues the VSSs of every newly active slice set; here the non-zero
    // frontier word is the unit, expanded at consumption time)
    wl_append(sh, WLn, &ctrl->wlc[ci], t, fm != 0, lane);
    // level once per discovered vertex: sparse words by their own lane, dense ones pooled per CTA
    const bool dense = __popc(fm) > 6;
    const uint32_t dmask = __ballot_sync(FULL, dense);
    if (dmask) {
      uint32_t base = 0;
      const uint32_t nd = (uint32_t)__popc(dmask);
      if (lane == 0) {
        base = atomicAdd(&sh.dcount, nd);
        if (base + nd <= DLIST_CAP) atomicMax(&sh.dvalid, base + nd);
      }
      base = __shfl_sync(FULL, base, 0);
      if (base + nd <= DLIST_CAP) {
        BLEST_ASSERT(!dense || base + __popc(dmask & ((1u << lane) - 1u)) < DLIST_CAP);
        if (dense) sh.dlist[base + __popc(dmask & ((1u << lane) - 1u))] = make_uint2(t, fm);
      } else {
        write_levels_dense(p, wb, fm, dmask, (int32_t)level, lane, c, store);  // pool full: the owner does them itself
      }
    }
    if (!dense) write_levels_sparse(p, t, fm, (int32_t)level, c, store);
  }
  __syncthreads();
  {
    const uint32_t nd = sh.dvalid;  // entries [0, nd) are valid: reservations are monotone, the first failure ends them
    for (uint32_t e = warp * 8u; e < nd; e += WARPS_PER_BLOCK * 8u)
      write_levels_list(p, &sh.dlist[e], min(8u, nd - e), (int32_t)level, lane, c, store);
  }
  wl_flush(sh, WLn, &ctrl->wlc[ci]);
  block_accumulate(sh, c, ctrl, ci);
}

// ---- bottom-up (Alg. 4, :466-494) fused with its finalisation ---------------------------------------------
// Resolve up to 8 unvisited vertices per lane (u[k], NONE = no vertex): does u have a neighbour in the frontier Fp?
// Inline heads first (one coalesced 8-byte load: first two neighbours), then -- for the few vertices with more than two
// neighbours and neither of the first two in the frontier -- the CSR scan of PAPER.md:479-487 from the third neighbour
// on, compacted over the warp (one such vertex per lane and round, four neighbours in flight).  Returns the lane's
// 8-bit found mask.  All 32 lanes must call.
constexpr uint32_t CSR_STAGE = 0x80000000u;  // list entry flag: heads already checked, continue with the CSR scan

template <bool DEFER>
__device__ __forceinline__ uint32_t bu_resolve(const BfsParams& p, const uint32_t* Fp, uint32_t* fshare, uint32_t* slotU,
                                               uint32_t* slotTag, uint32_t lane, const uint32_t (&u)[8], Counters& c,
                                               uint32_t* list, uint32_t& listCount) {
  constexpr int K = 8;
  constexpr uint32_t SERIAL_CAP = 64;
  uint2 h[K];
  uint32_t act = 0, staged = 0;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    h[k] = make_uint2(NONE, NONE);
    if (u[k] != NONE) {
      if (!DEFER && (u[k] & CSR_STAGE)) staged |= 1u << k;
      else {
        BLEST_ASSERT(u[k] < p.n);
        h[k] = __ldcs(&p.head[u[k]]);
        act |= 1u << k;
      }
    }
  }
  c.qbytes += 8u * (uint32_t)__popc(act);
  uint32_t found = 0, probed = 0;
  {
    uint32_t f[K];
#pragma unroll
    for (int k = 0; k < K; ++k) f[k] = (h[k].x != NONE) ? Fp[h[k].x >> 5] : 0u;
#pragma unroll
    for (int k = 0; k < K; ++k)
      if (h[k].x != NONE) {
        probed |= 1u << k;
        if ((f[k] >> (h[k].x & 31u)) & 1u) found |= 1u << k;
      }
  }
  c.scanned += (uint32_t)__popc(probed);
  uint32_t need = 0;
#pragma unroll
  for (int k = 0; k < K; ++k)
    if (h[k].y != NONE && !((found >> k) & 1u)) need |= 1u << k;
  if (__any_sync(FULL, need != 0)) {
    uint32_t f[K];
#pragma unroll
    for (int k = 0; k < K; ++k) f[k] = ((need >> k) & 1u) ? Fp[(h[k].y & 0x7FFFFFFFu) >> 5] : 0u;
#pragma unroll
    for (int k = 0; k < K; ++k)
      if (((need >> k) & 1u) && ((f[k] >> (h[k].y & 31u)) & 1u)) found |= 1u << k;
    c.scanned += (uint32_t)__popc(need);
  }
  uint32_t more = staged;
#pragma unroll
  for (int k = 0; k < K; ++k)
    if (((need >> k) & 1u) && !((found >> k) & 1u) && (h[k].y >> 31)) more |= 1u << k;
  if (!__any_sync(FULL, more != 0)) return found;

  uint32_t pos[K], total = 0;  // position of the lane's k-th vertex in the warp-wide list of such vertices
  const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    const uint32_t bal = __ballot_sync(FULL, (more >> k) & 1u);
    pos[k] = total + __popc(bal & lt);
    total += __popc(bal);
  }
  if (DEFER) {  // in-place (dense) mode: these vertices join the warp's list and are resolved later, 256 at a time
#pragma unroll
    for (int k = 0; k < K; ++k)
      if ((more >> k) & 1u) {
        BLEST_ASSERT(listCount + pos[k] < BU_LIST);
        list[listCount + pos[k]] = u[k] | CSR_STAGE;
        prefetch_l2(&p.rowptrIn[u[k]]);
      }
    listCount += total;
    __syncwarp();
    return found;
  }
  fshare[lane] = 0;
  for (uint32_t base = 0; base < total; base += 32u) {
    __syncwarp();
#pragma unroll
    for (int k = 0; k < K; ++k)
      if (((more >> k) & 1u) && pos[k] >= base && pos[k] < base + 32u) {
        slotU[pos[k] - base] = u[k];
        slotTag[pos[k] - base] = (uint32_t)k | (lane << 3);
      }
    __syncwarp();
    const bool mine = base + lane < total;
    uint32_t ptr = 0, e = 0, tag = 0;
    if (mine) {
      const uint32_t uu = slotU[lane] & ~CSR_STAGE;
      tag = slotTag[lane];
      ptr = __ldg(&p.rowptrIn[uu]) + 2u;
      e = __ldg(&p.rowptrIn[uu + 1]);
      c.qbytes += 8u;
    }
    bool f = false;
    const uint32_t stop = min(e, ptr + SERIAL_CAP);
    while (!f && ptr < stop) {  // four neighbours per step
      uint32_t v[4], fwd[4];
      const uint32_t cnt = min(4u, stop - ptr);
      BLEST_ASSERT((uint64_t)ptr + cnt <= p.nnz);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] = (uint32_t)j < cnt ? __ldg(&p.colidxIn[ptr + j]) : 0u;
#pragma unroll
      for (int j = 0; j < 4; ++j) fwd[j] = (uint32_t)j < cnt ? Fp[v[j] >> 5] : 0u;
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if ((uint32_t)j < cnt && ((fwd[j] >> (v[j] & 31u)) & 1u)) f = true;
      c.scanned += cnt;
      c.qbytes += 4u * cnt;
      ptr += cnt;
    }
    // long lists are finished by the whole warp
    uint32_t pend = __ballot_sync(FULL, mine && !f && ptr < e);
    while (pend) {
      const int src = __ffs(pend) - 1;
      pend &= pend - 1;
      const uint32_t B = __shfl_sync(FULL, ptr, src), E = __shfl_sync(FULL, e, src);
      bool ff = false;
      for (uint32_t b2 = B; b2 < E; b2 += 32u) {
        const uint32_t idx = b2 + lane;
        bool hit = false;
        if (idx < E) {
          const uint32_t v = __ldg(&p.colidxIn[idx]);
          hit = (Fp[v >> 5] >> (v & 31u)) & 1u;
          ++c.scanned;
          c.qbytes += 4u;
        }
        if (__ballot_sync(FULL, hit)) { ff = true; break; }
      }
      if ((int)lane == src) f = ff;
    }
    if (mine && f) atomicOr(&fshare[tag >> 3], 1u << (tag & 7u));
  }
  __syncwarp();
  found |= fshare[lane];
  __syncwarp();
  return found;
}

// One bottom-up level.  A warp step covers a GROUP of G words of the visited bitmap (lane = word; G = 8 on levels with
// many unvisited vertices so that the groups balance over the grid, 32 otherwise).  Dense groups are resolved in
// place, 8 words at a time with lane = bit, and the warp that owns the words writes V / F_next / levels without
// atomics; what the inline heads cannot decide goes to the warp's list.  The unvisited vertices of sparse groups go to
// the list directly.  The list is resolved 256 vertices at a time whatever words they come from (atomics on
// V / F_next: they are few), so a level with few unvisited vertices costs one sweep of V plus work proportional to
// their number.
__device__ __forceinline__ void bu_level(const BfsParams& p, LazyShared& sh, uint32_t level, const uint32_t* Fp, uint32_t* Fn,
                                         uint32_t* Fs, uint32_t* WLn, Ctrl* ctrl, uint32_t ci, unsigned long long nu, bool store) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  const uint32_t nSW = p.nSweepWords;
  const uint32_t G = (nu * 8ull > (unsigned long long)nSW * 32ull) ? 8u : 32u;  // > 1/8 of the sweep range unvisited
  const uint32_t nGroups = (nSW + G - 1u) / G;
  uint32_t* fshare = sh.buFound[warp];
  uint32_t* slotU = sh.buSlotU[warp];
  uint32_t* slotTag = sh.buSlotTag[warp];
  uint32_t* list = sh.buList[warp];
  uint32_t listCount = 0;
  bool batchRan = false;  // a list batch ran since the current group started
  Counters c;

  // resolve the last `cnt` (<= 256) vertices of the list
  auto run_batch = [&](uint32_t cnt) {
    const uint32_t start = listCount - cnt;
    uint32_t u[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) u[k] = (32u * k + lane < cnt) ? list[start + 32u * k + lane] : NONE;
    __syncwarp();
    listCount = start;
    const uint32_t found = bu_resolve<false>(p, Fp, fshare, slotU, slotTag, lane, u, c, list, listCount);
    uint32_t o[8], dg[8];
#pragma unroll
    for (int k = 0; k < 8; ++k)
      o[k] = (store && ((found >> k) & 1u)) ? (p.ipermW ? __ldg(&p.ipermW[u[k] & ~CSR_STAGE]) : (u[k] & ~CSR_STAGE)) : 0u;
#pragma unroll
    for (int k = 0; k < 8; ++k) dg[k] = ((found >> k) & 1u) ? __ldg(&p.deg[u[k] & ~CSR_STAGE]) : 0u;
    {
      uint32_t sum = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) sum += dg[k];
      c.mf += sum;
    }
    batchRan = true;
    uint32_t oldF[8];  // all eight returning atomics in flight before the first result is needed
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      oldF[k] = 1u;
      if ((found >> k) & 1u) {
        const uint32_t uu = u[k] & ~CSR_STAGE, bit = 1u << (uu & 31u);
        BLEST_ASSERT(o[k] < p.n && uu < p.n);
        if (store) p.lvl[o[k]] = (int32_t)level;
        atomicOr(&p.V[uu >> 5], bit);
        oldF[k] = atomicOr(&Fn[uu >> 5], bit);
      }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k)  // first bit of a word in this level: the word joins the list
      wl_append(sh, WLn, &ctrl->wlc[ci], (u[k] & ~CSR_STAGE) >> 5, oldF[k] == 0u, lane);
    c.nnew += __popc(found);
    c.unv -= __popc(found);
  };

  for (uint32_t g = gwarp; g < nGroups; g += nwarps) {
    const uint32_t gw = g * G, myw = gw + lane;
    const bool wlane = lane < G && myw < nSW;
    uint32_t curw = FULL;
    if (wlane) curw = __ldcg(&p.V[myw]);
    const uint32_t unvw = wlane ? (~curw & valid_mask(p, myw)) : 0u;  // padding bits read as visited (R11)
    if (wlane) Fs[myw] = 0;  // the frontier of two levels ago becomes the clean F_next of the next level
    const uint32_t cnt = __popc(unvw);
    const uint32_t incl = warp_incl_scan(cnt, lane);
    const uint32_t total = __shfl_sync(FULL, incl, 31);
    if (total == 0) continue;
    c.unv += cnt;
    batchRan = false;
    if (total > 8u * G) {
      // ---- dense group (> 1/4 unvisited): in place, 8 words at a time (lane = bit)
      uint32_t fmw = 0;  // new frontier bits of word myw
      const uint32_t nzWords = __ballot_sync(FULL, unvw != 0);
#pragma unroll 1
      for (uint32_t sub = 0; sub < G / 8u; ++sub) {
        if (!((nzWords >> (8u * sub)) & 0xFFu)) continue;
        if (listCount >= BU_BATCH) run_batch(BU_BATCH);  // room for up to 256 deferred vertices
        uint32_t u[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const uint32_t wbits = __shfl_sync(FULL, unvw, 8u * sub + k);
          u[k] = ((wbits >> lane) & 1u) ? (gw + 8u * sub + k) * 32u + lane : NONE;
        }
        const uint32_t found = bu_resolve<true>(p, Fp, fshare, slotU, slotTag, lane, u, c, list, listCount);
        uint32_t o[8], dg[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) o[k] = (store && ((found >> k) & 1u)) ? (p.ipermW ? __ldg(&p.ipermW[u[k]]) : u[k]) : 0u;
#pragma unroll
        for (int k = 0; k < 8; ++k) dg[k] = ((found >> k) & 1u) ? __ldg(&p.deg[u[k]]) : 0u;
        {
          uint32_t sum = 0;  // 8 degrees < 2^29 each
#pragma unroll
          for (int k = 0; k < 8; ++k) sum += dg[k];
          c.mf += sum;
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          BLEST_ASSERT(!((found >> k) & 1u) || (o[k] < p.n && u[k] < p.n));
          if (store && ((found >> k) & 1u)) p.lvl[o[k]] = (int32_t)level;  // lane = bit: coalesced when there is no reordering
          const uint32_t fmk = __ballot_sync(FULL, (found >> k) & 1u);
          if (lane == 8u * sub + k) fmw = fmk;
        }
      }
      // one atomic per word instead of one per lane; atomic because vertices of this word that were
      // deferred to the list may already have been resolved by run_batch
      bool newWord = false;
      if (fmw) {
        if (batchRan) {  // (warp-uniform) deferred vertices of this group may already have set bits in these words
          atomicOr(&p.V[myw], fmw);
          newWord = atomicOr(&Fn[myw], fmw) == 0u;
        } else {
          p.V[myw] = curw | fmw;
          Fn[myw] = fmw;
          newWord = true;
        }
      }
      __syncwarp();  // the plain stores precede this warp's later atomics on the same words (deferred vertices)
      c.nnew += __popc(fmw);
      c.unv -= __popc(fmw);
      wl_append(sh, WLn, &ctrl->wlc[ci], myw, newWord, lane);
    } else {
      // ---- sparse group: queue its unvisited vertices
      if (listCount + total > BU_LIST) run_batch(BU_BATCH);
      uint32_t at = listCount + incl - cnt;
      for (uint32_t bits = unvw; bits; bits &= bits - 1) {
        const uint32_t u = myw * 32u + (uint32_t)(__ffs(bits) - 1);
        BLEST_ASSERT(at < BU_LIST && u < p.n);
        list[at++] = u;
        prefetch_l2(&p.head[u]);
      }
      listCount += total;
      __syncwarp();
      if (listCount >= BU_BATCH) run_batch(BU_BATCH);
    }
  }
  while (listCount) run_batch(min(listCount, BU_BATCH));
  wl_flush(sh, WLn, &ctrl->wlc[ci]);
  block_accumulate(sh, c, ctrl, ci);
}

// Direction of level `level` (Eq. 6 analogue).  All threads evaluate it on the same
// counters, so the decision is grid-uniform.
__device__ __forceinline__ bool choose_bottom_up(const BfsParams& p, uint32_t level, unsigned long long nf,
                                                 unsigned long long mf, unsigned long long nu, unsigned long long mu) {
  if (p.switching == 2) return level >= 2;
  if (p.switching == 5) return (p.buMask >> min(level, 31u)) & 1u;
  if (p.switching != 0) return false;
  // Top-down examines every edge out of the frontier (one bitmap probe each) and sweeps the bitmaps once.
  // Bottom-up examines, for every unvisited vertex, neighbours until the first one in the frontier: with a fraction
  // mf/nnz of all edge endpoints in the frontier that is about nnz/mf per vertex, and never more than its degree.
  const float fmf = (float)mf, fnu = (float)nu;
  // ... in a graph whose neighbours are met in random order.  After the degree sort the first neighbours are the hubs,
  // which enter the frontier first: the traces fit (nnz/mf)^0.5 there (scanExp; 1 for unordered graphs).
  const float perVertex = fminf(powf((float)p.nnz / fmaxf(fmf, 1.0f), p.scanExp), fnu > 0.f ? (float)mu / fnu : 0.f);
  // top-down: every edge out of the frontier is read and probed (cTdEdge); a vertex it discovers costs an atomic, a
  // finalisation and a level write (cTdNew); mf edges thrown at nAct candidate vertices discover about
  // nu (1 - exp(-mf / nAct)) of the nu unvisited ones (exact for the uniform graph, an over-estimate for skewed ones)
  const float nAct = fmaxf((float)p.nSweepWords * 32.0f - (float)p.nIsoInSweep, 1.0f);
  const float newEst = fnu * (1.0f - __expf(-fmf / nAct));
  const float costTd = p.cTdEdge * fmf + p.cTdNew * newEst + p.cTdVertex * (float)nf + p.cTdWord * (float)p.nSweepWords;
  const float costBu = p.cBuVertex * fnu + p.cBuScan * fnu * perVertex + p.cBuWord * (float)p.nSweepWords;
  return costBu * 10.0f < p.eta * costTd;
}

template <int CONTR>
__global__ void __launch_bounds__(BLOCK_THREADS, 1) bfs_lazy_kernel(const __grid_constant__ BfsParams p) {
  extern __shared__ __align__(128) unsigned char lazy_smem[];
  LazyShared& sh = *reinterpret_cast<LazyShared*>(lazy_smem);
  Ctrl* ctrl = p.ctrl;
  // The control block is never memset between calls: the barrier counter is monotone over the launches on this
  // handle (stream-ordered), `epochBase` is where the previous launch left it, and the leader resets the per-call
  // fields below.  Only thread 0 of a CTA evaluates the barrier target, so only it needs the true epoch.
  if (threadIdx.x == 0) {
    sh.epoch = ld_volatile(&ctrl->epochBase);
    // LEVEL GUESS.  On a low-diameter graph one level discovers most of the component (config 4: level 3 finds 8.8 M of the
    // 11 M reachable vertices), and its scattered level writes + original-id loads are a third of that level's time.
    // The previous call on this handle (from a source of similar degree) left the level that discovered the most vertices in
    // ctrl->guess; this call
    // pre-fills levels_out with it instead of -1 (the vertices the traversal cannot reach -- p.negBits: everything
    // outside the source's component, known since blest_build -- still get -1), and the level that equals the guess
    // then writes no levels at all.  Every other level overwrites the guess as before, and every vertex of the
    // component is discovered at some level, so the result does not depend on the guess being right.
    const bool aligned = (((uintptr_t)p.lvl) & 15u) == 0;
    // (which level that is depends on how far the source is from the hubs: the guess is kept per class of source)
    const uint32_t sr = __ldg(&p.rowptr[p.src]), sd = __ldg(&p.rowptr[p.src + 1]) - sr;
    const uint32_t first = sd ? __ldg(&p.colidx[sr]) : 0u;  // lowest id = (after a degree sort) the highest degree
    sh.guessSlot = (31u - (uint32_t)__clz(sd + 1u)) * 32u + min(31u, 31u - (uint32_t)__clz(first + 1u));
    sh.guess = (p.negBits && aligned) ? ld_volatile(&ctrl->guess[sh.guessSlot]) : 0u;
    sh.bestCount = 0;
    sh.bestLevel = 0;
  }
  const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (uint64_t)gridDim.x * blockDim.x;
  const bool leader = (blockIdx.x == 0 && threadIdx.x == 0);
  if (threadIdx.x < 6) sh.acc[threadIdx.x] = 0;
  if (threadIdx.x == 0) sh.wlCnt = 0;
  if ((threadIdx.x & 31) == 0) {  // the warp's two tile-stage barriers: one arrival (the issuing lane) + the copies' bytes
    mbar_init(reinterpret_cast<uint64_t*>(&sh.tileBar[threadIdx.x >> 5][0]), 1u);
    mbar_init(reinterpret_cast<uint64_t*>(&sh.tileBar[threadIdx.x >> 5][1]), 1u);
    sh.tilePhase[threadIdx.x >> 5] = 0;
    mbar_init_fence();
  }
  if (leader) ctrl->t0 = globaltimer();

  // A4 per-call init: bitmaps cleared, V = F_curr = {src}; levels_out = -1 everywhere.
  const uint32_t nSW = p.nSweepWords, srcWord = p.src >> 5, srcBit = 1u << (p.src & 31u);
  const uint32_t nClear = (nSW + 7u) & ~7u;  // the bottom-up step reads 8 words at a time (buffers are padded)
  for (uint64_t i = gtid; i < nClear; i += nth) {
    const uint32_t x = (i == srcWord) ? srcBit : 0u;
    p.V[i] = x | __ldg(&p.isoBits[i]);
    p.F[0][i] = x;
    p.F[1][i] = 0;
    p.F[2][i] = 0;
  }
  __syncthreads();
  // levels = -1 everywhere (reading R1), before any level is written -- or the guessed level where the
  // traversal can reach
  if (sh.guess) {
    const uint32_t guess = sh.guess;
    uint4* o4 = reinterpret_cast<uint4*>(p.lvl);  // (16-byte aligned: checked above)
    const uint64_t n4 = (uint64_t)p.n >> 2;
    for (uint64_t i0 = gtid; i0 < n4; i0 += 4u * nth) {  // four 16-byte stores per round, their bitmap words loaded first
      uint32_t w[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint64_t i = i0 + (uint64_t)q * nth;
        w[q] = i < n4 ? __ldg(&p.negBits[i >> 3]) : 0u;
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint64_t i = i0 + (uint64_t)q * nth;
        const uint32_t bits = w[q] >> ((uint32_t)(i & 7u) * 4u);
        if (i < n4)
          o4[i] = make_uint4((bits & 1u) ? NONE : guess, (bits & 2u) ? NONE : guess, (bits & 4u) ? NONE : guess,
                             (bits & 8u) ? NONE : guess);
      }
    }
    const uint64_t v = (n4 << 2) + gtid;
    if (v < p.n) p.lvl[v] = ((__ldg(&p.negBits[v >> 5]) >> (v & 31u)) & 1u) ? -1 : (int32_t)guess;
  } else {
    uint32_t* o = reinterpret_cast<uint32_t*>(p.lvl);
    const uint64_t head = min((uint64_t)p.n, (uint64_t)((16u - ((uintptr_t)o & 15u)) & 15u) >> 2);
    const uint64_t n4 = ((uint64_t)p.n - head) >> 2;
    uint4* o4 = reinterpret_cast<uint4*>(o + head);
    const uint4 m1 = make_uint4(NONE, NONE, NONE, NONE);
    for (uint64_t i = gtid; i < n4; i += nth) o4[i] = m1;
    const uint64_t tail0 = head + (n4 << 2);
    if (gtid < head) o[gtid] = NONE;
    if (gtid < (uint64_t)p.n - tail0) o[tail0 + gtid] = NONE;
  }
  const uint32_t srcRow = __ldg(&p.rowptr[p.src]);
  const uint32_t srcDeg = __ldg(&p.rowptr[p.src + 1]) - srcRow;
  if (leader) {
    ctrl->error = 0;
    ctrl->nlevels = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      ctrl->qc[k] = 0; ctrl->qbytes[k] = 0; ctrl->unvisited[k] = 0; ctrl->newcount[k] = 0;
      ctrl->mf[k] = 0; ctrl->buScanned[k] = 0; ctrl->wlc[k] = 0; ctrl->nBig[k] = 0;
    }
    // level 0: the source itself (frontier = {src})
    p.WL[0][0] = srcWord;
    ctrl->wlc[0] = 1;
    ctrl->newcount[0] = 1;
    ctrl->mf[0] = srcDeg;
    // (the source is not counted twice when it is itself pre-marked: a directed graph's source of in-degree 0)
    ctrl->unvisited[0] = (unsigned long long)min((uint64_t)p.n, (uint64_t)nSW * 32u) - (p.srcPremarked ? 0u : 1u) - p.nIsoInSweep;
  }
  grid_barrier_sh(&ctrl->bar, &sh.epoch);
  if (leader) {
    ctrl->tInit = globaltimer() - ctrl->t0;
    p.lvl[p.srcLvl] = 0;  // L[src] = 0 (after the fill: ordered by the barrier)
  }

  if (threadIdx.x == 0) sh.degVisited = 0;  // sum of degrees of all visited vertices (only the deciding thread needs it)
  uint32_t level = 1;
  for (;; ++level) {
    const uint32_t cp = (level - 1) % 3u, ci = level % 3u, cn = (level + 1) % 3u;
    // one thread per CTA reads the level's control words (every warp reading them would queue on one L2 slice)
    if (threadIdx.x == 0) {
      sh.ctl[0] = ld_volatile(&ctrl->newcount[cp]);
      sh.ctl[1] = ld_volatile(&ctrl->mf[cp]);
      sh.ctl[2] = ld_volatile(&ctrl->unvisited[cp]);
      sh.ctl[3] = ld_volatile(&ctrl->wlc[cp]);
      // the switch (a powf and an expf) is evaluated once per CTA, not by every warp
      const unsigned long long dv = sh.degVisited + sh.ctl[1];
      if (sh.ctl[0] != 0 && sh.ctl[2] != 0) sh.degVisited = dv;  // (the level runs: its frontier joins the visited set)
      sh.buDecision = choose_bottom_up(p, level, sh.ctl[0], sh.ctl[1], sh.ctl[2], p.nnz > dv ? p.nnz - dv : 0ull) ? 1u : 0u;
      // the level that discovered the most vertices so far: the next call's guess (kept in shared memory: no registers)
      if (level >= 2u && sh.ctl[0] > sh.bestCount) { sh.bestCount = sh.ctl[0]; sh.bestLevel = level - 1u; }
    }
    __syncthreads();
    const unsigned long long nf = sh.ctl[0];
    const unsigned long long mf = sh.ctl[1];
    const unsigned long long unvAll = sh.ctl[2];
    const uint32_t wlCount = (uint32_t)sh.ctl[3];
    const bool bottomUp = sh.buDecision != 0u;
    __syncthreads();
    const bool storeLv = level != sh.guess;  // the pre-fill already holds this level
    if (nf == 0) break;  // empty frontier ("terminates at the first level with x = 0")
    if (unvAll == 0) break;  // nothing left that could be discovered (everything outside the component is pre-marked)
    const unsigned long long nu = unvAll;  // zero-degree vertices count as visited from the start
    const uint32_t* Fp = p.F[cp];
    uint32_t* Fn = p.F[ci];
    uint32_t* Fs = p.F[cn];
    if (leader) {  // recycle the counters of level+1 (last read at the top of level-1)
      ctrl->newcount[cn] = 0;
      ctrl->mf[cn] = 0;
      ctrl->unvisited[cn] = 0;
      ctrl->buScanned[cn] = 0;
      ctrl->qbytes[cn] = 0;
      ctrl->wlc[cn] = 0;
      ctrl->nBig[cn] = 0;
      ctrl->qc[cn] = 0;
    }
    if (level == 1 && !bottomUp && p.switching == 0) {
      // Level 1 needs no probe, no filter and no sweep: the neighbours of the source other than itself are all unvisited,
      // so each edge of the source finalises its target on the spot (one phase, one barrier instead of two and a sweep);
      // a duplicated CSR entry is caught by the returning atomic on F_next.
      Counters c;
      const uint32_t lane = threadIdx.x & 31;
      const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
      for (uint32_t base = gwarp * 32u; base < srcDeg; base += nwarps * 32u) {
        bool active = base + lane < srcDeg;
        const uint32_t v = active ? __ldcs(p.colidx + srcRow + base + lane) : 0u;
        active = active && v != p.src;  // a self-loop (src, src) discovers nothing: the source is the only visited vertex
        const uint32_t bit = 1u << (v & 31u);
        uint32_t old = FULL;
        if (active) old = atomicOr(&Fn[v >> 5], bit);
        const bool disc = active && !(old & bit);  // (a duplicated CSR entry is not discovered twice)
        uint32_t o = 0, dg = 0;
        if (disc) {
          o = p.ipermW ? __ldg(&p.ipermW[v]) : v;
          dg = __ldg(&p.deg[v]);
          atomicOr(&p.V[v >> 5], bit);
        }
        BLEST_ASSERT(!disc || (o < p.n && v < p.n));
        if (disc && storeLv) p.lvl[o] = 1;
        c.mf += dg;
        c.nnew += disc ? 1u : 0u;
        wl_append(sh, p.WL[1], &ctrl->wlc[ci], v >> 5, disc && old == 0u, lane);
      }
      c.unv = -(int32_t)c.nnew;
      if (gwarp == 0 && lane == 0) {
        c.unv += (int32_t)unvAll;
        c.qbytes += 8u + 4u * srcDeg;
      }
      wl_flush(sh, p.WL[1], &ctrl->wlc[ci]);
      block_accumulate(sh, c, ctrl, ci);
      grid_barrier_sh(&ctrl->bar, &sh.epoch);
      if (leader) sh.tStage1 = globaltimer();
    } else if (bottomUp) {
      bu_level(p, sh, level, Fp, Fn, Fs, p.WL[level & 1u], ctrl, ci, nu, storeLv);
      grid_barrier_sh(&ctrl->bar, &sh.epoch);
      if (leader) sh.tStage1 = globaltimer();
    } else {
      const Marks mk{p.V, Fn, p.hubFilter || mf > 4ull * nu, sh.hub, p.hubFilter ? HUB_BITS : 0u, p.n};
      if (p.hubFilter) {
        for (uint32_t i = threadIdx.x; i < HUB_BITS / 32; i += blockDim.x) sh.hub[i] = 0;
        __syncthreads();
      }
      td_phase_a<CONTR>(p, sh, p.WL[(level - 1) & 1u], wlCount, Fp, mk, ctrl, ci);
      grid_barrier_sh(&ctrl->bar, &sh.epoch);
      if (threadIdx.x == 0) sh.ctl[0] = ld_volatile(&ctrl->qc[ci]);
      __syncthreads();
      const uint32_t nChunks = (uint32_t)sh.ctl[0];
      __syncthreads();
      if (nChunks) {  // hubs: equal chunks spread over the grid
        td_phase_b<CONTR>(p, sh, min(nChunks, p.chunkCap), mk);
        grid_barrier_sh(&ctrl->bar, &sh.epoch);
      }
      if (leader) sh.tStage1 = globaltimer();
      td_finalize(p, sh, level, Fn, Fs, p.WL[level & 1u], ctrl, ci, storeLv);
      grid_barrier_sh(&ctrl->bar, &sh.epoch);
    }
    if (leader && p.trace && level - 1 < p.traceCap) {
      blest_level_trace_t r;
      r.level = level;
      r.mode = bottomUp ? 1u : 0u;
      r.q_entries = bottomUp ? 0u : wlCount;
      r.new_vertices = (uint32_t)ld_volatile(&ctrl->newcount[ci]);
      r.q_bytes = ld_volatile(&ctrl->qbytes[ci]);
      r.bu_scanned = ld_volatile(&ctrl->buScanned[ci]);
      const unsigned long long ua = ld_volatile(&ctrl->unvisited[ci]);
      r.unvisited = (uint32_t)(ua + p.nIsoInSweep + ((unsigned long long)p.n - min((uint64_t)p.n, (uint64_t)nSW * 32u)));
      r.reserved = (bottomUp ? 0u : ld_volatile(&ctrl->nBig[ci])) | (storeLv ? 0u : 0x80000000u);
      r.t_ns = globaltimer() - ctrl->t0;
      r.t_stage1_ns = sh.tStage1 - ctrl->t0;
      p.trace[level - 1] = r;
    }
  }
  if (leader) {
    ctrl->nlevels = level - 1;
    ctrl->guess[sh.guessSlot] = sh.bestLevel;
    ctrl->epochBase = sh.epoch;  // every CTA has executed the same barriers: the next launch continues from here
  }

  // A10 as a separate pass (p.gather): the levels were written in internal ids (coalesced, no iperm read) and go to
  // original ids here.  Used when levels_out is too big to be held in L2 by the persisting window: scattered 4-byte
  // writes then cost DRAM a read-modify-write each (measured: 100 ps per vertex on C3 + RCM against 10 ps for this pass).
  if (p.gather) {
    for (uint64_t v0 = gtid * 4; v0 < p.n; v0 += nth * 4) {
      uint32_t pv[4];
      int32_t lv[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) pv[j] = v0 + j < p.n ? __ldcs(&p.perm[v0 + j]) : 0u;
#pragma unroll
      for (int j = 0; j < 4; ++j) lv[j] = v0 + j < p.n ? p.lvl[pv[j]] : 0;
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (v0 + j < p.n) p.out[v0 + j] = lv[j];
    }
  }
}

__global__ void isolated_source_kernel(int32_t* out, uint32_t n, uint32_t src) {
  for (uint64_t v = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += (uint64_t)gridDim.x * blockDim.x)
    out[v] = (v == src) ? 0 : -1;
}

template <class K>
int coop_blocks(K kernel) {
  int dev = 0, sms = 0, perSm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (cudaFuncSetAttribute((const void*)kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LazyShared)) != cudaSuccess) return 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSm, kernel, BLOCK_THREADS, sizeof(LazyShared)) != cudaSuccess) return 0;
  return sms * (perSm > 0 ? 1 : 0);  // one CTA per SM: the cheapest grid barrier
}

template <class K>
cudaError_t coop_launch(K kernel, const BfsParams& p, int gridBlocks, cudaStream_t st, const void* persistPtr,
                        size_t persistBytes, float hitRatio) {
  void* args[] = {(void*)&p};
  // the hub bitmap is the last member: without the filter the launch leaves that shared memory to the L1
  const size_t smem = p.hubFilter ? sizeof(LazyShared) : offsetof(LazyShared, hub);
  // cooperative launch; the persisting-L2 window (if any) is an attribute of THIS launch, the stream is left alone
  cudaLaunchAttribute attrs[2];
  unsigned int na = 0;
  attrs[na].id = cudaLaunchAttributeCooperative;
  attrs[na].val.cooperative = 1;
  ++na;
  if (persistPtr && persistBytes) {
    attrs[na].id = cudaLaunchAttributeAccessPolicyWindow;
    attrs[na].val.accessPolicyWindow.base_ptr = const_cast<void*>(persistPtr);
    attrs[na].val.accessPolicyWindow.num_bytes = persistBytes;
    attrs[na].val.accessPolicyWindow.hitRatio = hitRatio;
    attrs[na].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    attrs[na].val.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    ++na;
  }
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(gridBlocks);
  cfg.blockDim = dim3(BLOCK_THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cfg.attrs = attrs;
  cfg.numAttrs = na;
  return cudaLaunchKernelExC(&cfg, (const void*)kernel, args);
}

}  // namespace

cudaError_t launch_bfs_lazy(const BfsParams& p, int gridBlocks, cudaStream_t st, const void* persistPtr, size_t persistBytes,
                            float hitRatio) {
  switch (p.contraction) {
    case 2: return coop_launch(bfs_lazy_kernel<2>, p, gridBlocks, st, persistPtr, persistBytes, hitRatio);
    case 3: return coop_launch(bfs_lazy_kernel<3>, p, gridBlocks, st, persistPtr, persistBytes, hitRatio);
    default: return coop_launch(bfs_lazy_kernel<1>, p, gridBlocks, st, persistPtr, persistBytes, hitRatio);
  }
}

// A source of degree 0 reaches nothing (SURVEY.md §8(b) "A source of degree 0 is legal").
cudaError_t launch_isolated_source(int32_t* out, uint32_t n, uint32_t src, cudaStream_t st) {
  const int threads = 256;
  const int blocks = (int)std::min<uint64_t>(((uint64_t)n + threads - 1) / threads, 148ull * 8);
  isolated_source_kernel<<<blocks, threads, 0, st>>>(out, n, src);
  return cudaGetLastError();
}

int max_coop_blocks_lazy() {  // also opts every instantiation into the dynamic shared-memory size
  const int a = coop_blocks(bfs_lazy_kernel<1>), b = coop_blocks(bfs_lazy_kernel<2>), c = coop_blocks(bfs_lazy_kernel<3>);
  return std::min(a, std::min(b, c));
}

}  // namespace blest
