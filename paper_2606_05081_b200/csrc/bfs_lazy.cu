// bfs_lazy.cu -- single-source BLEST traversal with lazy vertex updates (Alg. 3, :345-455) and the
// per-level switch to CUDA-core paths (§5.3, Eq. 6, Alg. 4), as ONE persistent cooperative kernel per call
// (PAPER.md:464, :496).  DESIGN.md "Lazy kernel" explains every deviation from the listing; in short:
//
//   state     one visited bitmap V and three rotating frontier bitmaps (level l reads F[(l-1)%3], marks F[l%3] and
//             clears F[(l+1)%3]); the paper's V_next XOR V_curr is F[l%3] AND NOT V.
//   top-down  Stage 1 consumes the list of non-zero frontier WORDS produced by the previous finalisation.  For every
//             newly active slice set it takes either the slice path -- the pull contraction over the
//             set's BVSS slices -- or, where the set has few active columns, the CSR edges of
//             its frontier vertices (the CUDA-core top-down path of north_star (e)).  Short segments are processed in
//             place, long ones (hub vertices / hub slice sets) are cut into equal chunks and spread over the grid.
//             Marks are filtered no-return atomic ORs.  Stage 2 is the finalisation sweep
//             (PAPER.md:399-446): L[u] = l once per discovered vertex, counters, next word list.
//   bottom-up Alg. 4 fused with its finalisation: the warp that owns word w of the visited bitmap
//             decides all 32 bits, so V, F_next, L and the counters are written in the same sweep (one barrier/level).
//   switch    start of each level: a byte-cost comparison of the two directions from the counters of the previous
//             finalisation (#unvisited as in Eq. 6, plus degree sums), scaled by eta.
//   hand-off  levels are written in internal ids (coalesced) and gathered into original ids once at the end (A10).
#include "bfs_kernels.cuh"

namespace blest {

namespace {

constexpr uint32_t FULL = 0xffffffffu;

struct LazyShared {
  unsigned long long acc[6];
  uint32_t wlCnt;
  uint32_t wlBase;
  uint32_t wl[WL_STAGE];
};

struct Counters {
  unsigned long long nnew = 0, unv = 0, mf = 0, scanned = 0, qbytes = 0;
};

// warp shuffle reduce -> shared atomics -> one global atomic per block and counter
__device__ __forceinline__ void block_accumulate(LazyShared& sh, const Counters& c, Ctrl* ctrl, uint32_t ci) {
  unsigned long long v[5] = {c.nnew, c.unv, c.mf, c.scanned, c.qbytes};
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
  for (uint32_t i = pos; i < WL_STAGE; ++i) sh.wl[i] = 0xFFFFFFFFu;
  return 0x80000000u | atomicAdd(wlc, cnt);
}
__device__ __forceinline__ void wl_store(LazyShared& sh, uint32_t* WLn, uint32_t slot, uint32_t w) {
  if (slot & 0x80000000u) WLn[slot & 0x7FFFFFFFu] = w;
  else sh.wl[slot] = w;
}

__device__ __forceinline__ uint32_t valid_mask(const BfsParams& p, uint32_t w) {
  return (w == p.nwords - 1 && (p.n & 31u)) ? ((1u << (p.n & 31u)) - 1u) : 0xFFFFFFFFu;
}

// Lazy mark: filtered no-return atomic OR into the next frontier.  V does not change during Stage 1,
// so its read may be served by L1; the frontier word is read at L2.
struct Marker {
  const uint32_t* V;
  uint32_t* Fn;
  __device__ __forceinline__ void operator()(uint32_t v) const {
    const uint32_t w = v >> 5, bit = 1u << (v & 31u);
    if (V[w] & bit) return;
    if (__ldcg(&Fn[w]) & bit) return;
    atomicOr(&Fn[w], bit);
  }
};

// ---- Stage 1 building blocks ------------------------------------------------------------------------------------
// Pull contraction over quads [a, a+nq) of one slice set with frontier word alpha: per lane a
// 128-bit row-id load and a 32-bit mask load, four quads in flight.  All 32 lanes take part (the MMA forms need it).
template <int CONTR>
__device__ __forceinline__ void warp_slices(const BfsParams& p, const Marker& mk, uint32_t a, uint32_t nq, uint32_t alpha,
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
        r[k] = __ldcs(p.rowIds + a + idx);
        m[k] = __ldcs(p.masks + a + idx);
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (base + 32u * k < nq) {  // warp-uniform
        const uint32_t hits = contract<CONTR>(m[k], alpha, lane);
        if (hits & 1u) mk(r[k].x);
        if (hits & 2u) mk(r[k].y);
        if (hits & 4u) mk(r[k].z);
        if (hits & 8u) mk(r[k].w);
      }
    }
  }
}

// CUDA-core top-down: every edge out of a frontier vertex is a mark candidate.
__device__ __forceinline__ void warp_edges(const BfsParams& p, const Marker& mk, uint32_t e0, uint32_t e1, uint32_t lane) {
  for (uint32_t base = e0; base < e1; base += 128u) {
    uint32_t v[4];
    bool ok[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t idx = base + 32u * k + lane;
      ok[k] = idx < e1;
      v[k] = ok[k] ? __ldcs(p.colidx + idx) : 0u;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (ok[k]) mk(v[k]);
  }
}

__device__ __forceinline__ void push_record(const BfsParams& p, Ctrl* ctrl, uint32_t ci, uint32_t type, uint32_t start,
                                            uint32_t count, uint32_t s) {
  const uint32_t per = type ? CHUNK_EDGES : CHUNK_QUADS;
  const uint32_t nent = (count + per - 1) / per;
  const uint32_t idx = atomicAdd(&ctrl->nBig[ci], 1u);
  const uint32_t pos = atomicAdd(&ctrl->qc[ci], nent);
  if (idx < p.recCap && (uint64_t)pos + nent <= p.chunkCap) p.recs[idx] = make_uint4(start, count, (s << 1) | type, pos);
  else atomicOr(&ctrl->error, 1u);
}

// Stage 1, top-down, phase A: one warp per non-zero frontier word.
template <int CONTR>
__device__ __forceinline__ void td_phase_a(const BfsParams& p, LazyShared& sh, const uint32_t* WLc, uint32_t wlCount,
                                           const uint32_t* Fp, uint32_t* Fn, Ctrl* ctrl, uint32_t ci) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  const Marker mk{p.V, Fn};
  const bool slicesAllowed = (p.switching != 3);
  const bool edgesAllowed = (p.switching != 1 && p.switching != 4);
  Counters c;
  for (uint32_t i = gwarp; i < wlCount; i += nwarps) {
    const uint32_t t = __ldcg(&WLc[i]);
    if (t == 0xFFFFFFFFu) continue;  // staging sentinel (wl_reserve)
    const uint32_t fw = Fp[t];
    const uint32_t u = t * 32u + lane;
    const bool mine = (fw >> lane) & 1u;
    uint32_t r0 = 0, deg = 0;
    if (mine) {
      r0 = __ldg(&p.rowptr[u]);
      deg = __ldg(&p.rowptr[u + 1]) - r0;
    }
    // the 8 lanes of group k = lane >> 3 stand for the 8 columns of slice set s = 4t + k
    uint32_t ds = deg;
    ds += __shfl_xor_sync(FULL, ds, 1);
    ds += __shfl_xor_sync(FULL, ds, 2);
    ds += __shfl_xor_sync(FULL, ds, 4);
    const uint32_t k = lane >> 3, s = t * 4u + k, byte = (fw >> (8u * k)) & 0xFFu;
    uint32_t a = 0, nq = 0;
    if (byte && slicesAllowed) {
      a = __ldg(&p.setPtr[s]);
      nq = __ldg(&p.setPtr[s + 1]) - a;
    }
    // slice path unless the set's active columns own fewer bytes as CSR edges (4 B per edge + row pointers) than
    // the whole set does as slices (20 B per quad); gamma scales the comparison (measured)
    bool useSlice = byte && nq && slicesAllowed;
    if (useSlice && edgesAllowed && 4.0f * (float)ds + 16.0f * (float)__popc(byte) < p.gamma * 20.0f * (float)nq) useSlice = false;
    const bool edgeMine = mine && !useSlice && deg > 0;
    if (edgeMine) c.qbytes += 4ull * deg;
    if (useSlice && (lane & 7u) == 0) c.qbytes += 20ull * nq;
    // (1) short adjacency lists: the owning lane scans them itself
    if (edgeMine && deg <= TINY_DEG)
      for (uint32_t e = r0; e < r0 + deg; ++e) mk(__ldcs(p.colidx + e));
    // (2) medium lists: the warp scans them together; long ones are deferred
    uint32_t pend = __ballot_sync(FULL, edgeMine && deg > TINY_DEG);
    while (pend) {
      const int srcLane = __ffs(pend) - 1;
      pend &= pend - 1;
      const uint32_t R0 = __shfl_sync(FULL, r0, srcLane), D = __shfl_sync(FULL, deg, srcLane);
      if (D <= BIG_EDGES) warp_edges(p, mk, R0, R0 + D, lane);
      else if (lane == 0) push_record(p, ctrl, ci, 1u, R0, D, 0u);
    }
    // (3) slice sets: contraction over the set's quads; hub sets are deferred
    uint32_t pendS = __ballot_sync(FULL, useSlice && (lane & 7u) == 0);
    while (pendS) {
      const int srcLane = __ffs(pendS) - 1;
      pendS &= pendS - 1;
      const uint32_t A = __shfl_sync(FULL, a, srcLane), NQ = __shfl_sync(FULL, nq, srcLane);
      const uint32_t AL = __shfl_sync(FULL, byte, srcLane), S = __shfl_sync(FULL, s, srcLane);
      if (NQ <= BIG_QUADS) warp_slices<CONTR>(p, mk, A, NQ, AL, lane);
      else if (lane == 0) push_record(p, ctrl, ci, 0u, A, NQ, S);
    }
  }
  block_accumulate(sh, c, ctrl, ci);
}

// Phase B1: one warp per deferred segment writes its chunk entries (32 per step).
__device__ __forceinline__ void td_phase_b1(const BfsParams& p, uint32_t nBig) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  for (uint32_t r = gwarp; r < nBig; r += nwarps) {
    const uint4 rec = p.recs[r];
    const uint32_t type = rec.z & 1u, s = rec.z >> 1, per = type ? CHUNK_EDGES : CHUNK_QUADS;
    const uint32_t nent = (rec.y + per - 1) / per;
    for (uint32_t i = lane; i < nent; i += 32) p.chunks[rec.w + i] = make_uint4(rec.x + i * per, min(per, rec.y - i * per), s, type);
  }
}

// Phase B2: one warp per chunk, round-robin: every warp gets the same share of the hubs' bytes.
template <int CONTR>
__device__ __forceinline__ void td_phase_b2(const BfsParams& p, uint32_t nChunks, const uint32_t* Fp, uint32_t* Fn) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  const Marker mk{p.V, Fn};
  const uint8_t* Fbytes = reinterpret_cast<const uint8_t*>(Fp);
  for (uint32_t i = gwarp; i < nChunks; i += nwarps) {
    const uint4 e = __ldcg(&p.chunks[i]);
    if (e.w) warp_edges(p, mk, e.x, e.x + e.y, lane);
    else warp_slices<CONTR>(p, mk, e.x, e.y, Fbytes[e.z], lane);
  }
}

// Stage 2 after a top-down Stage 1: frontier finalisation (readings R9/R10).
__device__ __forceinline__ void td_finalize(const BfsParams& p, LazyShared& sh, uint32_t level, uint32_t* Fn, uint32_t* Fs,
                                            uint32_t* WLn, Ctrl* ctrl, uint32_t ci) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  Counters c;
  for (uint32_t wb = gwarp * 32u; wb < p.nSweepWords; wb += nwarps * 32u) {
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
    uint32_t nz = __ballot_sync(FULL, fm != 0);
    if (nz) {
      // next level's work list (PAPER.md:420-440 enqueues the VSSs of every newly active slice set; here the non-zero
      // frontier word is the unit, expanded at consumption time)
      uint32_t base = 0;
      if (lane == 0) base = wl_reserve(sh, &ctrl->wlc[ci], (uint32_t)__popc(nz));
      base = __shfl_sync(FULL, base, 0);
      if (fm) wl_store(sh, WLn, base + __popc(nz & ((1u << lane) - 1u)), t);
      // L[u] = level once per discovered vertex, 32 consecutive vertices per step; degree sum for the switch
      while (nz) {
        const int srcLane = __ffs(nz) - 1;
        nz &= nz - 1;
        const uint32_t f = __shfl_sync(FULL, fm, srcLane);
        if ((f >> lane) & 1u) {
          const uint32_t u = (wb + srcLane) * 32u + lane;
          p.L[u] = (int32_t)level;
          c.mf += __ldg(&p.rowptr[u + 1]) - __ldg(&p.rowptr[u]);
        }
      }
    }
  }
  wl_flush(sh, WLn, &ctrl->wlc[ci]);
  block_accumulate(sh, c, ctrl, ci);
}

// Bottom-up level (Alg. 4, :466-494) fused with its finalisation.  Four words per warp step: the loads of
// the visited words, row pointers, first neighbours and their frontier bits are independent across the four.
__device__ __forceinline__ void bu_level(const BfsParams& p, LazyShared& sh, uint32_t level, const uint32_t* Fp, uint32_t* Fn,
                                         uint32_t* Fs, uint32_t* WLn, Ctrl* ctrl, uint32_t ci) {
  constexpr int K = 4;
  constexpr uint32_t SERIAL_CAP = 64;
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  const uint32_t nSW = p.nSweepWords;
  Counters c;
  auto in_frontier = [&](uint32_t v) -> bool { return (Fp[v >> 5] >> (v & 31u)) & 1u; };
  for (uint32_t w0 = gwarp; w0 < nSW; w0 += nwarps * K) {
    uint32_t cur[K], b[K], e[K];
    bool act[K], found[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const uint32_t w = w0 + k * nwarps;
      cur[k] = (w < nSW) ? __ldcg(&p.V[w]) : 0xFFFFFFFFu;
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const uint32_t w = w0 + k * nwarps;
      const uint32_t unv = (w < nSW) ? (~cur[k] & valid_mask(p, w)) : 0u;  // padding bits read as visited (R11)
      act[k] = (unv >> lane) & 1u;
      b[k] = e[k] = 0;
      if (act[k]) {
        const uint32_t u = w * 32u + lane;
        b[k] = __ldg(&p.rowptr[u]);
        e[k] = __ldg(&p.rowptr[u + 1]);
      }
    }
    uint32_t v0[K];
#pragma unroll
    for (int k = 0; k < K; ++k) v0[k] = (b[k] < e[k]) ? __ldg(&p.colidx[b[k]]) : 0xFFFFFFFFu;
#pragma unroll
    for (int k = 0; k < K; ++k) {
      found[k] = false;
      if (v0[k] != 0xFFFFFFFFu) {
        found[k] = in_frontier(v0[k]);
        ++c.scanned;
      }
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
      // remaining neighbours: the owning lane scans a bounded number, the warp finishes long lists together
      uint32_t ptr = b[k] + 1;
      bool more = false;
      if (b[k] < e[k] && !found[k]) {
        const uint32_t stop = min(e[k], ptr + SERIAL_CAP);
        for (; ptr < stop; ++ptr) {
          ++c.scanned;
          if (in_frontier(__ldg(&p.colidx[ptr]))) { found[k] = true; break; }
        }
        more = !found[k] && ptr < e[k];
      }
      uint32_t pend = __ballot_sync(FULL, more);
      while (pend) {
        const int srcLane = __ffs(pend) - 1;
        pend &= pend - 1;
        const uint32_t B = __shfl_sync(FULL, ptr, srcLane), E = __shfl_sync(FULL, e[k], srcLane);
        bool f = false;
        for (uint32_t base = B; base < E; base += 32u) {
          const uint32_t idx = base + lane;
          const bool h = idx < E && in_frontier(__ldg(&p.colidx[idx]));
          c.scanned += idx < E;
          if (__ballot_sync(FULL, h)) { f = true; break; }
        }
        if ((int)lane == srcLane) found[k] = f;
      }
    }
    uint32_t wl[K], wlN = 0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
      const uint32_t w = w0 + k * nwarps;
      const uint32_t fm = __ballot_sync(FULL, found[k]);
      if (w < nSW) {
        if (found[k]) {
          p.L[w * 32u + lane] = (int32_t)level;  // coalesced: lane = bit index
          c.mf += e[k] - b[k];
        }
        if (lane == 0) {
          if (fm) p.V[w] = cur[k] | fm;  // this warp owns word w: no atomic (PAPER.md:483 needs one per lane)
          Fn[w] = fm;
          Fs[w] = 0;
          c.nnew += __popc(fm);
          c.unv += __popc(~(cur[k] | fm) & valid_mask(p, w));
          if (fm) wl[wlN++] = w;
        }
      }
    }
    if (lane == 0 && wlN) {
      const uint32_t base = wl_reserve(sh, &ctrl->wlc[ci], wlN);
      for (uint32_t i = 0; i < wlN; ++i) wl_store(sh, WLn, base + i, wl[i]);
    }
  }
  wl_flush(sh, WLn, &ctrl->wlc[ci]);
  block_accumulate(sh, c, ctrl, ci);
}

// Direction of level `level` (Eq. 6 analogue).  All threads evaluate it on the same
// counters, so the decision is grid-uniform.
__device__ __forceinline__ bool choose_bottom_up(const BfsParams& p, uint32_t level, unsigned long long nf,
                                                 unsigned long long mf, unsigned long long nu, unsigned long long mu) {
  if (p.switching == 2) return true;
  if (p.switching == 5) return (p.buMask >> min(level, 31u)) & 1u;
  if (p.switching != 0) return false;
  // bytes each direction is expected to move: top-down reads every edge out of the frontier; bottom-up sweeps the
  // visited bitmap, reads the row pointers and first neighbours of every unvisited vertex and a fraction of the
  // remaining unvisited edges
  const float costTd = 4.0f * (float)mf + 32.0f * (float)nf;
  const float costBu = 12.0f * (float)p.nSweepWords + 48.0f * (float)nu + 0.5f * (float)mu;
  return costBu * 10.0f < p.eta * costTd;
}

template <int CONTR>
__global__ void __launch_bounds__(BLOCK_THREADS, 1) bfs_lazy_kernel(const __grid_constant__ BfsParams p) {
  __shared__ LazyShared sh;
  unsigned int epoch = 0;
  Ctrl* ctrl = p.ctrl;
  const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (uint64_t)gridDim.x * blockDim.x;
  const bool leader = (blockIdx.x == 0 && threadIdx.x == 0);
  if (threadIdx.x < 6) sh.acc[threadIdx.x] = 0;
  if (threadIdx.x == 0) sh.wlCnt = 0;
  if (leader) ctrl->t0 = globaltimer();

  // A4 per-call init: bitmaps cleared, V = F_curr = {src}.  The level array is NOT initialised:
  // it is written once per discovered vertex and read only where V is set (hand-off below).
  const uint32_t nSW = p.nSweepWords, srcWord = p.src >> 5, srcBit = 1u << (p.src & 31u);
  for (uint64_t i = gtid; i < nSW; i += nth) {
    const uint32_t x = (i == srcWord) ? srcBit : 0u;
    p.V[i] = x;
    p.F[0][i] = x;
    p.F[1][i] = 0;
    p.F[2][i] = 0;
  }
  const uint32_t srcDeg = __ldg(&p.rowptr[p.src + 1]) - __ldg(&p.rowptr[p.src]);
  if (leader) {
    // level 0: the source itself (L[src] = 0, frontier = {src})
    p.L[p.src] = 0;
    p.WL[0][0] = srcWord;
    ctrl->wlc[0] = 1;
    ctrl->newcount[0] = 1;
    ctrl->mf[0] = srcDeg;
    ctrl->unvisited[0] = (unsigned long long)min((uint64_t)p.n, (uint64_t)nSW * 32u) - 1u;
  }
  grid_barrier(&ctrl->bar, epoch);

  unsigned long long degVisited = 0;  // sum of degrees of all visited vertices
  uint32_t level = 1;
  for (;; ++level) {
    const uint32_t cp = (level - 1) % 3u, ci = level % 3u, cn = (level + 1) % 3u;
    const unsigned long long nf = ld_volatile(&ctrl->newcount[cp]);
    if (nf == 0) break;  // empty frontier ("terminates at the first level with x = 0")
    const unsigned long long mf = ld_volatile(&ctrl->mf[cp]);
    const unsigned long long unvAll = ld_volatile(&ctrl->unvisited[cp]);
    const uint32_t wlCount = ld_volatile(&ctrl->wlc[cp]);
    degVisited += mf;
    const unsigned long long nu = unvAll > p.nIsoInSweep ? unvAll - p.nIsoInSweep : 0ull;
    const unsigned long long mu = p.nnz > degVisited ? p.nnz - degVisited : 0ull;
    const bool bottomUp = choose_bottom_up(p, level, nf, mf, nu, mu);
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
    unsigned long long tStage1 = 0;
    if (bottomUp) {
      bu_level(p, sh, level, Fp, Fn, Fs, p.WL[level & 1u], ctrl, ci);
      grid_barrier(&ctrl->bar, epoch);
      if (leader) tStage1 = globaltimer();
    } else {
      td_phase_a<CONTR>(p, sh, p.WL[(level - 1) & 1u], wlCount, Fp, Fn, ctrl, ci);
      grid_barrier(&ctrl->bar, epoch);
      const uint32_t nBig = ld_volatile(&ctrl->nBig[ci]);
      if (nBig) {  // hubs: cut into equal chunks, spread over the grid
        td_phase_b1(p, min(nBig, p.recCap));
        grid_barrier(&ctrl->bar, epoch);
        td_phase_b2<CONTR>(p, min(ld_volatile(&ctrl->qc[ci]), p.chunkCap), Fp, Fn);
        grid_barrier(&ctrl->bar, epoch);
      }
      if (leader) tStage1 = globaltimer();
      td_finalize(p, sh, level, Fn, Fs, p.WL[level & 1u], ctrl, ci);
      grid_barrier(&ctrl->bar, epoch);
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
      r.unvisited = (uint32_t)(ua + ((unsigned long long)p.n - min((uint64_t)p.n, (uint64_t)nSW * 32u)));
      r.reserved = bottomUp ? 0u : ld_volatile(&ctrl->nBig[ci]);
      r.t_ns = globaltimer() - ctrl->t0;
      r.t_stage1_ns = tStage1 - ctrl->t0;
      p.trace[level - 1] = r;
    }
  }
  if (leader) ctrl->nlevels = level - 1;

  // A10 hand-off: levels in original ids, -1 = unreachable ("infinity"; reading R1)
  if (p.perm) {
    for (uint64_t v = gtid; v < p.n; v += nth) {
      const uint32_t pv = __ldg(&p.perm[v]);
      int32_t r = -1;
      if ((pv >> 5) < nSW && ((p.V[pv >> 5] >> (pv & 31u)) & 1u)) r = p.L[pv];
      p.out[v] = r;
    }
  } else {
    for (uint64_t v = gtid; v < p.n; v += nth) {
      const uint32_t w = (uint32_t)(v >> 5);
      const bool vis = w < nSW && ((p.V[w] >> (v & 31u)) & 1u);
      if (!vis) p.out[v] = -1;
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
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSm, kernel, BLOCK_THREADS, 0) != cudaSuccess) return 0;
  return sms * (perSm > 0 ? 1 : 0);  // one CTA per SM: the cheapest grid barrier
}

template <class K>
cudaError_t coop_launch(K kernel, const BfsParams& p, int gridBlocks, cudaStream_t st) {
  void* args[] = {(void*)&p};
  return cudaLaunchCooperativeKernel((const void*)kernel, dim3(gridBlocks), dim3(BLOCK_THREADS), args, 0, st);
}

}  // namespace

cudaError_t launch_bfs_lazy(const BfsParams& p, int gridBlocks, cudaStream_t st) {
  switch (p.contraction) {
    case 2: return coop_launch(bfs_lazy_kernel<2>, p, gridBlocks, st);
    case 3: return coop_launch(bfs_lazy_kernel<3>, p, gridBlocks, st);
    default: return coop_launch(bfs_lazy_kernel<1>, p, gridBlocks, st);
  }
}

// A source of degree 0 reaches nothing (SURVEY.md §8(b) "A source of degree 0 is legal").
cudaError_t launch_isolated_source(int32_t* out, uint32_t n, uint32_t src, cudaStream_t st) {
  const int threads = 256;
  const int blocks = (int)std::min<uint64_t>(((uint64_t)n + threads - 1) / threads, 148ull * 8);
  isolated_source_kernel<<<blocks, threads, 0, st>>>(out, n, src);
  return cudaGetLastError();
}

int max_coop_blocks_lazy() { return coop_blocks(bfs_lazy_kernel<2>); }

}  // namespace blest
