// bfs_kernels.cu -- single-source BLEST traversal as ONE persistent cooperative kernel per call.
//
//   bfs_lazy_kernel  : Alg. 3 (lazy two-stage) with, per level, either the work-queue stage
//                      (slice chunks = VSSs of active slice sets; plus CSR edge chunks where a slice set
//                      has few active columns -- the CUDA-core top-down path of north_star (e)) or the bottom-up
//                      CUDA-core stage (Alg. 4), chosen at the top of each level (Eq. 6 analogue).
//   bfs_eager_kernel : Alg. 2 for low-U_div / high-diameter graphs: one barrier per level, no
//                      Theta(n) sweep; the frontier word is derived from the level array and the "first to activate a
//                      slice set" test is an atomicMax on a per-set level stamp (reading R12).
#include "bfs_kernels.cuh"

namespace blest {

namespace {

struct SharedScratch {
  BigSeg bigList[WARPS_PER_BLOCK][BIG_CAP];
  uint32_t bigCnt[WARPS_PER_BLOCK];
  unsigned long long acc[4];
};

__device__ __forceinline__ void block_accumulate(SharedScratch& sh, unsigned long long v0, unsigned long long v1,
                                                 unsigned long long v2, unsigned long long v3, unsigned long long* g0,
                                                 unsigned long long* g1, unsigned long long* g2, unsigned long long* g3) {
  // warp shuffle reduce -> shared atomics -> one global atomic per block and counter
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    v0 += __shfl_down_sync(0xffffffffu, v0, d);
    v1 += __shfl_down_sync(0xffffffffu, v1, d);
    v2 += __shfl_down_sync(0xffffffffu, v2, d);
    v3 += __shfl_down_sync(0xffffffffu, v3, d);
  }
  if ((threadIdx.x & 31) == 0) {
    if (v0) atomicAdd(&sh.acc[0], v0);
    if (v1) atomicAdd(&sh.acc[1], v1);
    if (v2) atomicAdd(&sh.acc[2], v2);
    if (v3) atomicAdd(&sh.acc[3], v3);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (g0 && sh.acc[0]) atomicAdd(g0, sh.acc[0]);
    if (g1 && sh.acc[1]) atomicAdd(g1, sh.acc[1]);
    if (g2 && sh.acc[2]) atomicAdd(g2, sh.acc[2]);
    if (g3 && sh.acc[3]) atomicAdd(g3, sh.acc[3]);
    sh.acc[0] = sh.acc[1] = sh.acc[2] = sh.acc[3] = 0;
  }
  __syncthreads();
}

// Fill an int32/uint32 array of exactly `count` words with `value`, except index `special` which gets `sval`.
// Handles a destination that is only 4-byte aligned (caller-provided output buffers).
__device__ __forceinline__ void grid_fill_special(uint32_t* ptr, uint32_t value, uint64_t count, uint64_t special,
                                                  uint32_t sval) {
  const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (uint64_t)gridDim.x * blockDim.x;
  const uint64_t head = min(count, (uint64_t)((16u - ((uintptr_t)ptr & 15u)) & 15u) >> 2);
  const uint64_t n4 = (count - head) >> 2;
  uint4* p4 = reinterpret_cast<uint4*>(ptr + head);
  const uint4 v = make_uint4(value, value, value, value);
  for (uint64_t i = tid; i < n4; i += nth) p4[i] = v;
  const uint64_t tail0 = head + (n4 << 2);
  if (tid < head) ptr[tid] = value;
  if (tid < count - tail0) ptr[tail0 + tid] = value;
  // the owner of `special` rewrites it after its own vector store (same thread => ordered)
  if (special < count) {
    uint64_t owner;
    if (special < head) owner = special;
    else if (special >= tail0) owner = special - tail0;
    else owner = ((special - head) >> 2) % nth;
    if (tid == owner) ptr[special] = sval;
  }
}

// Decide, for one newly active slice set, between slice chunks (BVSS) and CSR edge chunks, and visit the resulting
// segments.  f(type, start, count, s).  Also returns the degree sum of the set's new frontier vertices.
template <class F>
__device__ __forceinline__ void visit_set_segments(const BfsParams& p, uint32_t s, uint32_t byte, bool tdEnabled,
                                                   unsigned long long& degSum, F&& f) {
  const uint32_t a = __ldg(&p.setPtr[s]), nq = __ldg(&p.setPtr[s + 1]) - a;
  bool td = false;
  if (tdEnabled) {
    uint32_t ds = 0;
    for (uint32_t b = byte; b; b &= b - 1) {
      const uint32_t u = s * 8u + (__ffs(b) - 1);
      ds += __ldg(&p.rowptr[u + 1]) - __ldg(&p.rowptr[u]);
    }
    degSum += ds;
    // bytes: 20 per quad (16 row ids + 4 masks) vs 4 per edge (+ 16 per vertex for the two row pointers and queue slack)
    td = (p.switching == 3) || ((float)(4u * ds + 16u * __popc(byte)) < p.gamma * (float)(20u * nq));
  }
  if (!td) {
    if (nq) f(0u, a, nq, s);
  } else {
    for (uint32_t b = byte; b; b &= b - 1) {
      const uint32_t u = s * 8u + (__ffs(b) - 1);
      const uint32_t r0 = __ldg(&p.rowptr[u]), r1 = __ldg(&p.rowptr[u + 1]);
      if (r1 > r0) f(1u, r0, r1 - r0, 0u);
    }
  }
}

// ---- Stage 2: frontier finalisation (Alg. 3 lines 33-50; reading R9/R10) ----------------------
__device__ __forceinline__ void stage2_finalize(const BfsParams& p, SharedScratch& sh, uint32_t level, uint2* Qn,
                                                unsigned int* qcn, unsigned long long* qbn, uint32_t par) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  const bool tdEnabled = (p.switching == 0 || p.switching == 3);
  unsigned long long unv = 0, nnew = 0, qb = 0, mf = 0;
  BigSeg* bigList = sh.bigList[warp];
  uint32_t* bigCnt = &sh.bigCnt[warp];
  for (uint64_t wb = (uint64_t)gwarp * 32; wb < p.nwords; wb += (uint64_t)nwarps * 32) {
    const uint32_t t = (uint32_t)wb + lane;
    uint32_t diff = 0, next = 0xFFFFFFFFu;
    if (t < p.nwords) {
      next = p.Vnext[t];
      const uint32_t cur = p.Vcurr[t];
      diff = next ^ cur;
      p.Fcurr[t] = diff;  // unconditional: no stale frontier words (reading R10)
      uint32_t valid = 0xFFFFFFFFu;
      if (t == p.nwords - 1 && (p.n & 31u)) valid = (1u << (p.n & 31u)) - 1u;
      unv += __popc(~next & valid);
    }
    uint32_t cnt = 0;
    if (diff) {
      p.Vcurr[t] = next;
      nnew += __popc(diff);
      for (uint32_t d = diff; d; d &= d - 1) {  // L[u] = level, once per discovered vertex
        const uint32_t u = t * 32u + (__ffs(d) - 1);
        p.out[p.iperm ? __ldg(&p.iperm[u]) : u] = (int32_t)level;
      }
#pragma unroll
      for (uint32_t set = 0; set < 4; ++set) {
        const uint32_t byte = (diff >> (8 * set)) & 0xFFu;
        if (byte)
          visit_set_segments(p, t * 4u + set, byte, tdEnabled, mf, [&](uint32_t type, uint32_t, uint32_t count, uint32_t) {
            cnt += seg_entries(type, count);
            qb += type ? 4ull * count : 20ull * count;
          });
      }
    }
    bool ok;
    uint32_t pos = warp_reserve(qcn, cnt, lane, p.qcap, &p.ctrl->error, ok);
    if (cnt && ok) {
      unsigned long long dummy = 0;
#pragma unroll
      for (uint32_t set = 0; set < 4; ++set) {
        const uint32_t byte = (diff >> (8 * set)) & 0xFFu;
        if (byte)
          visit_set_segments(p, t * 4u + set, byte, tdEnabled, dummy, [&](uint32_t type, uint32_t start, uint32_t count, uint32_t s) {
            emit_segment(Qn, pos, type, start, count, s, bigList, bigCnt);
          });
      }
    }
    flush_big_segments(Qn, bigList, bigCnt, lane);
  }
  block_accumulate(sh, unv, nnew, qb, mf, &p.ctrl->unvisited[par], &p.ctrl->newcount[par], qbn, &p.ctrl->mf[par]);
}

// ---- Stage 1, queue mode: pull contraction over slice chunks and CSR edge chunks ---------------
template <int CONTR>
__device__ __forceinline__ void stage1_queue(const BfsParams& p, const uint2* Qc, uint32_t qcount) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  const uint8_t* Fbytes = reinterpret_cast<const uint8_t*>(p.Fcurr);

  auto load_chunk = [&](uint2 e, uint4& rows, uint32_t& m, uint32_t& alpha) {
    rows = make_uint4(0, 0, 0, 0);
    m = 0;
    if (e.y & 0x80000000u) {  // CSR edge chunk: every edge out of a frontier vertex is a hit candidate
      const uint32_t cnt = e.y & 0x7FFFFFFFu;
      const uint32_t* c = p.colidx + e.x;
      if (lane < cnt) { rows.x = __ldg(c + lane); m |= 0xFFu; }
      if (lane + 32 < cnt) { rows.y = __ldg(c + lane + 32); m |= 0xFF00u; }
      if (lane + 64 < cnt) { rows.z = __ldg(c + lane + 64); m |= 0xFF0000u; }
      if (lane + 96 < cnt) { rows.w = __ldg(c + lane + 96); m |= 0xFF000000u; }
      alpha = 0xFFu;
    } else {  // slice chunk (one VSS): 128-bit row ids + 32-bit masks per lane, sigma-bit frontier word of the set
      const uint32_t nq = (e.y & 31u) + 1u, s = e.y >> 5;
      if (lane < nq) {
        rows = __ldg(p.rowIds + e.x + lane);
        m = __ldg(p.masks + e.x + lane);
      }
      alpha = Fbytes[s];
    }
  };
  auto mark = [&](uint32_t u) {  // lazy mark: filtered no-return atomic OR (RED) on V_next
    const uint32_t w = u >> 5, bit = 1u << (u & 31u);
    if (!(__ldcg(&p.Vnext[w]) & bit)) atomicOr(&p.Vnext[w], bit);
  };
  auto consume = [&](const uint4& rows, uint32_t m, uint32_t alpha) {
    const uint32_t hits = contract<CONTR>(m, alpha, lane);
    if (hits & 1u) mark(rows.x);
    if (hits & 2u) mark(rows.y);
    if (hits & 4u) mark(rows.z);
    if (hits & 8u) mark(rows.w);
  };

  uint32_t i = gwarp;
  for (; i + nwarps < qcount; i += 2 * nwarps) {  // two chunks in flight per warp
    const uint2 e0 = Qc[i], e1 = Qc[i + nwarps];
    uint4 r0, r1;
    uint32_t m0, m1, a0, a1;
    load_chunk(e0, r0, m0, a0);
    load_chunk(e1, r1, m1, a1);
    consume(r0, m0, a0);
    consume(r1, m1, a1);
  }
  if (i < qcount) {
    uint4 r0;
    uint32_t m0, a0;
    load_chunk(Qc[i], r0, m0, a0);
    consume(r0, m0, a0);
  }
}

// ---- Stage 1, bottom-up CUDA-core mode (Alg. 4) ------------------------------------------------
__device__ __forceinline__ void stage1_bottom_up(const BfsParams& p, SharedScratch& sh, uint32_t par) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
  unsigned long long scanned = 0;
  for (uint32_t w = gwarp; w < p.nwords; w += nwarps) {
    const uint32_t cur = p.Vcurr[w];
    uint32_t valid = 0xFFFFFFFFu;
    if (w == p.nwords - 1 && (p.n & 31u)) valid = (1u << (p.n & 31u)) - 1u;  // padding bits read as visited (R11)
    const uint32_t unv = ~cur & valid;
    bool found = false;
    if ((unv >> lane) & 1u) {
      const uint32_t u = w * 32u + lane;
      const uint32_t b = __ldg(&p.rowptr[u]), e = __ldg(&p.rowptr[u + 1]);
      for (uint32_t ptr = b; ptr < e; ++ptr) {
        const uint32_t v = __ldg(&p.colidx[ptr]);
        ++scanned;
        if ((p.Fcurr[v >> 5] >> (v & 31u)) & 1u) { found = true; break; }
      }
    }
    const uint32_t fm = __ballot_sync(0xffffffffu, found);
    if (lane == 0 && fm) p.Vnext[w] = cur | fm;  // this warp owns word w: no atomic needed
  }
  block_accumulate(sh, scanned, 0, 0, 0, &p.ctrl->buScanned[par], nullptr, nullptr, nullptr);
}

__device__ __forceinline__ bool choose_bottom_up(const BfsParams& p, uint32_t level, uint32_t unvisited,
                                                 unsigned long long qbytes, uint32_t qcount) {
  if (p.switching == 2) return true;
  if (p.switching == 5) return (p.buMask >> min(level, 31u)) & 1u;
  if (p.switching != 0) return false;
  // Eq. 6 restated in bytes: #unvisited < eta * |Q| with 640-byte VSSs  <=>  640 * #unvisited < eta * bytes(Q)
  return 640.0f * (float)unvisited < p.eta * (float)(qbytes + 8ull * qcount);
}

template <int CONTR>
__global__ void __launch_bounds__(BLOCK_THREADS, 1) bfs_lazy_kernel(const __grid_constant__ BfsParams p) {
  __shared__ SharedScratch sh;
  unsigned int epoch = 0;
  Ctrl* ctrl = p.ctrl;
  if (threadIdx.x < WARPS_PER_BLOCK) sh.bigCnt[threadIdx.x] = 0;
  if (threadIdx.x < 4) sh.acc[threadIdx.x] = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->t0 = globaltimer();

  // A4 per-call init: L = "infinity" (-1), bitmaps cleared, V_next = {src}.
  grid_fill_special(reinterpret_cast<uint32_t*>(p.out), 0xFFFFFFFFu, p.n, ~0ull, 0);
  grid_fill_special(p.Vcurr, 0u, p.nwords, ~0ull, 0);
  grid_fill_special(p.Vnext, 0u, p.nwords, p.src >> 5, 1u << (p.src & 31u));
  grid_barrier(&ctrl->bar, epoch);
  // Level 0 = the finalisation sweep over V_next = {src}: writes L[src] = 0, F_curr = {src}, enqueues src's slice set.
  stage2_finalize(p, sh, 0, p.Q[1], &ctrl->qc[1], &ctrl->qbytes[1], 0);
  grid_barrier(&ctrl->bar, epoch);

  uint32_t level = 1;
  for (;; ++level) {
    const uint32_t pp = (level - 1) & 1u, par = level & 1u;
    const unsigned long long newPrev = ld_volatile(&ctrl->newcount[pp]);
    if (newPrev == 0) break;  // empty frontier ("terminates at the first level with x = 0")
    const uint32_t qcount = ld_volatile(&ctrl->qc[par]);
    const unsigned long long qbytes = ld_volatile(&ctrl->qbytes[par]);
    const uint32_t unvPrev = (uint32_t)ld_volatile(&ctrl->unvisited[pp]);
    const bool bottomUp = choose_bottom_up(p, level, unvPrev, qbytes, qcount);
    // ---- Stage 1: lazy marking
    if (bottomUp) stage1_bottom_up(p, sh, par);
    else stage1_queue<CONTR>(p, p.Q[par], qcount);
    grid_barrier(&ctrl->bar, epoch);
    const unsigned long long tStage1 = (blockIdx.x == 0 && threadIdx.x == 0) ? globaltimer() : 0ull;
    // ---- Stage 2: frontier finalisation; counters consumed above are recycled here
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      ctrl->qc[par] = 0;
      ctrl->qbytes[par] = 0;
      ctrl->unvisited[pp] = 0;
      ctrl->newcount[pp] = 0;
      ctrl->mf[pp] = 0;
      ctrl->buScanned[pp] = 0;
    }
    stage2_finalize(p, sh, level, p.Q[par ^ 1u], &ctrl->qc[par ^ 1u], &ctrl->qbytes[par ^ 1u], par);
    grid_barrier(&ctrl->bar, epoch);
    if (blockIdx.x == 0 && threadIdx.x == 0 && p.trace && level - 1 < p.traceCap) {
      blest_level_trace_t r;
      r.level = level;
      r.mode = bottomUp ? 1u : 0u;
      r.q_entries = bottomUp ? 0u : qcount;
      r.new_vertices = (uint32_t)ld_volatile(&ctrl->newcount[par]);
      r.q_bytes = bottomUp ? 0ull : qbytes;
      r.bu_scanned = ld_volatile(&ctrl->buScanned[par]);
      r.unvisited = (uint32_t)ld_volatile(&ctrl->unvisited[par]);
      r.reserved = 0;
      r.t_ns = globaltimer() - ctrl->t0;
      r.t_stage1_ns = tStage1 - ctrl->t0;
      p.trace[level - 1] = r;
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->nlevels = level - 1;
}

// ---- Alg. 2: eager updates --------------------------------------------------------------------------------------
template <int CONTR>
__global__ void __launch_bounds__(BLOCK_THREADS, 1) bfs_eager_kernel(const __grid_constant__ BfsParams p) {
  __shared__ SharedScratch sh;
  unsigned int epoch = 0;
  Ctrl* ctrl = p.ctrl;
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  if (threadIdx.x < WARPS_PER_BLOCK) sh.bigCnt[threadIdx.x] = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->t0 = globaltimer();

  // init: L = -1 except L[src] = 0; set stamps = -1 except the source's set (level 0)
  grid_fill_special(reinterpret_cast<uint32_t*>(p.L), 0xFFFFFFFFu, p.n, p.src, 0u);
  grid_fill_special(reinterpret_cast<uint32_t*>(p.stamp), 0xFFFFFFFFu, p.Ns, p.src >> 3, 0u);
  if (gwarp == 0) {  // Q_curr = the VSSs of the source's slice set
    const uint32_t s0 = p.src >> 3, a = __ldg(&p.setPtr[s0]), nq = __ldg(&p.setPtr[s0 + 1]) - a;
    const uint32_t nent = seg_entries(0, nq);
    if (nent <= p.qcap) {
      for (uint32_t i = lane; i < nent; i += 32) write_entry(p.Q[1], 0, 0, a, nq, s0, i);
      if (lane == 0) ctrl->qc[1] = nent;
    } else if (lane == 0) atomicOr(&ctrl->error, 1u);
  }
  grid_barrier(&ctrl->bar, epoch);

  uint32_t level = 1;
  for (;; ++level) {
    const uint32_t qcount = ld_volatile(&ctrl->qc[level % 3u]);
    if (qcount == 0) break;
    const uint2* Qc = p.Q[level & 1u];
    uint2* Qn = p.Q[(level + 1) & 1u];
    unsigned int* qcn = &ctrl->qc[(level + 1) % 3u];
    if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->qc[(level + 2) % 3u] = 0;
    BigSeg* bigList = sh.bigList[warp];
    uint32_t* bigCnt = &sh.bigCnt[warp];
    for (uint32_t i = gwarp; i < qcount; i += nwarps) {
      const uint2 e = Qc[i];
      const uint32_t nq = (e.y & 31u) + 1u, s = e.y >> 5;
      uint4 rows = make_uint4(0, 0, 0, 0);
      uint32_t m = 0;
      if (lane < nq) {
        rows = __ldg(p.rowIds + e.x + lane);
        m = __ldg(p.masks + e.x + lane);
      }
      // frontier word alpha: column j of set s is in the frontier iff L[8s + j] == level - 1
      int lv = -2;
      if (lane < 8 && s * 8u + lane < p.n) lv = p.L[s * 8u + lane];
      const uint32_t alpha = __ballot_sync(0xffffffffu, lv == (int)level - 1) & 0xFFu;
      const uint32_t hits = contract<CONTR>(m, alpha, lane);
      uint32_t segA[4], segN[4], segS[4], nseg = 0, cnt = 0;
      const uint32_t ru[4] = {rows.x, rows.y, rows.z, rows.w};
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        if ((hits >> c) & 1u) {
          const uint32_t u = ru[c];
          if (p.L[u] < 0) {         // "if l < L[u]"; benign same-value race
            p.L[u] = (int32_t)level;
            const uint32_t so = u >> 3;
            const int old = atomicMax(&p.stamp[so], (int)level);  // PAPER.md:302-305 "old = 0": first to activate the set
            if (old < (int)level) {
              const uint32_t a = __ldg(&p.setPtr[so]), q = __ldg(&p.setPtr[so + 1]) - a;
              if (q) { segA[nseg] = a; segN[nseg] = q; segS[nseg] = so; ++nseg; cnt += seg_entries(0, q); }
            }
          }
        }
      }
      bool ok;
      uint32_t pos = warp_reserve(qcn, cnt, lane, p.qcap, &ctrl->error, ok);
      if (ok)
        for (uint32_t k = 0; k < nseg; ++k) emit_segment(Qn, pos, 0, segA[k], segN[k], segS[k], bigList, bigCnt);
      flush_big_segments(Qn, bigList, bigCnt, lane);
    }
    grid_barrier(&ctrl->bar, epoch);
    if (blockIdx.x == 0 && threadIdx.x == 0 && p.trace && level - 1 < p.traceCap) {
      blest_level_trace_t r;
      r.level = level;
      r.mode = 2u;
      r.q_entries = qcount;
      r.new_vertices = 0;
      r.q_bytes = 0;
      r.bu_scanned = 0;
      r.unvisited = 0;
      r.reserved = 0;
      r.t_ns = globaltimer() - ctrl->t0;
      r.t_stage1_ns = r.t_ns;
      p.trace[level - 1] = r;
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->nlevels = level - 1;
  // A10 hand-off: levels in original ids
  if (p.iperm) {
    for (uint64_t u = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; u < p.n; u += (uint64_t)gridDim.x * blockDim.x)
      p.out[__ldg(&p.iperm[u])] = p.L[u];
  }
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
cudaError_t launch_bfs_eager(const BfsParams& p, int gridBlocks, cudaStream_t st) {
  switch (p.contraction) {
    case 2: return coop_launch(bfs_eager_kernel<2>, p, gridBlocks, st);
    case 3: return coop_launch(bfs_eager_kernel<3>, p, gridBlocks, st);
    default: return coop_launch(bfs_eager_kernel<1>, p, gridBlocks, st);
  }
}
int max_coop_blocks_lazy() { return coop_blocks(bfs_lazy_kernel<2>); }
int max_coop_blocks_eager() { return coop_blocks(bfs_eager_kernel<2>); }

}  // namespace blest
