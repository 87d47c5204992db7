// bfs_eager.cu -- single-source BLEST traversal with eager updates as ONE persistent cooperative kernel per call
// (PAPER.md:464, :496).
//
//   bfs_eager_kernel : Alg. 2 for low-U_div / high-diameter graphs: one barrier per level, no
//                      Theta(n) sweep; the frontier word is derived from the level array and the "first to activate a
//                      slice set" test is an atomicMax on a per-set level stamp (reading R12).
#include "bfs_kernels.cuh"

namespace blest {

namespace {

struct SharedScratch {
  BigSeg bigList[WARPS_PER_BLOCK][BIG_CAP];
  uint32_t bigCnt[WARPS_PER_BLOCK];
  uint32_t qcount;  // queue length of the level, read by one thread and broadcast
};

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
      if (lane == 0) ctrl->tail = nent;
    } else if (lane == 0) report_overflow(ctrl, p.hostStatus);
  }
  // The queue tail is ONE monotone counter: the entries of level l+1 take positions [tEnd_l, tEnd_{l+1}) and live in
  // Q[(l+1) & 1] at (position - tEnd_l).  The barrier hands every CTA the tail, so no queue length is read or reset.
  uint32_t tStart = 0, tEnd = grid_barrier_tail(&ctrl->bar, epoch, &sh.qcount);

  uint32_t level = 1;
  for (;; ++level) {
    const uint32_t qcount = min(tEnd - tStart, p.qcap);  // (after an overflow the tail counts entries that were dropped)
    if (qcount == 0) break;
    const uint2* Qc = p.Q[level & 1u];
    uint2* Qn = p.Q[(level + 1) & 1u];
    BigSeg* bigList = sh.bigList[warp];
    uint32_t* bigCnt = &sh.bigCnt[warp];
    for (uint32_t i = gwarp; i < qcount; i += nwarps) {
      BLEST_ASSERT(i < p.qcap);
      const uint2 e = Qc[i];
      const uint32_t nq = (e.y & 31u) + 1u, s = e.y >> 5;
      BLEST_ASSERT(s < p.Ns && (uint64_t)e.x + nq <= p.nQuads);
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
      // the level of every row that hit, and (speculatively) the quad range of its slice set, in one round of loads
      int lu[4];
      uint32_t sa[4], sb[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        lu[c] = 0;
        sa[c] = sb[c] = 0;
        if ((hits >> c) & 1u) {
          BLEST_ASSERT(ru[c] < p.n);
          lu[c] = p.L[ru[c]];
          sa[c] = __ldg(&p.setPtr[ru[c] >> 3]);
          sb[c] = __ldg(&p.setPtr[(ru[c] >> 3) + 1]);
        }
      }
      int old[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        old[c] = (int)level;
        if (((hits >> c) & 1u) && lu[c] < 0) {  // "if l < L[u]"; benign same-value race
          p.L[ru[c]] = (int32_t)level;
          old[c] = atomicMax(&p.stamp[ru[c] >> 3], (int)level);  // PAPER.md:302-305 "old = 0": first to activate the set
        }
      }
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        if (old[c] < (int)level) {
          const uint32_t q = sb[c] - sa[c];
          if (q) { segA[nseg] = sa[c]; segN[nseg] = q; segS[nseg] = ru[c] >> 3; ++nseg; cnt += seg_entries(0, q); }
        }
      }
      bool ok;
      uint32_t pos = warp_reserve(&ctrl->tail, cnt, lane, 0xFFFFFFFFu, &ctrl->error, ok) - tEnd;
      {  // capacity of the next level's queue (the tail itself never wraps: every VSS is enqueued <= 8 times per call)
        const uint32_t tot = __reduce_add_sync(0xffffffffu, cnt), first = __shfl_sync(0xffffffffu, pos, 0);
        ok = tot == 0u || (uint64_t)first + tot <= p.qcap;
        if (!ok && lane == 0) report_overflow(ctrl, p.hostStatus);
      }
      BLEST_ASSERT(!ok || cnt == 0u || (uint64_t)pos + cnt <= p.qcap);
      if (ok)
        for (uint32_t k = 0; k < nseg; ++k) emit_segment(Qn, pos, 0, segA[k], segN[k], segS[k], bigList, bigCnt);
      flush_big_segments(Qn, bigList, bigCnt, lane);
    }
    tStart = tEnd;
    tEnd = grid_barrier_tail(&ctrl->bar, epoch, &sh.qcount);
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

cudaError_t launch_bfs_eager(const BfsParams& p, int gridBlocks, cudaStream_t st) {
  switch (p.contraction) {
    case 2: return coop_launch(bfs_eager_kernel<2>, p, gridBlocks, st);
    case 3: return coop_launch(bfs_eager_kernel<3>, p, gridBlocks, st);
    default: return coop_launch(bfs_eager_kernel<1>, p, gridBlocks, st);
  }
}
int max_coop_blocks_eager() { return coop_blocks(bfs_eager_kernel<2>); }

}  // namespace blest
