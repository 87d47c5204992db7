// msbfs_kernels.cu -- bit-packed multi-source BFS (§6.1, Alg. 5) and closeness accumulation (§6.2, Eq. 7-8).
//
// kappa = 32*KW BFS instances share one kappa-bit word per vertex, stored at getVI(u, rho) = (u mod 8)*rho + u/8
// so that Stage 2's thread-per-slice-set sweep is coalesced.  One persistent cooperative kernel
// loops over ALL source batches (PAPER.md:635 invokes the kernel ceil(n/kappa) times; here the batch loop is
// inside the kernel, so a closeness run is a single launch).
//
// Contraction: Alg. 5 lines 16-30 loop over the active BFS instances c with one ballot + two MMAs each.  On sm_100a
// there is no binary MMA; the same Boolean product [128 slices x 8] x [8 x kappa] is evaluated for all kappa
// instances at once as M = OR_{j in mask} F_curr^kappa[column j]  (8 selected ORs of kappa-bit words per slice).
// The per-instance loop, and with it activeSets, disappears; the per-set OR "A" of Alg. 5 line 51
// still decides which slice sets are enqueued.  dirtySets is kept as in the paper.
#include <mutex>

#include "bfs_kernels.cuh"

namespace blest {

namespace {

struct MsShared {
  BigSeg bigList[WARPS_PER_BLOCK][BIG_CAP];
  uint32_t bigCnt[WARPS_PER_BLOCK];
  unsigned long long acc;
  unsigned int tailSlot;  // broadcast slot of grid_barrier_tail
  uint32_t perSource[256];
  uint32_t fset[WARPS_PER_BLOCK][8 * 8];  // per warp: the kappa-bit frontier words of the current set's 8 columns
  unsigned long long cnt[WARPS_PER_BLOCK][5];  // per warp (lane 0): queue entries, quads, slices probed, fresh row
                                               // updates, dirty slice sets swept -- totals for the roofline (p.stats)
};

// One kappa-bit word (KW 32-bit words, naturally aligned) moved with a single vector access.
template <int KW>
__device__ __forceinline__ void load_words(const uint32_t* base, uint64_t idx, uint32_t (&w)[KW]) {
  if (KW == 1) w[0] = __ldcg(base + idx);
  else if (KW == 2) {
    const uint2 v = __ldcg(reinterpret_cast<const uint2*>(base) + idx);
    w[0] = v.x; w[KW > 1 ? 1 : 0] = v.y;
  } else {
#pragma unroll
    for (int q = 0; q < KW / 4; ++q) {
      const uint4 v = __ldcg(reinterpret_cast<const uint4*>(base) + idx * (KW / 4) + q);
      w[KW > 3 ? 4 * q : 0] = v.x; w[KW > 3 ? 4 * q + 1 : 0] = v.y; w[KW > 3 ? 4 * q + 2 : 0] = v.z; w[KW > 3 ? 4 * q + 3 : 0] = v.w;
    }
  }
}
template <int KW>
__device__ __forceinline__ void store_words(uint32_t* base, uint64_t idx, const uint32_t (&w)[KW]) {
  if (KW == 1) base[idx] = w[0];
  else if (KW == 2) reinterpret_cast<uint2*>(base)[idx] = make_uint2(w[0], w[KW > 1 ? 1 : 0]);
  else {
#pragma unroll
    for (int q = 0; q < KW / 4; ++q)
      reinterpret_cast<uint4*>(base)[idx * (KW / 4) + q] =
          make_uint4(w[KW > 3 ? 4 * q : 0], w[KW > 3 ? 4 * q + 1 : 0], w[KW > 3 ? 4 * q + 2 : 0], w[KW > 3 ? 4 * q + 3 : 0]);
  }
}
// No-return OR of the fresh bits, 64 bits per atomic where the word is that wide.
template <int KW>
__device__ __forceinline__ void red_or_words(uint32_t* base, uint64_t idx, const uint32_t (&f)[KW]) {
  if (KW == 1) {
    if (f[0]) atomicOr(base + idx, f[0]);
  } else {
#pragma unroll
    for (int h = 0; h < KW / 2; ++h) {
      const unsigned long long v = (unsigned long long)f[2 * h] | ((unsigned long long)f[KW > 1 ? 2 * h + 1 : 0] << 32);
      if (v) atomicOr(reinterpret_cast<unsigned long long*>(base) + idx * (KW / 2) + h, v);
    }
  }
}

template <int KW>
__device__ __forceinline__ void ms_stage1(const MsParams& p, MsShared& sh, const uint2* Qc, uint32_t qcount) {
  uint32_t* fset = sh.fset[threadIdx.x >> 5];
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5), nwarps = gridDim.x * WARPS_PER_BLOCK;
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
    // the first sigma lanes gather the kappa-bit frontier words of the set's 8 columns into shared
    // memory; every lane then reads the words its mask bits select (same address across lanes: a broadcast)
    __syncwarp();
    if (lane < 8) {
      uint32_t fv[KW];
      load_words<KW>(p.F, (uint64_t)lane * p.rho + s, fv);
#pragma unroll
      for (int w = 0; w < KW; ++w) fset[lane * KW + w] = fv[w];
    }
    __syncwarp();
    const uint32_t ru[4] = {rows.x, rows.y, rows.z, rows.w};
    uint32_t nProbe = 0, nFresh = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const uint32_t mb = (m >> (8 * c)) & 0xFFu;
      if (mb) {
        uint32_t M[KW];  // per-row kappa-bit accumulation buffer ("M[0..3]")
#pragma unroll
        for (int w = 0; w < KW; ++w) M[w] = 0;
        for (uint32_t b = mb; b; b &= b - 1) {  // M = OR over the set bits j of the mask of F_curr^kappa[column j]
          const uint32_t j = (uint32_t)__ffs(b) - 1u;
#pragma unroll
          for (int w = 0; w < KW; ++w) M[w] |= fset[j * KW + w];
        }
        const uint32_t u = ru[c];
        BLEST_ASSERT(u < p.n);
        const uint64_t idx = (uint64_t)(u & 7u) * p.rho + (u >> 3);  // getVI(u, rho)
        uint32_t any = 0;
#pragma unroll
        for (int w = 0; w < KW; ++w) any |= M[w];
        if (any) {  // one probe and one RED per row, each a single kappa-bit access
          uint32_t vn[KW], fresh[KW];
          load_words<KW>(p.Vn, idx, vn);
          ++nProbe;
          any = 0;
#pragma unroll
          for (int w = 0; w < KW; ++w) { fresh[w] = M[w] & ~vn[w]; any |= fresh[w]; }
          if (any) {
            red_or_words<KW>(p.Vn, idx, fresh);
            p.dirty[u >> 3] = 1;  // PAPER.md:583 dirtySets
            ++nFresh;
          }
        }
      }
    }
    if (p.stats) {
      const uint32_t tp = __reduce_add_sync(0xffffffffu, nProbe), tf = __reduce_add_sync(0xffffffffu, nFresh);
      if (lane == 0) {
        unsigned long long* cnt = sh.cnt[threadIdx.x >> 5];
        cnt[0] += 1; cnt[1] += nq; cnt[2] += tp; cnt[3] += tf;
      }
    }
  }
}

// PS: per-source counts (a source subset, reading R13) instead of the paper's target-side sums; a separate
// instantiation, so that its counters cost the all-vertices kernel no registers.
template <int KW, bool PS>
__device__ __forceinline__ void ms_stage2(const MsParams& p, MsShared& sh, uint32_t level, uint64_t b0, uint32_t nb,
                                          uint2* Qn, uint32_t tBase) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  BigSeg* bigList = sh.bigList[warp];
  uint32_t* bigCnt = &sh.bigCnt[warp];
  constexpr bool perSource = PS;
  uint32_t pacc[KW];  // per-source counts of this sweep kept by lane c mod 32 for instance c = 32 w + lane
#pragma unroll
  for (int w = 0; w < KW; ++w) pacc[w] = 0;
  for (uint64_t sb = (uint64_t)gwarp * 32; sb < p.Ns; sb += (uint64_t)nwarps * 32) {
    const uint32_t s = (uint32_t)sb + lane;  // consecutive threads -> consecutive slice sets
    uint32_t cnt = 0, a = 0, nq = 0;
    const bool isDirty = s < p.Ns && p.dirty[s];
    if (p.stats) {
      const uint32_t nd = __popc(__ballot_sync(0xffffffffu, isDirty));
      if (lane == 0) sh.cnt[warp][4] += nd;
    }
    // skip slice sets nobody marked.  With per-source counts the block is entered by the whole warp as
    // soon as one lane's set is dirty (clean lanes carry zero words), so that the counting below is warp-uniform.
    if (perSource ? __any_sync(0xffffffffu, isDirty) : isDirty) {
      if (isDirty) p.dirty[s] = 0;
      uint32_t A = 0;
      constexpr uint32_t R = KW <= 2 ? 8u : (KW == 4 ? 4u : 2u);  // rows whose words are in flight together
#pragma unroll
      for (uint32_t j0 = 0; j0 < 8; j0 += R) {
        uint32_t nx[R][KW], cu[R][KW];
#pragma unroll
        for (uint32_t r = 0; r < R; ++r) {
          const uint64_t idx = (uint64_t)(j0 + r) * p.rho + s;
          if (isDirty) {
            load_words<KW>(p.Vn, idx, nx[r]);
            load_words<KW>(p.Vc, idx, cu[r]);
          } else {
#pragma unroll
            for (int w = 0; w < KW; ++w) nx[r][w] = cu[r][w] = 0;
          }
        }
#pragma unroll
        for (uint32_t r = 0; r < R; ++r) {
          const uint32_t j = j0 + r;
          const uint64_t idx = (uint64_t)j * p.rho + s;
          uint32_t diff[KW], pc = 0, any = 0;
#pragma unroll
          for (int w = 0; w < KW; ++w) {
            diff[w] = nx[r][w] ^ cu[r][w];
            any |= diff[w];
            pc += __popc(diff[w]);
          }
          if (isDirty) store_words<KW>(p.F, idx, diff);  // PAPER.md:610 (unconditional for a swept set)
          if (perSource) {
            // Per-source counts (reading R13) = a positional popcount over the vertices: how many of the warp's 32 rows
            // have bit c set, for every instance c.  Few bits: one shared-memory atomic each.  Many (the dense middle
            // levels, where those atomics would pile up on kappa addresses): bit-sliced, one ballot per instance, the
            // count kept by lane c mod 32 in a register.
            const uint32_t tot = __reduce_add_sync(0xffffffffu, pc);
            if (tot > 32u) {
#pragma unroll
              for (int w = 0; w < KW; ++w) {
#pragma unroll 8
                for (uint32_t b = 0; b < 32u; ++b) {
                  const uint32_t k = (uint32_t)__popc(__ballot_sync(0xffffffffu, (diff[w] >> b) & 1u));
                  if (lane == b) pacc[w] += k;
                }
              }
            } else if (any) {
#pragma unroll
              for (int w = 0; w < KW; ++w)
                for (uint32_t d = diff[w]; d; d &= d - 1) atomicAdd(&sh.perSource[w * 32u + (__ffs(d) - 1)], 1u);
            }
          }
          if (any) {
            store_words<KW>(p.Vc, idx, nx[r]);
            A |= any;
            if (p.levels) {
              const uint32_t u = s * 8u + j;
              const uint32_t uo = p.iperm ? __ldg(&p.iperm[u]) : u;
#pragma unroll
              for (int w = 0; w < KW; ++w)
                for (uint32_t d = diff[w]; d; d &= d - 1) {
                  const uint32_t c = w * 32u + (__ffs(d) - 1);
                  BLEST_ASSERT(c < nb && uo < p.n);
                  p.levels[(b0 + c) * (uint64_t)p.n + uo] = (int32_t)level;
                }
            }
            if (p.farT) p.farT[idx] += (unsigned long long)level * pc;  // Eq. 7: far[idx] += l * popc(diff)
            if (p.reachT) p.reachT[idx] += pc;
          }
        }
      }
      if (A) {  // active in at least one BFS: enqueue all VSSs of the set
        a = __ldg(&p.setPtr[s]);
        nq = __ldg(&p.setPtr[s + 1]) - a;
        cnt = seg_entries(0, nq);
      }
    }
    bool ok;
    // one monotone queue tail for the whole launch (it shares the barrier's word, see grid_barrier_tail); positions
    // are relative to the tail at the start of this sweep; modular arithmetic makes a 32-bit wrap harmless
    uint32_t pos = warp_reserve(&p.ctrl->tail, cnt, lane, 0xFFFFFFFFu, &p.ctrl->error, ok) - tBase;
    {
      const uint32_t tot = __reduce_add_sync(0xffffffffu, cnt), first = __shfl_sync(0xffffffffu, pos, 0);
      ok = tot == 0u || (uint64_t)first + tot <= p.qcap;
      if (!ok && lane == 0) report_overflow(p.ctrl, p.hostStatus);
    }
    BLEST_ASSERT(!(cnt && ok) || (uint64_t)pos + cnt <= p.qcap);
    if (cnt && ok) emit_segment(Qn, pos, 0, a, nq, s, bigList, bigCnt);
    flush_big_segments(Qn, bigList, bigCnt, lane);
  }
  if (perSource) {
#pragma unroll
    for (int w = 0; w < KW; ++w)
      if (pacc[w]) atomicAdd(&sh.perSource[w * 32u + lane], pacc[w]);
  }
  __syncthreads();
  if (perSource && threadIdx.x < nb) {
    const uint32_t k = sh.perSource[threadIdx.x];
    if (k) {
      if (p.farS) atomicAdd(&p.farS[b0 + threadIdx.x], (unsigned long long)level * k);
      if (p.reachS) atomicAdd(&p.reachS[b0 + threadIdx.x], k);
    }
  }
  __syncthreads();
  if (threadIdx.x < 256) sh.perSource[threadIdx.x] = 0;
  __syncthreads();
}

template <int KW, bool PS>
__global__ void __launch_bounds__(BLOCK_THREADS, 1) msbfs_kernel(const __grid_constant__ MsParams p) {
  __shared__ MsShared sh;
  constexpr uint32_t KAPPA = 32u * KW;
  unsigned int epoch = 0;
  Ctrl* ctrl = p.ctrl;
  const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (uint64_t)gridDim.x * blockDim.x;
  if (threadIdx.x < WARPS_PER_BLOCK) sh.bigCnt[threadIdx.x] = 0;
  if (threadIdx.x < 256) sh.perSource[threadIdx.x] = 0;
  if (threadIdx.x == 0) sh.acc = 0;
  if (threadIdx.x < WARPS_PER_BLOCK * 5) sh.cnt[threadIdx.x / 5][threadIdx.x % 5] = 0;
  __syncthreads();
  const uint64_t stateWords = (uint64_t)p.rho * 8u * KW;
  unsigned long long nLevels = 0, nBatches = 0;

  uint32_t tStart = 0, tEnd = 0;  // queue tail before / after the sweep that filled the current level's queue
  for (uint64_t b0 = 0; b0 < p.nsrcs; b0 += KAPPA) {
    const uint32_t nb = (uint32_t)min((uint64_t)KAPPA, p.nsrcs - b0);
    // init(srcs, ...) (reading R16): visited words cleared, bit c of source c set, its set marked dirty
    grid_fill32(p.Vc, 0u, stateWords);
    grid_fill32(p.Vn, 0u, stateWords);
    if (p.levels) {
      uint32_t* base = reinterpret_cast<uint32_t*>(p.levels + b0 * (uint64_t)p.n);
      for (uint64_t i = gtid; i < (uint64_t)nb * p.n; i += nth) base[i] = 0xFFFFFFFFu;
    }
    grid_barrier(&ctrl->bar, epoch);
    if (gtid < nb) {
      const uint32_t c = (uint32_t)gtid;
      const uint32_t so = p.srcs ? p.srcs[b0 + c] : (uint32_t)(p.srcBase + b0 + c);
      const uint32_t si = p.perm ? __ldg(&p.perm[so]) : so;
      const uint64_t idx = (uint64_t)(si & 7u) * p.rho + (si >> 3);
      atomicOr(&p.Vn[idx * KW + (c >> 5)], 1u << (c & 31u));
      p.dirty[si >> 3] = 1;
    }
    grid_barrier(&ctrl->bar, epoch);
    // level 0 = the finalisation sweep over the sources themselves (far += 0, reach += 1, level 0, enqueue their sets)
    ms_stage2<KW, PS>(p, sh, 0, b0, nb, p.Q[1], tEnd);
    {
      const uint32_t t = grid_barrier_tail(&ctrl->bar, epoch, &sh.tailSlot);
      tStart = tEnd;
      tEnd = t;
    }
    for (uint32_t level = 1;; ++level) {
      const uint32_t par = level & 1u;
      // a level whose sweep enqueued nothing discovered nothing (every discovered vertex has a neighbour, so its slice
      // set has slices): the queue length the barrier returned is the termination test
      const uint32_t qcount = min(tEnd - tStart, p.qcap);  // (after an overflow the tail counts dropped entries)
      if (qcount == 0) break;
      ++nLevels;
      ms_stage1<KW>(p, sh, p.Q[par], qcount);
      grid_barrier(&ctrl->bar, epoch);
      ms_stage2<KW, PS>(p, sh, level, b0, nb, p.Q[par ^ 1u], tEnd);
      const uint32_t t = grid_barrier_tail(&ctrl->bar, epoch, &sh.tailSlot);
      tStart = tEnd;
      tEnd = t;
    }
    ++nBatches;
  }
  if (p.stats) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) {
      const unsigned long long* cnt = sh.cnt[threadIdx.x >> 5];
#pragma unroll
      for (int k = 0; k < 5; ++k)
        if (cnt[k]) atomicAdd(&p.stats[k], cnt[k]);
    }
    if (gtid == 0) { p.stats[5] = nLevels; p.stats[6] = nBatches; }
  }
}

__global__ void closeness_finalize_kernel(uint32_t n, uint32_t rho, const uint32_t* perm, const unsigned long long* farT,
                                          const uint32_t* reachT, const unsigned long long* farS, const uint32_t* reachS,
                                          uint64_t nsrcs, double* cc, unsigned long long* farOut, uint32_t* reachOut) {
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nsrcs; i += (uint64_t)gridDim.x * blockDim.x) {
    unsigned long long far;
    uint32_t reach;
    if (farT) {  // target-side sums (reading R13): source i = original vertex i
      const uint32_t ui = perm ? perm[i] : (uint32_t)i;
      const uint64_t idx = (uint64_t)(ui & 7u) * rho + (ui >> 3);
      far = farT[idx];
      reach = reachT[idx];
    } else {
      far = farS[i];
      reach = reachS[i];
    }
    if (farOut) farOut[i] = far;
    if (reachOut) reachOut[i] = reach;
    // Eq. 8 with the component-size normalisation (reading R14): one IEEE fp64 division
    if (cc) cc[i] = far == 0 ? 0.0 : (double)(reach - 1u) / (double)far;
  }
}

template <class K>
int coop_blocks(K kernel) {
  int dev = 0, sms = 0, perSm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSm, kernel, BLOCK_THREADS, 0) != cudaSuccess) return 0;
  return sms * (perSm > 0 ? 1 : 0);
}

}  // namespace

cudaError_t launch_msbfs(const MsParams& p, int gridBlocks, cudaStream_t st) {
  void* args[] = {(void*)&p};
  const void* k = nullptr;
  const bool ps = p.farS != nullptr || p.reachS != nullptr;
  switch (p.kappa) {
    case 32: k = ps ? (const void*)msbfs_kernel<1, true> : (const void*)msbfs_kernel<1, false>; break;
    case 64: k = ps ? (const void*)msbfs_kernel<2, true> : (const void*)msbfs_kernel<2, false>; break;
    case 128: k = ps ? (const void*)msbfs_kernel<4, true> : (const void*)msbfs_kernel<4, false>; break;
    case 256: k = ps ? (const void*)msbfs_kernel<8, true> : (const void*)msbfs_kernel<8, false>; break;
    default: return cudaErrorInvalidValue;
  }
  return cudaLaunchCooperativeKernel(k, dim3(gridBlocks), dim3(BLOCK_THREADS), args, 0, st);
}

cudaError_t launch_closeness_finalize(uint32_t n, uint32_t rho, const uint32_t* perm, const unsigned long long* farT,
                                      const uint32_t* reachT, const unsigned long long* farS, const uint32_t* reachS,
                                      uint64_t nsrcs, double* cc, unsigned long long* farOut, uint32_t* reachOut,
                                      cudaStream_t st) {
  const int threads = 256;
  const int blocks = (int)std::min<uint64_t>((nsrcs + threads - 1) / threads, 148ull * 8);
  closeness_finalize_kernel<<<blocks > 0 ? blocks : 1, threads, 0, st>>>(n, rho, perm, farT, reachT, farS, reachS, nsrcs, cc,
                                                                          farOut, reachOut);
  return cudaGetLastError();
}

// ---- allocation-free entry (blest_closeness_noalloc) ---------------------------------------------------------------
// Some callers cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// For them the scratch of ONE multi-source call lives in this file-scope device array (about 6.2 MiB, held by every GPU
// that loads the library until the process exits):
//   [ F | Vc | Vn ]   3 x NOALLOC_MAX_STATE_BYTES   the kappa-bit state arrays
//   [ dirty ]         NOALLOC_MAX_SETS bytes        dirtySets
//   [ farS ]          NOALLOC_MAX_SRCS x 8          per-source farness   (must start at zero)
//   [ reachS ]        NOALLOC_MAX_SRCS x 4          per-source reach     (must start at zero)
//   [ srcs ]          NOALLOC_MAX_SRCS x 4          sanitised copy of the caller's source ids
// All calls of the process share it and it keeps the last call's contents: dirty / farS / reachS are cleared at the
// start of every call (stream-ordered memsets), F / Vc / Vn are cleared or written by the kernel before they are read.
// Two calls that overlap on the GPU (different streams, no ordering) race on it.
namespace {
constexpr size_t NA_OFF_F = 0, NA_OFF_VC = NOALLOC_MAX_STATE_BYTES, NA_OFF_VN = 2 * NOALLOC_MAX_STATE_BYTES;
constexpr size_t NA_OFF_DIRTY = 3 * NOALLOC_MAX_STATE_BYTES;
constexpr size_t NA_OFF_FAR = NA_OFF_DIRTY + NOALLOC_MAX_SETS;
constexpr size_t NA_OFF_REACH = NA_OFF_FAR + (size_t)NOALLOC_MAX_SRCS * 8;
constexpr size_t NA_OFF_SRCS = NA_OFF_REACH + (size_t)NOALLOC_MAX_SRCS * 4;
constexpr size_t NA_BYTES = NA_OFF_SRCS + (size_t)NOALLOC_MAX_SRCS * 4;
static_assert(NA_OFF_FAR % 256 == 0 && NA_OFF_REACH % 256 == 0 && NA_OFF_SRCS % 256 == 0, "sub-arrays stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_noallocScratch[NA_BYTES];

// In host code `g_noallocScratch` is a host-side stand-in, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, once per device, with that device current.
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_naMutex;
unsigned char* g_naPtr[NA_MAX_DEVICES] = {};

cudaError_t noalloc_scratch(unsigned char** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_naMutex);
  if (!g_naPtr[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_noallocScratch);
    if (e != cudaSuccess) return e;
    g_naPtr[dev] = static_cast<unsigned char*>(ptr);
  }
  *out = g_naPtr[dev];
  return cudaSuccess;
}

// Sanitised copy of the caller's source ids into the scratch (device code names the array directly).
__global__ void noalloc_copy_srcs_kernel(const uint32_t* __restrict__ srcs, uint32_t nsrcs, uint32_t n) {
  uint32_t* dst = reinterpret_cast<uint32_t*>(g_noallocScratch + NA_OFF_SRCS);
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < nsrcs; i += gridDim.x * blockDim.x) dst[i] = min(srcs[i], n - 1u);
}
}  // namespace

cudaError_t launch_closeness_noalloc(MsParams p, const uint32_t* srcsDev, uint32_t nsrcs, int gridBlocks, double* out,
                                     cudaStream_t st) {
  unsigned char* base = nullptr;
  cudaError_t e = noalloc_scratch(&base);
  if (e != cudaSuccess) return e;
  p.F = reinterpret_cast<uint32_t*>(base + NA_OFF_F);
  p.Vc = reinterpret_cast<uint32_t*>(base + NA_OFF_VC);
  p.Vn = reinterpret_cast<uint32_t*>(base + NA_OFF_VN);
  p.dirty = base + NA_OFF_DIRTY;
  p.farS = reinterpret_cast<unsigned long long*>(base + NA_OFF_FAR);
  p.reachS = reinterpret_cast<uint32_t*>(base + NA_OFF_REACH);
  p.srcs = reinterpret_cast<const uint32_t*>(base + NA_OFF_SRCS);
  p.srcBase = 0;
  p.nsrcs = nsrcs;
  p.farT = nullptr;
  p.reachT = nullptr;
  p.levels = nullptr;
  p.stats = nullptr;
  // what must start at zero (the array keeps the last call's contents): dirtySets and the per-source sums
  e = cudaMemsetAsync(base + NA_OFF_DIRTY, 0, NA_OFF_SRCS - NA_OFF_DIRTY, st);
  if (e != cudaSuccess) return e;
  noalloc_copy_srcs_kernel<<<(nsrcs + 255) / 256, 256, 0, st>>>(srcsDev, nsrcs, p.n);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  e = launch_msbfs(p, gridBlocks, st);
  if (e != cudaSuccess) return e;
  return launch_closeness_finalize(p.n, p.rho, nullptr, nullptr, nullptr, p.farS, p.reachS, nsrcs, out, nullptr, nullptr, st);
}

int max_coop_blocks_msbfs() {
  return std::min(std::min(coop_blocks(msbfs_kernel<4, false>), coop_blocks(msbfs_kernel<8, false>)),
                  std::min(coop_blocks(msbfs_kernel<4, true>), coop_blocks(msbfs_kernel<8, true>)));
}

}  // namespace blest
