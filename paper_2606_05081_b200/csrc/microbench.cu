// microbench.cu -- in-repo evidence kernels: contraction self-test, tensor-pipe peak of the two
// MMA forms available to a warp on sm_100a, grid-barrier latency.
#include "bfs_kernels.cuh"

namespace blest {

namespace {

// Every (mask byte, alpha) pair in every byte position, warp-uniform alpha as in the traversal kernels.
template <int CONTR>
__global__ void contraction_selftest_kernel(unsigned long long* mismatches) {
  const uint32_t lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const uint32_t alpha = warp & 0xFFu;  // 256 warps cover all alphas
  unsigned long long bad = 0;
  for (uint32_t it = 0; it < 64; ++it) {
    // lane's four bytes: rotate through all 256 values in each position, different value per position
    const uint32_t b0 = (it * 4 + lane * 8 + 0) & 0xFFu, b1 = (it * 4 + lane * 8 + 85) & 0xFFu;
    const uint32_t b2 = (it * 4 + lane * 8 + 170) & 0xFFu, b3 = (255u - ((it * 4 + lane * 8) & 0xFFu));
    for (uint32_t k = 0; k < 4; ++k) {
      const uint32_t m = ((b0 + k) & 0xFFu) | (((b1 + k) & 0xFFu) << 8) | (((b2 + k) & 0xFFu) << 16) | (((b3 - k) & 0xFFu) << 24);
      const uint32_t got = contract<CONTR>(m, alpha, lane);
      uint32_t want = 0;
      for (uint32_t c = 0; c < 4; ++c) want |= ((((m >> (8 * c)) & 0xFFu) & alpha) != 0u ? 1u : 0u) << c;
      bad += (got != want);
    }
  }
  if (bad) atomicAdd(mismatches, bad);
}

// Tensor-pipe peak: ILP independent accumulator chains per warp, no memory traffic.
template <int KIND, int ILP>
__global__ void __launch_bounds__(1024, 1) mma_peak_kernel(uint32_t iters, int* sink) {
  int c[ILP][4];
#pragma unroll
  for (int i = 0; i < ILP; ++i) c[i][0] = c[i][1] = c[i][2] = c[i][3] = 0;
  const uint32_t a = threadIdx.x * 0x9E3779B9u, b = blockIdx.x * 0x85EBCA6Bu + 1u;
  for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
      if (KIND == 2) {
        asm volatile("mma.sync.aligned.m8n8k128.row.col.s32.b1.b1.s32.and.popc {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+r"(c[i][0]), "+r"(c[i][1]) : "r"(a + i), "r"(b));
      } else {
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                     : "+r"(c[i][0]), "+r"(c[i][1]), "+r"(c[i][2]), "+r"(c[i][3])
                     : "r"(a + i), "r"(a ^ b), "r"(a + 7u), "r"(b + i), "r"(b), "r"(a));
      }
    }
  }
  int s = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
  if (s == 0x7FFFFFFF) *sink = s;
}

__global__ void __launch_bounds__(BLOCK_THREADS, 1) barrier_bench_kernel(unsigned int* bar, uint32_t iters,
                                                                         unsigned long long* nsOut) {
  unsigned int epoch = 0;
  grid_barrier(bar, epoch);
  const unsigned long long t0 = globaltimer();
  for (uint32_t i = 0; i < iters; ++i) grid_barrier(bar, epoch);
  const unsigned long long t1 = globaltimer();
  if (blockIdx.x == 0 && threadIdx.x == 0) *nsOut = t1 - t0;
}

// L2 bandwidth: `iters` passes of a 16-byte-per-thread copy over buffers small enough to stay L2-resident (read + write
// bytes are counted); the launch configuration of the persistent kernels (one 1024-thread CTA per SM).
__global__ void __launch_bounds__(BLOCK_THREADS, 1) l2_copy_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst,
                                                                   uint64_t n16, uint32_t iters) {
  const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (uint64_t)gridDim.x * blockDim.x;
  for (uint32_t it = 0; it < iters; ++it) {
    uint64_t i = tid;
    for (; i + 3 * nth < n16; i += 4 * nth) {  // four independent 16-byte loads in flight per thread
      const uint4 a = __ldcg(src + i), b = __ldcg(src + i + nth), c = __ldcg(src + i + 2 * nth), d = __ldcg(src + i + 3 * nth);
      dst[i] = a; dst[i + nth] = b; dst[i + 2 * nth] = c; dst[i + 3 * nth] = d;
    }
    for (; i < n16; i += nth) dst[i] = __ldcg(src + i);
  }
}

// ---- tcgen05.mma kind::i8 (5th-generation tensor cores, accumulator in TMEM): peak of the form north_star (b) names
// as the alternative to mma.sync b1.  One CTA per SM; thread 0 issues `iters` MMAs of shape M = 128, N = n, K = 32
// (int8 x int8 -> int32) on shared-memory operands that are all ones, commits them to an mbarrier, and the four warps
// read the accumulator back with tcgen05.ld: every element must equal 32 * iters (independent of the operand layout,
// so the check pins the instruction, the descriptors' reach and the TMEM read-back, not a particular swizzle).
constexpr uint32_t TC_SMEM_BYTES = 48u << 10;  // operands + slack: any address the descriptors can generate holds ones

__device__ __forceinline__ uint64_t umma_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  // SM100 shared-memory matrix descriptor: start address >> 4 [0,14) | leading-dimension byte offset >> 4 [16,30) |
  // stride-dimension byte offset >> 4 [32,46) | descriptor version 1 [46,48) | swizzle mode 0 = none [61,64)
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}

__global__ void __launch_bounds__(128, 1) tcgen05_i8_peak_kernel(uint32_t iters, uint32_t n, unsigned int* bad) {
  extern __shared__ __align__(1024) unsigned char tc_smem[];
  __shared__ uint32_t tmemBase;
  __shared__ __align__(8) uint64_t mbar;
  for (uint32_t i = threadIdx.x; i < TC_SMEM_BYTES / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(tc_smem)[i] = 0x01010101u;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy stores -> visible to the tensor core's reads
  const uint32_t warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmemBase)), "r"(256u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x == 0) {
    mbar_init(&mbar, 1u);
    mbar_init_fence();
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t taddr = tmemBase;
  if (threadIdx.x == 0) {
    // K-major, no swizzle: 8 x 16-byte core matrices, 128 B apart along K, 256 B apart along M / N
    const uint64_t descA = umma_smem_desc(smem_u32(tc_smem), 128u, 256u);
    const uint64_t descB = umma_smem_desc(smem_u32(tc_smem) + 8192u, 128u, 256u);
    // instruction descriptor: D = S32 (2 << 4), A = B = signed int8 (1 << 7, 1 << 10), both K-major, N >> 3 at [17,23), M >> 4 at [24,29)
    const uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((128u >> 4) << 24);
    for (uint32_t it = 0; it < iters; ++it) {
      const uint32_t acc = it ? 1u : 0u;
      asm volatile(
          "{\n"
          ".reg .pred p;\n"
          "setp.ne.b32 p, %4, 0;\n"
          "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n"
          "}\n" ::"r"(taddr),
          "l"(descA), "l"(descB), "r"(idesc), "r"(acc)
          : "memory");
    }
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&mbar)) : "memory");
  }
  mbar_wait(&mbar, 0u);
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  // read-back: warp w owns TMEM lanes 32w .. 32w+31 (= rows of D), 8 columns per load
  unsigned int wrong = 0;
  for (uint32_t c0 = 0; c0 < n; c0 += 8) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr + ((32u * warp) << 16) + c0)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int j = 0; j < 8; ++j) wrong += r[j] != 32u * iters;
  }
  if (wrong) atomicAdd(bad, wrong);
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(256u) : "memory");
}

}  // namespace

cudaError_t run_tcgen05_peak(uint32_t iters, uint32_t n, int blocks, unsigned int* dBad, double* macsPerLaunch) {
  static bool attr = false;
  if (!attr) {
    cudaError_t e = cudaFuncSetAttribute((const void*)tcgen05_i8_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    attr = true;
  }
  tcgen05_i8_peak_kernel<<<blocks, 128, TC_SMEM_BYTES>>>(iters, n, dBad);
  *macsPerLaunch = (double)blocks * iters * 128.0 * n * 32.0;
  return cudaGetLastError();
}

cudaError_t run_l2_copy(const uint4* src, uint4* dst, uint64_t n16, uint32_t iters, int blocks) {
  l2_copy_kernel<<<blocks, BLOCK_THREADS>>>(src, dst, n16, iters);
  return cudaGetLastError();
}

cudaError_t run_contraction_selftest(int contraction, unsigned long long* dMismatch) {
  switch (contraction) {
    case 1: contraction_selftest_kernel<1><<<64, 128>>>(dMismatch); break;
    case 2: contraction_selftest_kernel<2><<<64, 128>>>(dMismatch); break;
    case 3: contraction_selftest_kernel<3><<<64, 128>>>(dMismatch); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_mma_peak(int kind, uint32_t iters, int blocks, int* dSink, double* macsPerLaunch) {
  constexpr int ILP = 8;
  if (kind == 2) {
    mma_peak_kernel<2, ILP><<<blocks, 1024>>>(iters, dSink);
    *macsPerLaunch = (double)blocks * 32.0 * iters * ILP * (8.0 * 8.0 * 128.0);
  } else if (kind == 3) {
    mma_peak_kernel<3, ILP><<<blocks, 1024>>>(iters, dSink);
    *macsPerLaunch = (double)blocks * 32.0 * iters * ILP * (16.0 * 8.0 * 32.0);
  } else {
    return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

// Thread-block cluster primitives (the sm_90+/sm_100 feature a small-frontier mode would use): `iters` back-to-back
// cluster barriers (barrier.cluster.arrive.release + wait.acquire: every thread of every CTA of the cluster) and a chain
// of `iters` dependent loads from the shared memory of the OTHER CTAs (mapa + ld.shared::cluster), one cluster of 1 024-thread
// CTAs.  out[0] = ns of the barriers, out[1] = ns of the loads, out[2] = the chain's last value (keeps the loads alive).
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__global__ void __launch_bounds__(BLOCK_THREADS, 1) cluster_bench_kernel(uint32_t iters, unsigned long long* out) {
  __shared__ uint32_t slot[32];
  uint32_t rank, nctas;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(nctas));
  if (threadIdx.x < 32) slot[threadIdx.x] = (threadIdx.x * 7u + 1u) & 31u;  // a permutation of 0..31: the chain's next index
  cluster_sync_all();
  const unsigned long long t0 = globaltimer();
  for (uint32_t i = 0; i < iters; ++i) cluster_sync_all();
  const unsigned long long t1 = globaltimer();
  if (rank == 0 && threadIdx.x == 0) {
    uint32_t idx = 0, cta = 1u % nctas;
    const unsigned long long t2 = globaltimer();
    for (uint32_t i = 0; i < iters; ++i) {
      uint32_t remote;
      asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(&slot[idx])), "r"(cta));
      asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(idx) : "r"(remote) : "memory");
      cta = cta + 1u == nctas ? (nctas > 1u ? 1u : 0u) : cta + 1u;
    }
    const unsigned long long t3 = globaltimer();
    out[0] = t1 - t0;
    out[1] = t3 - t2;
    out[2] = idx;
  }
  cluster_sync_all();  // no CTA leaves while its shared memory may still be read
}

cudaError_t run_cluster_bench(int clusterCtas, uint32_t iters, unsigned long long* dOut) {
  cudaError_t e = cudaSuccess;
  if (clusterCtas > 8) {
    e = cudaFuncSetAttribute(cluster_bench_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)clusterCtas);
  cfg.blockDim = dim3(BLOCK_THREADS);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)clusterCtas;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, cluster_bench_kernel, iters, dOut);
}

cudaError_t run_barrier_bench(unsigned int* dBar, uint32_t iters, int blocks, unsigned long long* dNs) {
  void* args[] = {(void*)&dBar, (void*)&iters, (void*)&dNs};
  return cudaLaunchCooperativeKernel((const void*)barrier_bench_kernel, dim3(blocks), dim3(BLOCK_THREADS), args, 0, 0);
}

}  // namespace blest
