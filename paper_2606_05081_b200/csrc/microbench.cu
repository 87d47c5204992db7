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

}  // namespace

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

cudaError_t run_barrier_bench(unsigned int* dBar, uint32_t iters, int blocks, unsigned long long* dNs) {
  void* args[] = {(void*)&dBar, (void*)&iters, (void*)&dNs};
  return cudaLaunchCooperativeKernel((const void*)barrier_bench_kernel, dim3(blocks), dim3(BLOCK_THREADS), args, 0, 0);
}

}  // namespace blest
