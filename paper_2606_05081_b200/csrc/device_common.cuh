// device_common.cuh -- shared device-side pieces of the BLEST kernels: control block, grid barrier, work-queue
// entry encoding, warp-aggregated queue expansion, slice x frontier-word contraction forms.
#pragma once
#include <cassert>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/blest.h"

// Debug build (python -m paper_2606_05081_b200.build --debug -> libblest_debug.so, -DBLEST_DEBUG): every queue / list /
// chunk / bitmap / graph-array index of the kernels is bounds-checked with a device assert (compute-sanitizer is closed on
// this GPU pool; tests/test_gpu_parity.py runs the small-graph suite against this build).
#ifdef BLEST_DEBUG
#define BLEST_ASSERT(cond) assert(cond)
#else
#define BLEST_ASSERT(cond) ((void)0)
#endif

namespace blest {

constexpr int BLOCK_THREADS = 1024;
constexpr int WARPS_PER_BLOCK = BLOCK_THREADS / 32;
constexpr uint32_t TD_CHUNK = 128;     // edges per edge-chunk queue entry (4 per lane)
constexpr uint32_t VSS_QUADS = 32;     // quads per slice-chunk queue entry = one VSS (tau = 128 slices)
constexpr uint32_t BIG_SEG = 32;       // segments expanding to more entries than this are written warp-cooperatively
constexpr uint32_t BIG_CAP = 16;       // per-warp capacity of the cooperative-expansion list

// Control block in global memory, zeroed by the host before every launch.
struct Ctrl {
  unsigned int bar;    // monotone grid-barrier arrival counter
  unsigned int tail;   // eager kernel: monotone work-queue tail; shares an aligned 8-byte word with `bar`, so the
                       // barrier's spin load returns both (one round trip less per level)
  unsigned int error;  // bit 0: work-queue overflow
  unsigned int nlevels;
  unsigned int qc[4];               // work-queue entry counters (rotating)
  unsigned long long qbytes[4];     // graph bytes covered by the work of each level (rotating)
  unsigned long long unvisited[4];  // per level (rotating)
  unsigned long long newcount[4];
  unsigned long long mf[4];         // sum of degrees of the vertices discovered at this level
  unsigned long long buScanned[4];  // neighbours scanned by the bottom-up stage
  unsigned long long t0;            // %globaltimer at kernel start
  unsigned long long tInit;         // lazy kernel: ns from kernel start to the end of the per-call init
  unsigned int wlc[4];              // lazy kernel: frontier word-list lengths (rotating, level mod 3)
  unsigned int nBig[4];             // lazy kernel: deferred big segments of the level (rotating)
  unsigned int epochBase;           // lazy kernel: grid barriers executed by earlier launches on this control block.  That
                                    // kernel's block is zeroed once at build; every launch resets the per-call fields
                                    // itself and leaves `bar` = epochBase * gridDim (mod 2^32), so no memset precedes a call
  unsigned int guess[32 * 32];      // lazy kernel: the level that discovered the most vertices in the last call on this handle
                                    // from a source of the same class (0 = none yet): the next such call pre-fills levels_out
                                    // with it (bfs_lazy.cu "level guess").  Class = (floor(log2(degree + 1)),
                                    // floor(log2(internal id of the first neighbour + 1))): how far the source is from the hubs
};

// Work-queue overflow: flagged in the control block of the call (blest_get_trace) and latched in the handle's
// host-mapped status word (blest_last_status; include/blest.h "Asynchrony").
__device__ __forceinline__ void report_overflow(Ctrl* ctrl, unsigned int* hostStatus) {
  atomicOr(&ctrl->error, 1u);
  if (hostStatus) *(volatile unsigned int*)hostStatus = 1u;
}

// ---- TMA bulk copy (cp.async.bulk, 1-D) + mbarrier: global -> shared staging without registers or LSU slots ----------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// One thread: announce `bytes` of asynchronous traffic on the barrier's current phase and count as its one arrival.
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Bulk copy of `bytes` (multiple of 16; both addresses 16-byte aligned) that completes on `bar`.
__device__ __forceinline__ void bulk_g2s(void* dstSmem, const void* srcGlobal, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dstSmem)),
               "l"(srcGlobal), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

__device__ __forceinline__ unsigned long long globaltimer() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// Grid-wide barrier for a co-resident (cooperative) launch: one release-RMW per block on a monotone counter,
// thread 0 spins with acquire loads (PAPER.md:464 GRIDSYNC; hand-rolled so a level costs one L2 round trip).
__device__ __forceinline__ void grid_barrier(unsigned int* bar, unsigned int& epoch) {
  __syncthreads();
  ++epoch;
  if (threadIdx.x == 0) {
    const unsigned int target = epoch * gridDim.x;
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
    unsigned int v;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
    } while ((int)(v - target) < 0);  // wrap-safe: the counter is monotone over billions of barriers (closeness runs)
  }
  __syncthreads();
}

// The same barrier with the epoch kept in a shared-memory word that only thread 0 touches (no register of the other
// threads): the lazy kernel sits at its register limit.
__device__ __forceinline__ void grid_barrier_sh(unsigned int* bar, unsigned int* epochSlot) {
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned int epoch = *epochSlot + 1u;
    *epochSlot = epoch;
    const unsigned int target = epoch * gridDim.x;
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
    unsigned int v;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
    } while ((int)(v - target) < 0);
  }
  __syncthreads();
}

// Same barrier on the {bar, tail} word: returns the queue tail as it stands once every CTA has arrived (each CTA's
// appends precede its arrival, so the value is final).  `slot` is a shared-memory word for the broadcast.
__device__ __forceinline__ unsigned int grid_barrier_tail(unsigned int* bar, unsigned int& epoch, unsigned int* slot) {
  __syncthreads();
  ++epoch;
  if (threadIdx.x == 0) {
    const unsigned int target = epoch * gridDim.x;
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
    unsigned long long v;
    do {
      asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(bar) : "memory");
    } while ((int)((unsigned int)v - target) < 0);  // wrap-safe, as above
    *slot = (unsigned int)(v >> 32);
  }
  __syncthreads();
  return *slot;
}

__device__ __forceinline__ unsigned int ld_volatile(const unsigned int* p) { return *(const volatile unsigned int*)p; }
__device__ __forceinline__ unsigned long long ld_volatile(const unsigned long long* p) {
  return *(const volatile unsigned long long*)p;
}

// 16-byte grid-stride fill (count32 = number of 32-bit words; ptr 16-byte aligned, count32 padded to 4 by the host).
__device__ __forceinline__ void grid_fill32(uint32_t* ptr, uint32_t value, uint64_t count32) {
  uint4* p4 = reinterpret_cast<uint4*>(ptr);
  const uint64_t n4 = count32 >> 2;
  const uint4 v = make_uint4(value, value, value, value);
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (uint64_t)gridDim.x * blockDim.x) p4[i] = v;
  for (uint64_t i = (n4 << 2) + (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count32; i += (uint64_t)gridDim.x * blockDim.x)
    ptr[i] = value;
}

// ---- work-queue entries ----------------------------------------------------------------------------
// x = first quad (slice chunk) or first edge (edge chunk); y = type bit 31 | payload.
__device__ __forceinline__ uint2 make_slice_entry(uint32_t quad, uint32_t nq, uint32_t s) {
  return make_uint2(quad, (s << 5) | (nq - 1));
}
__device__ __forceinline__ uint2 make_edge_entry(uint32_t edge, uint32_t cnt) { return make_uint2(edge, 0x80000000u | cnt); }

struct BigSeg { uint32_t type_s, start, count, pos; };

// Expansion of one segment (a slice set's quads or a vertex's edges) into queue entries at Q[pos..].
__device__ __forceinline__ uint32_t seg_entries(uint32_t type, uint32_t count) {
  return type ? (count + TD_CHUNK - 1) / TD_CHUNK : (count + VSS_QUADS - 1) / VSS_QUADS;
}
__device__ __forceinline__ void write_entry(uint2* Q, uint32_t pos, uint32_t type, uint32_t start, uint32_t count,
                                            uint32_t s, uint32_t i) {
  BLEST_ASSERT(i < seg_entries(type, count));
  if (type) Q[pos + i] = make_edge_entry(start + i * TD_CHUNK, min(TD_CHUNK, count - i * TD_CHUNK));
  else Q[pos + i] = make_slice_entry(start + i * VSS_QUADS, min(VSS_QUADS, count - i * VSS_QUADS), s);
}
__device__ __forceinline__ void emit_segment(uint2* Q, uint32_t& pos, uint32_t type, uint32_t start, uint32_t count,
                                             uint32_t s, BigSeg* bigList, uint32_t* bigCnt) {
  const uint32_t nent = seg_entries(type, count);
  bool deferred = false;
  if (nent > BIG_SEG) {
    uint32_t k = atomicAdd(bigCnt, 1u);
    if (k < BIG_CAP) { bigList[k] = BigSeg{(s << 1) | type, start, count, pos}; deferred = true; }
  }
  if (!deferred)
    for (uint32_t i = 0; i < nent; ++i) write_entry(Q, pos, type, start, count, s, i);
  pos += nent;
}
// Called by the whole warp after all lanes emitted: long segments are written 32 entries at a time.
__device__ __forceinline__ void flush_big_segments(uint2* Q, BigSeg* bigList, uint32_t* bigCnt, uint32_t lane) {
  __syncwarp();
  const uint32_t nb = min(*bigCnt, BIG_CAP);
  for (uint32_t k = 0; k < nb; ++k) {
    const BigSeg g = bigList[k];
    const uint32_t type = g.type_s & 1, s = g.type_s >> 1, nent = seg_entries(type, g.count);
    for (uint32_t i = lane; i < nent; i += 32) write_entry(Q, g.pos, type, g.start, g.count, s, i);
  }
  __syncwarp();
  if (lane == 0) *bigCnt = 0;
  __syncwarp();
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= (uint32_t)d) v += t;
  }
  return v;
}

// Reserve `cnt` entries per lane with one atomic per warp.  Returns this lane's first position; ok = fits.
__device__ __forceinline__ uint32_t warp_reserve(unsigned int* counter, uint32_t cnt, uint32_t lane, uint32_t cap,
                                                 unsigned int* errorFlag, bool& ok) {
  const uint32_t incl = warp_incl_scan(cnt, lane);
  const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
  uint32_t base = 0;
  if (total) {
    if (lane == 31) base = atomicAdd(counter, total);
    base = __shfl_sync(0xffffffffu, base, 31);
  }
  ok = (uint64_t)base + total <= cap;
  if (!ok && lane == 0) atomicOr(errorFlag, 1u);
  return base + incl - cnt;
}

// ---- the slice x frontier-word contraction (Eq. 2, §5.1) -----------------------------------
// m = four 8-bit masks (slice c in bits 8c..8c+7), alpha = 8-bit frontier word of the slice set (warp-uniform).
// Returns a 4-bit hit mask: bit c set iff (mask_c AND alpha) != 0, i.e. popc(mask_c AND alpha) > 0.
__device__ __forceinline__ uint32_t contract_alu(uint32_t m, uint32_t alpha) {
  const uint32_t x = m & (alpha * 0x01010101u);
  const uint32_t nz = (((x & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | x) & 0x80808080u;  // bit 8c+7 set iff byte c != 0
  return ((nz >> 7) & 1u) | ((nz >> 14) & 2u) | ((nz >> 21) & 4u) | ((nz >> 28) & 8u);
}

// The paper's layout (PAPER.md:203 Fig. 3, :213-217): two m8n8k128 b1 and.popc MMAs per 128 slices; fragA = two
// packed masks in the low 16 bits; fragB non-zero only in lanes t mod 9 == 0 (alpha) and t mod 9 == 4 (alpha << 8);
// every fragC popcount belongs to the issuing lane.  All 32 lanes must call (m = 0 for idle lanes).
// NOTE: sm_100a has no BMMA unit; ptxas lowers this instruction to an int8 IMMA sequence.
__device__ __forceinline__ uint32_t contract_b1(uint32_t m, uint32_t alpha, uint32_t lane) {
  const uint32_t r9 = lane % 9u;
  const uint32_t fragB = (r9 == 0u) ? alpha : ((r9 == 4u) ? (alpha << 8) : 0u);
  int c0 = 0, c1 = 0, c2 = 0, c3 = 0;
  const uint32_t a_lo = m & 0xFFFFu, a_hi = m >> 16;
  asm volatile("mma.sync.aligned.m8n8k128.row.col.s32.b1.b1.s32.and.popc {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+r"(c0), "+r"(c1) : "r"(a_lo), "r"(fragB));
  asm volatile("mma.sync.aligned.m8n8k128.row.col.s32.b1.b1.s32.and.popc {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+r"(c2), "+r"(c3) : "r"(a_hi), "r"(fragB));
  return (c0 != 0 ? 1u : 0u) | (c1 != 0 ? 2u : 0u) | (c2 != 0 ? 4u : 0u) | (c3 != 0 ? 8u : 0u);
}

// int8 tensor-core form: native IMMA m16n8k32 u8 with the mask bits expanded to bytes (2 IMMAs per 128 slices).
// MMA row r = the mask word of one lane (4 slices = 4 K-groups of 8 bits): A[r][8i+j] = bit j of slice i;
// B[8i+j][col] = (col == i) ? bit j of alpha : 0, so D[r][i] = popc(mask_i AND alpha).  MMA #1 takes the words of
// lanes 0..15, MMA #2 of lanes 16..31.  Fragment layout (PTX ISA, m16n8k32 .u8): g = lane>>2, t = lane&3;
// a0: row g, k 4t..4t+3 | a1: row g+8 | a2: row g, k 16+4t.. | a3: row g+8, k 16+4t..; b0: k 4t.., col g | b1: k 16+4t..;
// c0/c1: row g, cols 2t, 2t+1 | c2/c3: row g+8.  All 32 lanes must call.
__device__ __forceinline__ uint32_t nibble_to_bytes(uint32_t word, uint32_t byteIdx, uint32_t hiNibble) {
  const uint32_t nib = (word >> (8u * byteIdx + 4u * hiNibble)) & 0xFu;
  return (nib * 0x00204081u) & 0x01010101u;  // bit k of the nibble -> byte k (0 or 1)
}
__device__ __forceinline__ uint32_t contract_u8(uint32_t m, uint32_t alpha, uint32_t lane) {
  const uint32_t g = lane >> 2, t = lane & 3u, sl = t >> 1, hi = t & 1u;
  const uint32_t ab = nibble_to_bytes(alpha, 0, hi);
  const uint32_t b0 = (g == sl) ? ab : 0u, b1 = (g == 2u + sl) ? ab : 0u;
  uint32_t flags = 0;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const uint32_t w0 = __shfl_sync(0xffffffffu, m, 16 * k + g), w1 = __shfl_sync(0xffffffffu, m, 16 * k + 8 + g);
    const uint32_t a0 = nibble_to_bytes(w0, sl, hi), a1 = nibble_to_bytes(w1, sl, hi);
    const uint32_t a2 = nibble_to_bytes(w0, 2u + sl, hi), a3 = nibble_to_bytes(w1, 2u + sl, hi);
    int c0 = 0, c1 = 0, c2 = 0, c3 = 0;
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.u8.u8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(c0), "+r"(c1), "+r"(c2), "+r"(c3) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
    flags |= ((c0 != 0 ? 1u : 0u) | (c1 != 0 ? 2u : 0u) | (c2 != 0 ? 4u : 0u) | (c3 != 0 ? 8u : 0u)) << (4 * k);
  }
  // row r of MMA k belongs to lane 16k + r; its columns 0,1 sit in lane 4(r&7) (c0,c1 or c2,c3), columns 2,3 in lane 4(r&7)+1
  const uint32_t r = lane & 15u, shift = 4u * (lane >> 4) + 2u * (r >> 3);
  const uint32_t fa = __shfl_sync(0xffffffffu, flags, 4u * (r & 7u)), fb = __shfl_sync(0xffffffffu, flags, 4u * (r & 7u) + 1u);
  return ((fa >> shift) & 3u) | (((fb >> shift) & 3u) << 2);
}

template <int CONTR>
__device__ __forceinline__ uint32_t contract(uint32_t m, uint32_t alpha, uint32_t lane) {
  if (CONTR == 2) return contract_b1(m, alpha, lane);
  if (CONTR == 3) return contract_u8(m, alpha, lane);
  return contract_alu(m, alpha);
}

}  // namespace blest
