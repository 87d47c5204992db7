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


constexpr uint32_t PULL_SMALL = 8;      // pull level: rows of up to this many neighbours are scanned by their own lane,
constexpr uint32_t PULL_LONG = 1024;    // longer ones by their warp, rows beyond this by the whole CTA
constexpr uint32_t PULL_LONG_CAP = 64;  // (per CTA and level; further ones stay with their warp)

struct MsShared {
  BigSeg bigList[WARPS_PER_BLOCK][BIG_CAP];
  uint32_t bigCnt[WARPS_PER_BLOCK];
  unsigned long long acc;
  unsigned int tailSlot;  // broadcast slot of grid_barrier_tail
  uint32_t perSource[256];
  alignas(16) uint32_t fset[WARPS_PER_BLOCK][8 * 8];  // per warp: the kappa-bit frontier words of the current set's 8 columns
  alignas(16) uint32_t tab[WARPS_PER_BLOCK][32 * 8];  // per warp: ORs of the subsets of columns 0..3 / 4..7 (ms_stage1)
  unsigned long long tPh[5], tMark;  // phase times of CTA 0 (blest_get_ms_phases)
  uint32_t liveAcc[8];               // OR of the frontier words this CTA produced in the current level (pull levels)
  unsigned int updAcc;               // rows this CTA updated in the current pull level
  unsigned int longCnt;              // pull level: rows of more than PULL_LONG neighbours met by this CTA ...
  uint4 longRow[PULL_LONG_CAP];      // ... {row, first, end of its neighbour list, 0}: scanned by the whole CTA
  uint32_t longAcc[PULL_LONG_CAP][8];  // ... and the OR of the frontier words its warps found
  unsigned long long cnt[WARPS_PER_BLOCK][7];  // per warp (lane 0): queue entries, quads, slices probed, fresh row
                                               // updates, dirty slice sets swept, pull: rows scanned, neighbours read
                                               // -- totals for the roofline (p.stats)
};

// One kappa-bit word (KW 32-bit words, naturally aligned) moved with a single vector access.
// MsShared is larger than the 48 KB a kernel may declare statically: it lives in dynamic shared memory.
extern __shared__ __align__(16) unsigned char msDyn[];

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

// Stage 1 in its first form: one entry at a time, the contraction as a loop over the mask bits.  Kept for kappa = 256,
// where the pipelined table form below is 8 % slower (32-byte table entries, one slice's probe in flight at a time).
template <int KW>
__device__ __forceinline__ void ms_stage1_loop(const MsParams& p, MsShared& sh, const uint2* Qc, uint32_t qcount) {
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

// Shared-memory table entry e (a kappa-bit word) of a warp's fset / tab.
template <int KW>
__device__ __forceinline__ void tab_load(const uint32_t* tab, uint32_t e, uint32_t (&w)[KW]) {
  if (KW == 1) w[0] = tab[e];
  else if (KW == 2) {
    const uint2 v = reinterpret_cast<const uint2*>(tab)[e];
    w[0] = v.x; w[KW > 1 ? 1 : 0] = v.y;
  } else {
#pragma unroll
    for (int q = 0; q < KW / 4; ++q) {
      const uint4 v = reinterpret_cast<const uint4*>(tab)[e * (KW / 4) + q];
      w[KW > 3 ? 4 * q : 0] = v.x; w[KW > 3 ? 4 * q + 1 : 0] = v.y; w[KW > 3 ? 4 * q + 2 : 0] = v.z; w[KW > 3 ? 4 * q + 3 : 0] = v.w;
    }
  }
}
template <int KW>
__device__ __forceinline__ void tab_store(uint32_t* tab, uint32_t e, const uint32_t (&w)[KW]) {
  if (KW == 1) tab[e] = w[0];
  else if (KW == 2) reinterpret_cast<uint2*>(tab)[e] = make_uint2(w[0], w[KW > 1 ? 1 : 0]);
  else {
#pragma unroll
    for (int q = 0; q < KW / 4; ++q)
      reinterpret_cast<uint4*>(tab)[e * (KW / 4) + q] =
          make_uint4(w[KW > 3 ? 4 * q : 0], w[KW > 3 ? 4 * q + 1 : 0], w[KW > 3 ? 4 * q + 2 : 0], w[KW > 3 ? 4 * q + 3 : 0]);
  }
}

// The operands of one work-queue entry (a VSS: up to 32 quads of one slice set).
template <int KW>
struct MsEntry {
  uint4 rows;
  uint32_t m;
  uint32_t fv[KW];  // lanes 0..7: the kappa-bit frontier word of column `lane` of the set
};
template <int KW>
__device__ __forceinline__ void ms_fetch(const MsParams& p, const uint2 e, bool valid, uint32_t lane, MsEntry<KW>& d) {
  const uint32_t nq = valid ? (e.y & 31u) + 1u : 0u, s = e.y >> 5;
  BLEST_ASSERT(!valid || (s < p.Ns && (uint64_t)e.x + nq <= p.nQuads));
  d.rows = make_uint4(0, 0, 0, 0);
  d.m = 0;
  if (lane < nq) {
    d.rows = __ldg(p.rowIds + e.x + lane);
    d.m = __ldg(p.masks + e.x + lane);
  }
#pragma unroll
  for (int w = 0; w < KW; ++w) d.fv[w] = 0;
  if (valid && lane < 8) load_words<KW>(p.F, (uint64_t)lane * p.rho + s, d.fv);
}

// Stage 1.  One work-queue entry per warp step, lane = quad.  ncu (round 2, profiles/r02e_c5.md): the
// stage is bound by the length of each warp's own instruction stream (about 220 dependent warp instructions per VSS, a
// third of them the divergent loop over the mask bits, plus three exposed round trips: queue word -> row ids / masks /
// frontier words -> probes), not by L1, L2 or issue slots.  Hence
//  * the loop is software-pipelined: while the probes of entry i are in flight the warp holds the queue word of entry
//    i + 2 and the operands of entry i + 1;
//  * the contraction M = OR_{j in mask} F_curr^kappa[column j] is a table look-up: per VSS the warp builds, from the set's
//    eight frontier words, the OR of every subset of columns 0..3 (entries 0..15, lane = entry) and of columns 4..7
//    (entries 16..31); a slice needs tab[mask & 15] | tab[16 + (mask >> 4)], two shared-memory reads, no loop;
//  * the V_next probes of a lane's slices are issued together, before the first RED.
template <int KW>
__device__ __forceinline__ void ms_stage1(const MsParams& p, MsShared& sh, const uint2* Qc, uint32_t qcount) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  if (gwarp >= qcount) return;
  uint32_t* fset = sh.fset[warp];
  uint32_t* tab = sh.tab[warp];
  constexpr int G = KW <= 2 ? 4 : (KW == 4 ? 2 : 1);  // slices of a lane whose probes are in flight together
  constexpr uint32_t WB = 4u * KW;                    // bytes per kappa-bit word
  const uint32_t rho = p.rho;
  unsigned char* const vnBase = reinterpret_cast<unsigned char*>(p.Vn);
  MsEntry<KW> cur, nxt;
  uint2 eN = make_uint2(0, 0);  // queue word of the entry after the current one
  BLEST_ASSERT(gwarp < p.qcap);
  ms_fetch<KW>(p, Qc[gwarp], true, lane, cur);
  if (gwarp + nwarps < qcount) eN = Qc[gwarp + nwarps];
  uint32_t nProbe = 0, nFresh = 0, nEnt = 0, nQuad = 0;
  const uint32_t tsel = lane & 15u, tbase = (lane >> 4) * 4u;  // this lane's table entry: subset tsel of columns tbase..+3
  for (uint32_t i = gwarp; i < qcount; i += nwarps) {
    // the frontier words of the current set -> shared memory -> subset table
    __syncwarp();
    if (lane < 8) tab_store<KW>(fset, lane, cur.fv);
    __syncwarp();
    {
      uint32_t t[KW];
#pragma unroll
      for (int w = 0; w < KW; ++w) t[w] = 0;
#pragma unroll
      for (uint32_t b = 0; b < 4; ++b) {
        uint32_t f[KW];
        tab_load<KW>(fset, tbase + b, f);
        const uint32_t on = 0u - ((tsel >> b) & 1u);
#pragma unroll
        for (int w = 0; w < KW; ++w) t[w] |= f[w] & on;
      }
      tab_store<KW>(tab, lane, t);
    }
    __syncwarp();
    // next entry's operands and the queue word after it
    ms_fetch<KW>(p, eN, i + nwarps < qcount, lane, nxt);  // (no overflow: qcount <= qcap < 2^31)
    if ((uint64_t)i + 2ull * nwarps < qcount) eN = Qc[i + 2u * nwarps];
    const uint32_t ru[4] = {cur.rows.x, cur.rows.y, cur.rows.z, cur.rows.w};
#pragma unroll
    for (int c0 = 0; c0 < 4; c0 += G) {
      uint32_t M[G][KW], vn[G][KW];  // per-row kappa-bit accumulation buffer ("M[0..3]")
      unsigned char* addr[G];
      uint32_t live = 0;
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const uint32_t mb = (cur.m >> (8 * (c0 + g))) & 0xFFu;
        uint32_t hi[KW];
        tab_load<KW>(tab, mb & 15u, M[g]);
        tab_load<KW>(tab, 16u + (mb >> 4), hi);
        uint32_t any = 0;
#pragma unroll
        for (int w = 0; w < KW; ++w) { M[g][w] |= hi[w]; any |= M[g][w]; }
        const uint32_t u = ru[c0 + g];
        BLEST_ASSERT(!any || u < p.n);
        addr[g] = vnBase + (size_t)((u & 7u) * rho + (u >> 3)) * WB;  // getVI(u, rho): below 2^32 words (n <= 2^29)
        if (any) live |= 1u << g;
      }
      // one probe and one RED per row, each a single kappa-bit access; the probes of the group first
#pragma unroll
      for (int g = 0; g < G; ++g) {
#pragma unroll
        for (int w = 0; w < KW; ++w) vn[g][w] = 0xFFFFFFFFu;
        if ((live >> g) & 1u) load_words<KW>(reinterpret_cast<const uint32_t*>(addr[g]), 0, vn[g]);
      }
      nProbe += (uint32_t)__popc(live);
#pragma unroll
      for (int g = 0; g < G; ++g) {
        uint32_t fresh[KW], any = 0;
#pragma unroll
        for (int w = 0; w < KW; ++w) { fresh[w] = M[g][w] & ~vn[g][w]; any |= fresh[w]; }
        if (any) {
          red_or_words<KW>(reinterpret_cast<uint32_t*>(addr[g]), 0, fresh);
          p.dirty[ru[c0 + g] >> 3] = 1;  // PAPER.md:583 dirtySets
          ++nFresh;
        }
      }
    }
    ++nEnt;
    nQuad += (uint32_t)__popc(__ballot_sync(0xffffffffu, cur.m != 0u || cur.rows.x != 0u || cur.rows.y != 0u));
    cur = nxt;
  }
  if (p.stats) {  // totals for the roofline: one reduction per warp and stage
    const uint32_t tp = __reduce_add_sync(0xffffffffu, nProbe), tf = __reduce_add_sync(0xffffffffu, nFresh);
    if (lane == 0) {
      unsigned long long* cnt = sh.cnt[warp];
      cnt[0] += nEnt; cnt[1] += nQuad; cnt[2] += tp; cnt[3] += tf;
    }
  }
}

// The sources that still have a frontier.  live[l mod 3] = OR of the frontier words of the vertices at distance l - 1
// (what level l expands); level l - 1 accumulates it, level l reads it and clears the slot level l + 1 accumulates.
template <int KW>
__device__ __forceinline__ void publish_live(const MsParams& p, MsShared& sh, const uint32_t (&lv)[KW], uint32_t forLevel) {
#pragma unroll
  for (int w = 0; w < KW; ++w) {
    const uint32_t r = __reduce_or_sync(0xffffffffu, lv[w]);
    if ((threadIdx.x & 31) == 0 && r) atomicOr(&sh.liveAcc[w], r);
  }
  __syncthreads();
  if (threadIdx.x < KW) {
    const uint32_t r = sh.liveAcc[threadIdx.x];
    if (r) atomicOr(&p.live[(forLevel % 3u) * 8u + threadIdx.x], r);
    sh.liveAcc[threadIdx.x] = 0;
  }
}

// A PULL level (the multi-source counterpart of PAPER.md Alg. 4; north_star (e)): every row u that some live source has
// not reached ORs the frontier words of its neighbours, V[u] |= (OR_{v in N(u)} F[v]) & live & ~V[u], and stops as soon as
// every live source it lacks is covered.  The owner of the row finalises it on the spot (Stage 2 of Alg. 5 fused: frontier
// word, Eq. 7 accumulation), so the level needs no RED, no dirtySets, no work queue and one grid barrier.  Measured reason
// (profiles/r02e_c5.md): on config 5 the top-down levels that mark many rows are bound by the REDs (a sweep that marks
// nothing: 24 us; the same sweep at level 3, 1 M REDs: 61 us), and once most rows hold every live source a pull sweep
// skips them after one coalesced load.  Lane = row (4 consecutive slice sets per warp step: the words of a step are 8 x 32
// contiguous bytes); rows of up to PULL_SMALL neighbours are scanned by their own lane, longer ones by the whole warp, 64
// neighbours per round.  A batch switches once (kernel loop) and stays in pull mode: V_next is not maintained here.
// The groups are assigned statically in natural order.  Measured alternatives on config 5: claiming groups from one
// global counter, +20 % (13 K same-address atomics per level at about 2.5 ns each); a list ordered by degree sum with the
// heaviest groups paired with the lightest, +8 % (the heavy groups then run at the same time); the first pull level sits at
// the rate one SM's L1 forwards scattered sectors (7.6 M frontier words / 148 SMs x 2 cycles = 52 us of its 60 us).
template <int KW>
__device__ __forceinline__ void ms_pull_level(const MsParams& p, MsShared& sh, uint32_t level, const uint32_t* Fc, uint32_t* Fn) {
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gwarp = blockIdx.x * WARPS_PER_BLOCK + warp, nwarps = gridDim.x * WARPS_PER_BLOCK;
  const uint32_t rho = p.rho;
  uint32_t live[KW], lv[KW];
#pragma unroll
  for (int w = 0; w < KW; ++w) {
    live[w] = __ldcg(&p.live[(level % 3u) * 8u + w]);
    lv[w] = 0;
  }
  uint32_t nUpd = 0, nRows = 0, nNbr = 0;  // rows updated / scanned, neighbours read (per lane)
  const uint32_t nGroups = (p.Ns + 3u) / 4u;
  for (uint32_t g = gwarp; g < nGroups; g += nwarps) {
    const uint32_t s = 4u * g + (lane >> 3), j = lane & 7u, u = 8u * s + j;
    const bool valid = s < p.Ns && u < p.n;
    const uint64_t idx = (uint64_t)j * rho + s;  // getVI(u, rho)
    uint32_t vc[KW], need[KW], acc[KW], anyNeed = 0;
#pragma unroll
    for (int w = 0; w < KW; ++w) vc[w] = 0xFFFFFFFFu;
    if (valid) load_words<KW>(p.Vc, idx, vc);
#pragma unroll
    for (int w = 0; w < KW; ++w) { need[w] = live[w] & ~vc[w]; anyNeed |= need[w]; acc[w] = 0; }
    uint32_t r0 = 0, r1 = 0;
    if (anyNeed) { r0 = __ldg(&p.rowptr[u]); r1 = __ldg(&p.rowptr[u + 1]); }
    const uint32_t deg = r1 - r0;
    nRows += anyNeed ? 1u : 0u;
    if (deg != 0 && deg <= PULL_SMALL) {  // short row: own lane, up to four neighbours in flight
      for (uint32_t k = r0; k < r1; k += 4u) {
        nNbr += min(4u, r1 - k);
        uint32_t f[4][KW];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
#pragma unroll
          for (int w = 0; w < KW; ++w) f[q][w] = 0;
          if (k + q < r1) {
            const uint32_t v = __ldg(&p.colidx[k + q]);
            BLEST_ASSERT(v < p.n);
            load_words<KW>(Fc, (uint64_t)(v & 7u) * rho + (v >> 3), f[q]);
          }
        }
        uint32_t lack = 0;
#pragma unroll
        for (int w = 0; w < KW; ++w) {
          acc[w] |= f[0][w] | f[1][w] | f[2][w] | f[3][w];
          lack |= need[w] & ~acc[w];
        }
        if (!lack) break;
      }
    }
    // longer rows: the whole warp, one row at a time, 128 neighbours per round, until every source the row lacks is
    // covered.  (Concatenating the lists of the group's rows and walking them together, with shared-memory atomics per
    // neighbour, was measured 30-45 % slower on config 5: it gives up the early exit.)
    // (rows beyond PULL_LONG neighbours are left to the whole CTA, below: one warp would need deg / 128 rounds for them --
    // measured on config 5, first pull level: the slowest CTA took 110 us against a mean of 68)
    bool deferred = false;
    if (KW >= 4 && deg > PULL_LONG) {  // (kappa = 64: measured 3 % slower with the CTA phase, kappa = 128: 9 % faster)
      const uint32_t k = atomicAdd(&sh.longCnt, 1u);
      if (k < PULL_LONG_CAP) {
        sh.longRow[k] = make_uint4(u, r0, r1, 0u);
        deferred = true;
      }
    }
    uint32_t big = __ballot_sync(0xffffffffu, deg > PULL_SMALL && !deferred);
    while (big) {
      const int src = __ffs(big) - 1;
      big &= big - 1;
      const uint32_t b = __shfl_sync(0xffffffffu, r0, src), e = __shfl_sync(0xffffffffu, r1, src);
      uint32_t nd[KW], a[KW], red[KW];
#pragma unroll
      for (int w = 0; w < KW; ++w) { nd[w] = __shfl_sync(0xffffffffu, need[w], src); a[w] = 0; red[w] = 0; }
      // (all the loads of a round are issued before the first use: written out, the generic loop form serialised them
      // and cost 30 % of the level)
      for (uint32_t k = b; k < e; k += 128u) {
        if (lane == 0) nNbr += min(128u, e - k);
        uint32_t f0[KW], f1[KW], f2[KW], f3[KW];
#pragma unroll
        for (int w = 0; w < KW; ++w) f0[w] = f1[w] = f2[w] = f3[w] = 0;
        const uint32_t k0 = k + lane, k1 = k + 32u + lane, k2 = k + 64u + lane, k3 = k + 96u + lane;
        uint32_t v0 = 0, v1 = 0, v2 = 0, v3 = 0;
        if (k0 < e) v0 = __ldg(&p.colidx[k0]);
        if (k1 < e) v1 = __ldg(&p.colidx[k1]);
        if (k2 < e) v2 = __ldg(&p.colidx[k2]);
        if (k3 < e) v3 = __ldg(&p.colidx[k3]);
        BLEST_ASSERT(v0 < p.n && v1 < p.n && v2 < p.n && v3 < p.n);
        if (k0 < e) load_words<KW>(Fc, (uint64_t)(v0 & 7u) * rho + (v0 >> 3), f0);
        if (k1 < e) load_words<KW>(Fc, (uint64_t)(v1 & 7u) * rho + (v1 >> 3), f1);
        if (k2 < e) load_words<KW>(Fc, (uint64_t)(v2 & 7u) * rho + (v2 >> 3), f2);
        if (k3 < e) load_words<KW>(Fc, (uint64_t)(v3 & 7u) * rho + (v3 >> 3), f3);
        uint32_t lack = 0;
#pragma unroll
        for (int w = 0; w < KW; ++w) {
          a[w] |= (f0[w] | f1[w] | f2[w] | f3[w]) & nd[w];
          red[w] = __reduce_or_sync(0xffffffffu, a[w]);
          lack |= nd[w] & ~red[w];
        }
        if (!lack) break;
      }
      if ((int)lane == src) {
#pragma unroll
        for (int w = 0; w < KW; ++w) acc[w] = red[w];
      }
    }
    if (valid && !deferred) {
      uint32_t nw[KW], anyNew = 0, pc = 0;
#pragma unroll
      for (int w = 0; w < KW; ++w) { nw[w] = acc[w] & need[w]; anyNew |= nw[w]; pc += __popc(nw[w]); lv[w] |= nw[w]; }
      store_words<KW>(Fn, idx, nw);  // always: the array still holds the frontier of two levels ago
      if (anyNew) {
#pragma unroll
        for (int w = 0; w < KW; ++w) vc[w] |= nw[w];
        store_words<KW>(p.Vc, idx, vc);
        if (p.farT) p.farT[idx] += (unsigned long long)level * pc;  // Eq. 7: far[idx] += l * popc(diff)
        if (p.reachT) p.reachT[idx] += pc;
        ++nUpd;
      }
    }
  }
  // the CTA's long rows: every warp scans a 128-neighbour share per round, the partial ORs meet in shared memory, one
  // thread per row finalises it
  if (KW >= 4) {
    __syncthreads();
    const uint32_t nLong = min(sh.longCnt, PULL_LONG_CAP);
    for (uint32_t i = 0; i < nLong; ++i) {
      const uint4 row = sh.longRow[i];
      uint32_t a[KW], nd[KW];
      {
        uint32_t vc[KW];
        load_words<KW>(p.Vc, (uint64_t)(row.x & 7u) * rho + (row.x >> 3), vc);  // (one address per warp: a broadcast)
#pragma unroll
        for (int w = 0; w < KW; ++w) { nd[w] = live[w] & ~vc[w]; a[w] = 0; }
      }
      for (uint32_t k = row.y + warp * 128u; k < row.z; k += WARPS_PER_BLOCK * 128u) {
        {  // stop as soon as the warps together have covered every source the row lacks
          uint32_t lack = 0;
#pragma unroll
          for (int w = 0; w < KW; ++w) lack |= nd[w] & ~*(volatile uint32_t*)&sh.longAcc[i][w];
          if (!lack) break;
        }
        uint32_t f0[KW], f1[KW], f2[KW], f3[KW];
#pragma unroll
        for (int w = 0; w < KW; ++w) f0[w] = f1[w] = f2[w] = f3[w] = 0;
        const uint32_t k0 = k + lane, k1 = k + 32u + lane, k2 = k + 64u + lane, k3 = k + 96u + lane;
        uint32_t v0 = 0, v1 = 0, v2 = 0, v3 = 0;
        if (k0 < row.z) v0 = __ldg(&p.colidx[k0]);
        if (k1 < row.z) v1 = __ldg(&p.colidx[k1]);
        if (k2 < row.z) v2 = __ldg(&p.colidx[k2]);
        if (k3 < row.z) v3 = __ldg(&p.colidx[k3]);
        BLEST_ASSERT(v0 < p.n && v1 < p.n && v2 < p.n && v3 < p.n);
        if (k0 < row.z) load_words<KW>(Fc, (uint64_t)(v0 & 7u) * rho + (v0 >> 3), f0);
        if (k1 < row.z) load_words<KW>(Fc, (uint64_t)(v1 & 7u) * rho + (v1 >> 3), f1);
        if (k2 < row.z) load_words<KW>(Fc, (uint64_t)(v2 & 7u) * rho + (v2 >> 3), f2);
        if (k3 < row.z) load_words<KW>(Fc, (uint64_t)(v3 & 7u) * rho + (v3 >> 3), f3);
#pragma unroll
        for (int w = 0; w < KW; ++w) {
          a[w] = (f0[w] | f1[w] | f2[w] | f3[w]) & nd[w];
          const uint32_t r = __reduce_or_sync(0xffffffffu, a[w]);
          if (lane == 0 && r) atomicOr(&sh.longAcc[i][w], r);
        }
        if (lane == 0) nNbr += min(128u, row.z - k);
      }
    }
    __syncthreads();
    if (threadIdx.x < nLong) {
      const uint4 row = sh.longRow[threadIdx.x];
      const uint64_t idx = (uint64_t)(row.x & 7u) * rho + (row.x >> 3);
      uint32_t vc[KW], nw[KW], anyNew = 0, pc = 0;
      load_words<KW>(p.Vc, idx, vc);
#pragma unroll
      for (int w = 0; w < KW; ++w) {
        nw[w] = sh.longAcc[threadIdx.x][w] & live[w] & ~vc[w];
        sh.longAcc[threadIdx.x][w] = 0;
        anyNew |= nw[w]; pc += __popc(nw[w]); lv[w] |= nw[w];
      }
      store_words<KW>(Fn, idx, nw);
      if (anyNew) {
#pragma unroll
        for (int w = 0; w < KW; ++w) vc[w] |= nw[w];
        store_words<KW>(p.Vc, idx, vc);
        if (p.farT) p.farT[idx] += (unsigned long long)level * pc;
        if (p.reachT) p.reachT[idx] += pc;
        ++nUpd;
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) sh.longCnt = 0;
  }
  // the level's termination test is the queue tail (kernel loop): it advances by the number of rows updated
  {
    const uint32_t tot = __reduce_add_sync(0xffffffffu, nUpd);
    if (lane == 0 && tot) atomicAdd(&sh.updAcc, tot);
    if (p.stats) {
      const uint32_t tr = __reduce_add_sync(0xffffffffu, nRows), tn = __reduce_add_sync(0xffffffffu, nNbr);
      if (lane == 0) { sh.cnt[warp][5] += tr; sh.cnt[warp][6] += tn; }
    }
  }
  publish_live<KW>(p, sh, lv, level + 1u);  // (contains a __syncthreads after the accumulation above)
  if (threadIdx.x == 0) {
    if (sh.updAcc) atomicAdd(&p.ctrl->tail, sh.updAcc);
    sh.updAcc = 0;
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
  uint32_t lv[KW];    // OR of the frontier words this thread wrote: the sources still alive (ms_pull_level)
#pragma unroll
  for (int w = 0; w < KW; ++w) pacc[w] = lv[w] = 0;
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
          if (!perSource) {
#pragma unroll
            for (int w = 0; w < KW; ++w) lv[w] |= diff[w];
          }
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
  } else if (p.live) {
    publish_live<KW>(p, sh, lv, level + 1u);
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
  MsShared& sh = *reinterpret_cast<MsShared*>(msDyn);
  constexpr uint32_t KAPPA = 32u * KW;
  unsigned int epoch = 0;
  Ctrl* ctrl = p.ctrl;
  const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (uint64_t)gridDim.x * blockDim.x;
  if (threadIdx.x < WARPS_PER_BLOCK) sh.bigCnt[threadIdx.x] = 0;
  if (threadIdx.x < 256) sh.perSource[threadIdx.x] = 0;
  if (threadIdx.x == 0) { sh.acc = 0; sh.updAcc = 0; sh.longCnt = 0; }
  if (threadIdx.x < PULL_LONG_CAP * 8) sh.longAcc[threadIdx.x / 8][threadIdx.x % 8] = 0;
  if (threadIdx.x < 8) sh.liveAcc[threadIdx.x] = 0;
  if (threadIdx.x < WARPS_PER_BLOCK * 7) sh.cnt[threadIdx.x / 7][threadIdx.x % 7] = 0;
  __syncthreads();
  const uint64_t stateWords = (uint64_t)p.rho * 8u * KW;
  unsigned long long nLevels = 0, nBatches = 0, nPull = 0;

  // phase times as thread 0 of CTA 0 sees them (blest_get_ms_phases): init, Stage 1, its barrier, Stage 2, its barrier;
  // accumulated in shared memory by that one thread
  const bool timing = p.stats != nullptr && gtid == 0;
  if (threadIdx.x == 0) {
    for (int k = 0; k < 5; ++k) sh.tPh[k] = 0;
    sh.tMark = globaltimer();
  }
  auto phase = [&](int k) {
    if (timing) {
      const unsigned long long t = globaltimer();
      sh.tPh[k] += t - sh.tMark;
      sh.tMark = t;
    }
  };
  uint32_t tStart = 0, tEnd = 0;  // queue tail before / after the sweep that filled the current level's queue
  for (uint64_t b0 = 0; b0 < p.nsrcs; b0 += KAPPA) {
    const uint32_t nb = (uint32_t)min((uint64_t)KAPPA, p.nsrcs - b0);
    // init(srcs, ...) (reading R16): visited words cleared, bit c of source c set, its set marked dirty
    grid_fill32(p.Vc, 0u, stateWords);
    grid_fill32(p.Vn, 0u, stateWords);
    if (!PS && p.pullMin && p.live) {
      // a pull level reads the frontier word of EVERY neighbour, also of rows no sweep of this batch has written: those
      // must not hold another batch's bits (bits left by an earlier level of this batch are harmless: such a source has
      // reached all neighbours of that row since)
      grid_fill32(p.F, 0u, stateWords);
      if (gtid < 24) p.live[gtid] = 0;
    }
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
    phase(0);
    bool pull = false;      // this batch has switched to pull levels
    uint32_t* Fcur = p.F;   // the array that holds the current frontier
    uint32_t* Falt = p.F2;
    for (uint32_t level = 1;; ++level) {
      const uint32_t par = level & 1u;
      // a level whose sweep enqueued nothing discovered nothing (every discovered vertex has a neighbour, so its slice
      // set has slices): the queue length the barrier returned is the termination test
      const uint32_t qcount = min(tEnd - tStart, p.qcap);  // (after an overflow the tail counts dropped entries)
      if (qcount == 0) break;
      ++nLevels;
      if (!PS && p.pullMin && p.live) {
        if (gtid < 8) p.live[((level + 2u) % 3u) * 8u + gtid] = 0;  // the slot the NEXT level accumulates into
        // (kappa = 256: the pull level's 32-byte words spill at 64 registers per thread and it measures 4 % slower: never)
        if (KW < 8 && !pull && !p.levels && level >= 2u && qcount >= p.pullMin) pull = true;
      }
      if (!PS && pull) {
        ++nPull;
        const unsigned long long tp0 = timing ? globaltimer() : 0ull;
        ms_pull_level<KW>(p, sh, level, Fcur, Falt);
        phase(1);
        const uint32_t t = grid_barrier_tail(&ctrl->bar, epoch, &sh.tailSlot);
        phase(2);
        if (timing && nLevels <= MS_TRACE_LEVELS) {
          unsigned long long* rec = p.stats + 16 + 4 * (nLevels - 1);
          rec[0] = ((unsigned long long)(level | 0x80000000u) << 32) | qcount;  // bit 63: pull level
          rec[1] = globaltimer() - tp0;
          rec[2] = 0;
          rec[3] = t - tEnd;  // rows updated
        }
        uint32_t* x = Fcur; Fcur = Falt; Falt = x;
        tStart = tEnd;
        tEnd = t;
        continue;
      }
      const unsigned long long tl0 = timing ? globaltimer() : 0ull;
      if (KW == 8) ms_stage1_loop<KW>(p, sh, p.Q[par], qcount);
      else ms_stage1<KW>(p, sh, p.Q[par], qcount);
      phase(1);
      grid_barrier(&ctrl->bar, epoch);
      phase(2);
      const unsigned long long tl1 = timing ? globaltimer() : 0ull;
      ms_stage2<KW, PS>(p, sh, level, b0, nb, p.Q[par ^ 1u], tEnd);
      phase(3);
      const uint32_t t = grid_barrier_tail(&ctrl->bar, epoch, &sh.tailSlot);
      phase(4);
      if (timing && nLevels <= MS_TRACE_LEVELS) {  // per-level record of the launch's first levels
        const unsigned long long tl2 = globaltimer();
        unsigned long long* rec = p.stats + 16 + 4 * (nLevels - 1);
        rec[0] = ((unsigned long long)level << 32) | qcount;
        rec[1] = tl1 - tl0;  // Stage 1 + its barrier
        rec[2] = tl2 - tl1;  // Stage 2 + its barrier
        rec[3] = t - tEnd;   // entries enqueued for the next level
      }
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
      if (cnt[5]) atomicAdd(&p.stats[13], cnt[5]);
      if (cnt[6]) atomicAdd(&p.stats[7], cnt[6]);
    }
    if (gtid == 0) {
      p.stats[5] = nLevels;
      p.stats[6] = nBatches;
      p.stats[14] = nPull;
      for (int k = 0; k < 5; ++k) p.stats[8 + k] = sh.tPh[k];
    }
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
  // MsShared is dynamic shared memory beyond the 48 KB default: opt in once per kernel (and device)
  if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MsShared)) != cudaSuccess) return 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSm, kernel, BLOCK_THREADS, sizeof(MsShared)) != cudaSuccess) return 0;
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
  return cudaLaunchCooperativeKernel(k, dim3(gridBlocks), dim3(BLOCK_THREADS), args, sizeof(MsShared), st);
}

// far0 += far1, reach0 += reach1 (the target-side sums of a concurrent lane, api.cu launch_ms_lanes)
namespace {
__global__ void add_partial_sums_kernel(unsigned long long* far0, uint32_t* reach0, const unsigned long long* far1,
                                        const uint32_t* reach1, uint64_t count) {
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (uint64_t)gridDim.x * blockDim.x) {
    if (far0 && far1) far0[i] += far1[i];
    if (reach0 && reach1) reach0[i] += reach1[i];
  }
}
}  // namespace
cudaError_t launch_add_partial_sums(unsigned long long* far0, uint32_t* reach0, const unsigned long long* far1,
                                    const uint32_t* reach1, uint64_t count, cudaStream_t st) {
  const int threads = 256;
  const int blocks = (int)std::min<uint64_t>((count + threads - 1) / threads, 148ull * 8);
  add_partial_sums_kernel<<<blocks > 0 ? blocks : 1, threads, 0, st>>>(far0, reach0, far1, reach1, count);
  return cudaGetLastError();
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

int max_coop_blocks_msbfs() {  // (also opts every instantiation into its dynamic shared memory)
  int b = coop_blocks(msbfs_kernel<1, false>);
  b = std::min(b, coop_blocks(msbfs_kernel<1, true>));
  b = std::min(b, coop_blocks(msbfs_kernel<2, false>));
  b = std::min(b, coop_blocks(msbfs_kernel<2, true>));
  b = std::min(b, coop_blocks(msbfs_kernel<4, false>));
  b = std::min(b, coop_blocks(msbfs_kernel<4, true>));
  b = std::min(b, coop_blocks(msbfs_kernel<8, false>));
  b = std::min(b, coop_blocks(msbfs_kernel<8, true>));
  return b;
}

}  // namespace blest
