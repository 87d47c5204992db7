// bfs_kernels.cuh -- parameter blocks and launch wrappers of the persistent traversal kernels.
#pragma once
#include "device_common.cuh"

namespace blest {

struct BfsParams {
  // graph (immutable during traversal)
  uint32_t n, Ns, nwords, qcap;
  uint64_t nnz;
  const uint32_t* setPtr;  // Ns+1 quad offsets
  const uint4* rowIds;     // nQuads
  const uint32_t* masks;   // nQuads
  const uint32_t* rowptr;  // internal (reordered) CSR, n+1
  const uint32_t* colidx;
  const uint32_t* iperm;   // internal -> original id, or nullptr when no reordering
  // state
  uint32_t* Vcurr;
  uint32_t* Vnext;
  uint32_t* Fcurr;
  uint2* Q[2];
  int32_t* out;    // levels in ORIGINAL ids (device)
  int32_t* L;      // eager: levels in internal ids (== out when iperm == nullptr)
  int32_t* stamp;  // eager: last level at which a slice set was enqueued
  Ctrl* ctrl;
  blest_level_trace_t* trace;
  uint32_t traceCap;
  uint32_t src;  // internal id
  int switching;
  int contraction;
  uint32_t buMask;  // switching == 5: level l runs bottom-up iff bit min(l,31) is set
  float eta, gamma;
};

struct MsParams {
  uint32_t n, Ns, rho, qcap;
  const uint32_t* setPtr;
  const uint4* rowIds;
  const uint32_t* masks;
  const uint32_t* perm;   // original -> internal, or nullptr
  const uint32_t* iperm;  // internal -> original, or nullptr
  uint32_t* F;            // kappa-bit words at getVI index: [rho*8][KW]
  uint32_t* Vc;
  uint32_t* Vn;
  uint8_t* dirty;  // Ns
  uint2* Q[2];
  Ctrl* ctrl;
  const uint32_t* srcs;  // device, original ids; nullptr = identity (source i = vertex i)
  uint64_t nsrcs;
  // outputs (any may be nullptr)
  int32_t* levels;              // [nsrcs][n] original ids
  unsigned long long* farT;     // target-side accumulation, indexed by getVI(internal id) (Eq. 7)
  uint32_t* reachT;
  unsigned long long* farS;     // per-source accumulation [nsrcs]
  uint32_t* reachS;
  int kappa;
};

cudaError_t launch_bfs_lazy(const BfsParams& p, int gridBlocks, cudaStream_t st);
cudaError_t launch_bfs_eager(const BfsParams& p, int gridBlocks, cudaStream_t st);
cudaError_t launch_msbfs(const MsParams& p, int gridBlocks, cudaStream_t st);
cudaError_t launch_closeness_finalize(uint32_t n, uint32_t rho, const uint32_t* perm, const unsigned long long* farT,
                                      const uint32_t* reachT, const unsigned long long* farS, const uint32_t* reachS,
                                      uint64_t nsrcs, double* cc, unsigned long long* farOut, uint32_t* reachOut,
                                      cudaStream_t st);
int max_coop_blocks_lazy();
int max_coop_blocks_eager();
int max_coop_blocks_msbfs();

}  // namespace blest
