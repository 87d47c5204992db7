// host_graph.h -- host-side pre-processing structures of the BLEST path (reorder, BVSS build, U_div).
#pragma once
#include <cstdint>
#include <vector>

namespace blest {

constexpr uint32_t SIGMA = 8;          // slice width sigma
constexpr uint32_t THETA = 4;          // slices per lane, theta = 32 / sigma
constexpr uint32_t QUADS_PER_VSS = 32; // one quad (4 slices) per lane
constexpr uint32_t JACCARD_WINDOW = 1u << 16;  // W of JaccardWithWindows

struct HostCsr {
  uint32_t n = 0;
  uint64_t nnz = 0;
  std::vector<uint32_t> rowptr, colidx;
};

// BVSS in this library's HBM layout: every slice set is stored as
// ceil(slices/4) quads; quad q holds rowIds[4q..4q+3] (one uint4) and masks[q] (four 8-bit masks, slice c in
// bits 8c..8c+7, bit j = column 8s+j: PAPER.md:302).  VSS v of set s = quads [setPtr[s] + 32(v - realPtrs[s]), +32).
struct HostBvss {
  uint32_t n = 0, Ns = 0, Nv = 0;
  uint64_t nSlices = 0, nQuads = 0;
  std::vector<uint32_t> setPtr;        // Ns+1, quad offsets
  std::vector<uint32_t> rowIds;        // 4*nQuads
  std::vector<uint32_t> masks;         // nQuads
  std::vector<uint32_t> realPtrs;      // Ns+1
  std::vector<uint32_t> virtualToReal; // Nv
  double uDiv = 0.0;
};

// Status codes mirror include/blest.h.
int check_csr(const HostCsr& g, bool validate_symmetry);
// perm[orig] = new id.  kind: 1 RCM, 2 degree-descending (ties by id), 3 JaccardWithWindows (Alg. 1) on
// top of the degree order.
void make_permutation(const HostCsr& g, int kind, std::vector<uint32_t>& perm);
void relabel_csr(const HostCsr& g, const std::vector<uint32_t>& perm, HostCsr& out);
int build_bvss(const HostCsr& g, HostBvss& b);
// From device-built arrays: fills realPtrs / virtualToReal / uDiv given setPtr, rowIds, masks.
void finish_bvss(HostBvss& b);

}  // namespace blest
