// host_graph.cpp -- host pre-processing of the BLEST path: CSR checks, reordering (§4), BVSS build
// (§3.1) and the update-divergence statistic.  OpenMP over slice sets / rows.
#include "host_graph.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <numeric>
#include <omp.h>

#include "../../include/blest.h"

namespace blest {

int check_csr(const HostCsr& g, bool validate_symmetry) {
  const uint32_t n = g.n;
  if (n == 0 || n > (1u << 29)) return BLEST_ERANGE;
  if (g.nnz > 0xFFFFFFFFull) return BLEST_ERANGE;
  if (g.rowptr[0] != 0 || g.rowptr[n] != (uint32_t)g.nnz) return BLEST_EINVAL;
  int bad = 0;  // 1 unsorted, 2 rowptr decreasing, 4 range
#pragma omp parallel for schedule(dynamic, 4096) reduction(| : bad)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    uint32_t b = g.rowptr[i], e = g.rowptr[i + 1];
    if (e < b || e > g.nnz) { bad |= 2; continue; }  // malformed rowptr: never walk colidx past nnz
    for (uint32_t p = b; p < e; ++p) {
      if (g.colidx[p] >= n) bad |= 4;
      if (p > b && g.colidx[p] < g.colidx[p - 1]) bad |= 1;
    }
  }
  if (bad & 2) return BLEST_EINVAL;
  if (bad & 4) return BLEST_ENOTSYM;  // column id out of range: treated as malformed structure
  if (bad & 1) return BLEST_EUNSORTED;
  if (validate_symmetry) {
    int asym = 0;
#pragma omp parallel for schedule(dynamic, 4096) reduction(| : asym)
    for (int64_t i = 0; i < (int64_t)n; ++i)
      for (uint32_t p = g.rowptr[i]; p < g.rowptr[i + 1]; ++p) {
        uint32_t v = g.colidx[p];
        const uint32_t* b = g.colidx.data() + g.rowptr[v];
        const uint32_t* e = g.colidx.data() + g.rowptr[v + 1];
        if (!std::binary_search(b, e, (uint32_t)i)) asym = 1;
      }
    if (asym) return BLEST_ENOTSYM;
  }
  return BLEST_OK;
}

// ---- reordering (A1) -----------------------------------------------------------------------------
static void rcm_order(const HostCsr& g, std::vector<uint32_t>& order) {
  // Reverse Cuthill-McKee: BFS-like visit order, the unvisited neighbours of each popped vertex
  // appended in ascending degree; components started from their lowest-degree vertex; finally reversed.
  const uint32_t n = g.n;
  std::vector<uint32_t> deg(n), byDeg(n);
  for (uint32_t i = 0; i < n; ++i) deg[i] = g.rowptr[i + 1] - g.rowptr[i];
  std::iota(byDeg.begin(), byDeg.end(), 0u);
  std::stable_sort(byDeg.begin(), byDeg.end(), [&](uint32_t a, uint32_t b) { return deg[a] < deg[b]; });
  std::vector<uint8_t> seen(n, 0);
  order.clear();
  order.reserve(n);
  std::vector<uint32_t> nb;
  for (uint32_t k = 0; k < n; ++k) {
    uint32_t s = byDeg[k];
    if (seen[s]) continue;
    seen[s] = 1;
    size_t head = order.size();
    order.push_back(s);
    while (head < order.size()) {
      uint32_t u = order[head++];
      nb.clear();
      for (uint32_t p = g.rowptr[u]; p < g.rowptr[u + 1]; ++p) {
        uint32_t v = g.colidx[p];
        if (!seen[v]) { seen[v] = 1; nb.push_back(v); }
      }
      std::sort(nb.begin(), nb.end(), [&](uint32_t a, uint32_t b) { return deg[a] != deg[b] ? deg[a] < deg[b] : a < b; });
      order.insert(order.end(), nb.begin(), nb.end());
    }
  }
  std::reverse(order.begin(), order.end());
}

void make_permutation(const HostCsr& g, int kind, std::vector<uint32_t>& perm) {
  const uint32_t n = g.n;
  std::vector<uint32_t> order;  // order[new] = orig
  if (kind == 1) {
    rcm_order(g, order);
  } else {
    order.resize(n);
    std::iota(order.begin(), order.end(), 0u);
    std::stable_sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) {
      return (g.rowptr[a + 1] - g.rowptr[a]) > (g.rowptr[b + 1] - g.rowptr[b]);
    });
  }
  perm.resize(n);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < (int64_t)n; ++i) perm[order[i]] = (uint32_t)i;
}

void relabel_csr(const HostCsr& g, const std::vector<uint32_t>& perm, HostCsr& out) {
  const uint32_t n = g.n;
  out.n = n;
  out.nnz = g.nnz;
  out.rowptr.assign((size_t)n + 1, 0);
  out.colidx.resize(g.nnz);
  for (uint32_t i = 0; i < n; ++i) out.rowptr[perm[i] + 1] = g.rowptr[i + 1] - g.rowptr[i];
  for (uint32_t i = 0; i < n; ++i) out.rowptr[i + 1] += out.rowptr[i];
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    uint32_t* dst = out.colidx.data() + out.rowptr[perm[i]];
    uint32_t d = g.rowptr[i + 1] - g.rowptr[i];
    const uint32_t* src = g.colidx.data() + g.rowptr[i];
    for (uint32_t k = 0; k < d; ++k) dst[k] = perm[src[k]];
    std::sort(dst, dst + d);
  }
}

// ---- BVSS build (A2) -----------------------------------------------------------------------------
// Slice set s covers columns [8s, 8s+8).  The graph is symmetric, so the rows with a non-zero in column j are
// the neighbours of j: the slices of set s are the distinct vertices of the union of the 8 (sorted) adjacency
// lists, each with the mask of which of the 8 lists contain it.  An 8-way merge emits them in
// ascending row id (reading R8).  emit == nullptr: count only.
template <class Emit>
static inline uint64_t merge_set(const HostCsr& g, uint32_t s, Emit&& emit) {
  uint32_t p[SIGMA], e[SIGMA];
  for (uint32_t j = 0; j < SIGMA; ++j) {
    uint64_t v = (uint64_t)s * SIGMA + j;
    if (v < g.n) { p[j] = g.rowptr[v]; e[j] = g.rowptr[v + 1]; }
    else { p[j] = e[j] = 0; }
  }
  uint64_t cnt = 0;
  for (;;) {
    uint32_t best = 0xFFFFFFFFu;
    for (uint32_t j = 0; j < SIGMA; ++j)
      if (p[j] < e[j]) best = std::min(best, g.colidx[p[j]]);
    if (best == 0xFFFFFFFFu) break;
    uint32_t mask = 0;
    for (uint32_t j = 0; j < SIGMA; ++j)
      while (p[j] < e[j] && g.colidx[p[j]] == best) { mask |= 1u << j; ++p[j]; }  // duplicates collapse
    emit(cnt, best, mask);
    ++cnt;
  }
  return cnt;
}

int build_bvss(const HostCsr& g, HostBvss& b) {
  const uint32_t n = g.n;
  const uint32_t Ns = (uint32_t)(((uint64_t)n + SIGMA - 1) / SIGMA);
  b.n = n;
  b.Ns = Ns;
  std::vector<uint64_t> cnt((size_t)Ns + 1, 0);
#pragma omp parallel for schedule(dynamic, 512)
  for (int64_t s = 0; s < (int64_t)Ns; ++s)
    cnt[s + 1] = merge_set(g, (uint32_t)s, [](uint64_t, uint32_t, uint32_t) {});
  b.setPtr.assign((size_t)Ns + 1, 0);
  uint64_t slices = 0, quads = 0;
  for (uint32_t s = 0; s < Ns; ++s) {
    slices += cnt[s + 1];
    quads += (cnt[s + 1] + 3) / 4;
    if (quads > 0xFFFFFFFFull) return BLEST_ERANGE;
    b.setPtr[s + 1] = (uint32_t)quads;
  }
  b.nSlices = slices;
  b.nQuads = quads;
  b.rowIds.assign((size_t)quads * 4, 0);
  b.masks.assign((size_t)quads, 0);
#pragma omp parallel for schedule(dynamic, 512)
  for (int64_t s = 0; s < (int64_t)Ns; ++s) {
    const uint64_t base = (uint64_t)b.setPtr[s] * 4;
    uint32_t last = 0;
    uint64_t c = merge_set(g, (uint32_t)s, [&](uint64_t k, uint32_t row, uint32_t mask) {
      b.rowIds[base + k] = row;
      b.masks[(base + k) >> 2] |= mask << (8 * ((base + k) & 3));
      last = row;
    });
    // padding slices: a valid row id with an all-zero mask ("zero-padded ... arbitrary row IDs")
    for (uint64_t k = c; k < (uint64_t)(b.setPtr[s + 1] - b.setPtr[s]) * 4; ++k) b.rowIds[base + k] = last;
  }
  finish_bvss(b);
  return BLEST_OK;
}

void finish_bvss(HostBvss& b) {
  const uint32_t Ns = b.Ns;
  b.realPtrs.assign((size_t)Ns + 1, 0);
  uint64_t nv = 0;
  for (uint32_t s = 0; s < Ns; ++s) {
    nv += (b.setPtr[s + 1] - b.setPtr[s] + QUADS_PER_VSS - 1) / QUADS_PER_VSS;
    b.realPtrs[s + 1] = (uint32_t)nv;
  }
  b.Nv = (uint32_t)nv;
  b.virtualToReal.resize(nv);
#pragma omp parallel for schedule(dynamic, 4096)
  for (int64_t s = 0; s < (int64_t)Ns; ++s)
    for (uint32_t v = b.realPtrs[s]; v < b.realPtrs[s + 1]; ++v) b.virtualToReal[v] = (uint32_t)s;

  // Update divergence (reading R20): per VSS, for each of the theta = 4 columns of the 32 x 4
  // VSS matrix (slices at lane*4 + c), the population standard deviation of the row ids with non-zero mask;
  // set divergence = mean over non-empty columns; U_div = mean over all VSSs.
  double total = 0.0;
#pragma omp parallel for schedule(dynamic, 4096) reduction(+ : total)
  for (int64_t v = 0; v < (int64_t)nv; ++v) {
    uint32_t s = b.virtualToReal[v];
    uint64_t q0 = (uint64_t)b.setPtr[s] + (uint64_t)(v - b.realPtrs[s]) * QUADS_PER_VSS;
    uint64_t q1 = std::min<uint64_t>(q0 + QUADS_PER_VSS, b.setPtr[s + 1]);
    double acc = 0.0;
    int cols = 0;
    for (uint32_t c = 0; c < THETA; ++c) {
      double sum = 0.0, sq = 0.0;
      uint32_t k = 0;
      for (uint64_t q = q0; q < q1; ++q)
        if ((b.masks[q] >> (8 * c)) & 0xFF) { sum += (double)b.rowIds[q * 4 + c]; ++k; }
      if (k) {
        const double mean = sum / k;  // two-pass: ids up to 2^29 would cancel in E[r^2] - mean^2
        for (uint64_t q = q0; q < q1; ++q)
          if ((b.masks[q] >> (8 * c)) & 0xFF) { double d = (double)b.rowIds[q * 4 + c] - mean; sq += d * d; }
        acc += std::sqrt(sq / k);
        ++cols;
      }
    }
    if (cols) total += acc / cols;
  }
  b.uDiv = nv ? total / (double)nv : 0.0;
}

}  // namespace blest
