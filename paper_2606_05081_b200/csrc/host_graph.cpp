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

// JaccardWithWindows (§4.1, Alg. 1, :116-184): the columns of every window of W consecutive ids are greedily
// grouped into slice sets of sigma columns whose row neighbourhoods overlap (Eq. 3), so that the slices of a set carry
// more than one bit (a denser mask = fewer slices = fewer BVSS bytes per edge).  `g` is symmetric, so nbrs_A = nbrs_A^T
// = the sorted adjacency list, and nbrs(i) restricted to a window is a contiguous sub-range found by binary search.
// slotOf[j] = new id of column j (the paper's pi^-1[j*] <- slot); windows run in parallel (Alg. 1 line 1).
// Readings: "a highest-degree unassigned column" (lines 6, 13) breaks ties by the lowest id; a window's last slice set
// may be short (n not a multiple of sigma); the listing is garbled in PAPER.md and follows the prose of :127-129.
static void jaccard_with_windows(const HostCsr& g, uint32_t W, std::vector<uint32_t>& slotOf) {
  const uint32_t n = g.n;
  slotOf.assign(n, 0);
  const int64_t nWin = ((int64_t)n + W - 1) / W;
#pragma omp parallel
  {
    std::vector<uint64_t> inR(((size_t)n + 63) / 64, 0);  // membership of the current slice set's row set R
    std::vector<uint32_t> rList, inter(W, 0), Q, byDeg(W);
    std::vector<uint8_t> assigned(W, 0);
#pragma omp for schedule(dynamic, 1)
    for (int64_t w = 0; w < nWin; ++w) {
      const uint32_t ws = (uint32_t)(w * W), we = (uint32_t)std::min<uint64_t>((uint64_t)ws + W, n), width = we - ws;
      std::fill(assigned.begin(), assigned.begin() + width, 0);
      for (uint32_t k = 0; k < width; ++k) byDeg[k] = ws + k;
      std::stable_sort(byDeg.begin(), byDeg.begin() + width, [&](uint32_t a, uint32_t b) {
        return (g.rowptr[a + 1] - g.rowptr[a]) > (g.rowptr[b + 1] - g.rowptr[b]);
      });
      uint32_t nextByDeg = 0;  // byDeg[nextByDeg..] holds every unassigned column at or after the best one
      uint64_t sizeR = 0;
      auto highest_unassigned = [&]() -> uint32_t {
        while (assigned[byDeg[nextByDeg] - ws]) ++nextByDeg;
        return byDeg[nextByDeg];
      };
      // R <- R u nbrs(j); every new row i bumps inter[] of the unassigned window columns it touches (Alg. 1 l.16-22 / l.9)
      auto absorb = [&](uint32_t j) {
        for (uint32_t e = g.rowptr[j]; e < g.rowptr[j + 1]; ++e) {
          const uint32_t i = g.colidx[e];
          if ((inR[i >> 6] >> (i & 63)) & 1ull) continue;
          inR[i >> 6] |= 1ull << (i & 63);
          rList.push_back(i);
          ++sizeR;
          const uint32_t* b = g.colidx.data() + g.rowptr[i];
          const uint32_t* en = g.colidx.data() + g.rowptr[i + 1];
          for (const uint32_t* q = std::lower_bound(b, en, ws); q < en && *q < we; ++q) {
            const uint32_t k = *q - ws;
            if (assigned[k]) continue;
            if (inter[k]++ == 0) Q.push_back(*q);
          }
        }
      };
      for (uint32_t ss = ws; ss < we; ss += SIGMA) {
        const uint32_t se = std::min(ss + SIGMA, we);
        sizeR = 0;
        uint32_t j = highest_unassigned();  // seed (line 6)
        assigned[j - ws] = 1;
        slotOf[j] = ss;
        absorb(j);
        for (uint32_t l = ss + 1; l < se; ++l) {
          uint32_t best = 0xFFFFFFFFu;
          double bestScore = -1.0;
          size_t keep = 0;
          for (size_t t = 0; t < Q.size(); ++t) {  // argmax over Q of inter / (|R| + deg - inter) (line 14)
            const uint32_t c = Q[t];
            if (assigned[c - ws]) continue;  // taken since it entered Q
            Q[keep++] = c;
            const double it = inter[c - ws], dg = g.rowptr[c + 1] - g.rowptr[c];
            const double score = it / ((double)sizeR + dg - it);
            if (score > bestScore || (score == bestScore && c < best)) { bestScore = score; best = c; }
          }
          Q.resize(keep);
          j = best != 0xFFFFFFFFu ? best : highest_unassigned();  // Q empty: fallback (line 13)
          assigned[j - ws] = 1;
          slotOf[j] = l;
          absorb(j);
        }
        for (uint32_t i : rList) inR[i >> 6] &= ~(1ull << (i & 63));
        rList.clear();
        for (uint32_t c : Q) inter[c - ws] = 0;
        Q.clear();
      }
      std::fill(inter.begin(), inter.begin() + width, 0);
    }
  }
}

void make_permutation(const HostCsr& g, int kind, std::vector<uint32_t>& perm) {
  const uint32_t n = g.n;
  if (kind == 3) {
    // Degree order first, then JaccardWithWindows inside windows of the degree order: on a graph whose natural ids are a
    // random relabelling (BASELINE.json's RMAT configs) a window of natural ids has no structure to exploit, while a
    // window of the degree order holds columns of similar degree -- the hubs, whose neighbourhoods overlap most, first.
    std::vector<uint32_t> p1, slotOf;
    make_permutation(g, 2, p1);
    HostCsr g1;
    relabel_csr(g, p1, g1);
    jaccard_with_windows(g1, JACCARD_WINDOW, slotOf);
    perm.resize(n);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) perm[i] = slotOf[p1[i]];
    return;
  }
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
