// graphgen/gen.cpp -- seeded synthetic graph generators (input plumbing only).
//
// This module is shared by the CPU oracle's tests and by the CUDA path's tests / bench.  It holds
// NONE of the method's arithmetic (no BFS, no BVSS, no bitmaps): it only draws edges from a seeded
// counter-based hash and turns an edge list into a symmetric, loop-free, duplicate-free uint32 CSR,
// the input format BASELINE.json's configs name.  Shapes follow DESIGN.md "Input recipe":
//   * RMAT (Graph500 a,b,c,d per bit level, optional seeded relabelling)          -> configs 1, 4, 5
//   * 4-connected 2-D grid, row-major ids, each lattice edge deleted with prob. p  -> config 2
//   * uniform G(n,m), i.i.d. endpoints                                             -> config 3
// Every draw is a pure function of (seed, edge index), so results do not depend on thread count.
#include <algorithm>
#include <atomic>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <omp.h>

namespace {

inline uint64_t mix64(uint64_t x) {  // splitmix64 finaliser
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}
inline uint64_t draw(uint64_t seed, uint64_t idx, uint64_t stream) {
  return mix64(mix64(seed ^ (stream * 0xD6E8FEB86659FD93ull)) + idx);
}
inline uint64_t bounded(uint64_t h, uint64_t n) {  // unbiased enough: 64x64 -> high 64
  return (uint64_t)(((unsigned __int128)h * n) >> 64);
}

}  // namespace

extern "C" {

// RMAT edge list.  m = edge_factor << scale edges; per bit level one 32-bit uniform chooses the
// quadrant with probabilities (a, b, c, d = 1-a-b-c).  perm (may be NULL) relabels vertex ids.
void gg_rmat_edges(int scale, uint64_t m, uint64_t seed, double a, double b, double c,
                   const uint32_t* perm, uint32_t* src, uint32_t* dst) {
  const uint64_t ta = (uint64_t)(a * 4294967296.0);
  const uint64_t tb = (uint64_t)((a + b) * 4294967296.0);
  const uint64_t tc = (uint64_t)((a + b + c) * 4294967296.0);
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < (int64_t)m; ++e) {
    uint32_t u = 0, v = 0;
    uint64_t h = 0;
    for (int lvl = 0; lvl < scale; ++lvl) {
      if ((lvl & 1) == 0) h = draw(seed, (uint64_t)e, 1 + (lvl >> 1));
      uint64_t r = (lvl & 1) ? (h >> 32) : (h & 0xFFFFFFFFull);
      uint32_t ub, vb;
      if (r < ta) { ub = 0; vb = 0; }
      else if (r < tb) { ub = 0; vb = 1; }
      else if (r < tc) { ub = 1; vb = 0; }
      else { ub = 1; vb = 1; }
      u = (u << 1) | ub;
      v = (v << 1) | vb;
    }
    if (perm) { u = perm[u]; v = perm[v]; }
    src[e] = u;
    dst[e] = v;
  }
}

// Seeded Fisher-Yates permutation of [0, n).
void gg_random_perm(uint32_t n, uint64_t seed, uint32_t* perm) {
  for (uint32_t i = 0; i < n; ++i) perm[i] = i;
  for (uint32_t i = n; i > 1; --i) {
    uint32_t j = (uint32_t)bounded(draw(seed, i, 77), i);
    std::swap(perm[i - 1], perm[j]);
  }
}

// 4-connected rows x cols lattice, vertex id r*cols + c.  Lattice edge k (horizontal edges first,
// then vertical) is kept iff its uniform draw >= delete_frac.  Returns the number of kept edges;
// src/dst must hold rows*(cols-1) + (rows-1)*cols entries.
uint64_t gg_grid_edges(uint32_t rows, uint32_t cols, double delete_frac, uint64_t seed,
                       uint32_t* src, uint32_t* dst) {
  const uint64_t nh = (uint64_t)rows * (cols - 1), nv = (uint64_t)(rows - 1) * cols;
  const uint64_t thr = (uint64_t)(delete_frac * 18446744073709551616.0);
  uint64_t kept = 0;
  // serial compaction keeps the edge order (and thus the output) independent of thread count
  for (uint64_t k = 0; k < nh + nv; ++k) {
    if (delete_frac > 0.0 && draw(seed, k, 3) < thr) continue;
    uint32_t u, v;
    if (k < nh) { uint32_t r = (uint32_t)(k / (cols - 1)), c = (uint32_t)(k % (cols - 1)); u = r * cols + c; v = u + 1; }
    else { uint64_t kk = k - nh; uint32_t r = (uint32_t)(kk / cols), c = (uint32_t)(kk % cols); u = r * cols + c; v = u + cols; }
    src[kept] = u; dst[kept] = v; ++kept;
  }
  return kept;
}

// Uniform G(n, m): both endpoints i.i.d. uniform on [0, n).
void gg_gnm_edges(uint32_t n, uint64_t m, uint64_t seed, uint32_t* src, uint32_t* dst) {
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < (int64_t)m; ++e) {
    src[e] = (uint32_t)bounded(draw(seed, (uint64_t)e, 5), n);
    dst[e] = (uint32_t)bounded(draw(seed, (uint64_t)e, 6), n);
  }
}

// Edge list -> symmetric CSR: drop self-loops, add the reverse of every edge, sort every row, drop
// duplicates.  rowptr has n+1 entries; colidx must hold 2*m entries (upper bound).  Returns nnz, or
// UINT64_MAX if nnz would not fit uint32.
uint64_t gg_edges_to_csr(uint32_t n, uint64_t m, const uint32_t* src, const uint32_t* dst,
                         uint32_t* rowptr, uint32_t* colidx) {
  std::vector<uint64_t> off((size_t)n + 1, 0);
  {
    std::vector<std::atomic<uint32_t>> deg(n);
    for (auto& d : deg) d.store(0, std::memory_order_relaxed);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < (int64_t)m; ++e) {
      uint32_t u = src[e], v = dst[e];
      if (u == v) continue;
      deg[u].fetch_add(1, std::memory_order_relaxed);
      deg[v].fetch_add(1, std::memory_order_relaxed);
    }
    for (uint32_t i = 0; i < n; ++i) off[i + 1] = off[i] + deg[i].load(std::memory_order_relaxed);
  }
  const uint64_t raw = off[n];
  std::vector<uint32_t> adj(raw);
  {
    std::vector<std::atomic<uint64_t>> cur(n);
    for (uint32_t i = 0; i < n; ++i) cur[i].store(off[i], std::memory_order_relaxed);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < (int64_t)m; ++e) {
      uint32_t u = src[e], v = dst[e];
      if (u == v) continue;
      adj[cur[u].fetch_add(1, std::memory_order_relaxed)] = v;
      adj[cur[v].fetch_add(1, std::memory_order_relaxed)] = u;
    }
  }
  std::vector<uint32_t> ucount(n);
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    uint32_t* b = adj.data() + off[i];
    uint32_t* e = adj.data() + off[i + 1];
    std::sort(b, e);
    ucount[i] = (uint32_t)(std::unique(b, e) - b);
  }
  uint64_t nnz = 0;
  for (uint32_t i = 0; i < n; ++i) { rowptr[i] = (uint32_t)nnz; nnz += ucount[i]; }
  if (nnz > 0xFFFFFFFFull) return UINT64_MAX;
  rowptr[n] = (uint32_t)nnz;
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t i = 0; i < (int64_t)n; ++i)
    std::memcpy(colidx + rowptr[i], adj.data() + off[i], (size_t)ucount[i] * sizeof(uint32_t));
  return nnz;
}

int gg_num_threads(void) { return omp_get_max_threads(); }

}  // extern "C"
