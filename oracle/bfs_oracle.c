/* oracle/bfs_oracle.c -- the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct implementation of what the BLEST hot path computes, written from
 * the paper, independent of the CUDA path: it shares no code, header,
 * table or helper with paper_2606_05081_b200/ and reads only the ORIGINAL uint32 CSR (no BVSS, no
 * permutation, no bitmaps).  Row u lists the out-neighbours of u: for the symmetric configs that is
 * simply the neighbours; for a directed graph the queue BFS follows the edge direction, which is
 * Eq. 1 with A = the transposed adjacency matrix.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.
 *
 * BLEST is exact, not approximate (PAPER.md:59 "The emulation is exact"; :337-339 the lazy scheme and
 * switching only change when work happens), so the oracle is the plain DEFINITION of the result:
 *
 *   level[i] = k such that x_i^(k) = 1 under x^(k+1) = (A x^(k)) AND NOT v^(k), x_s^(0) = 1
 *              (Eq. 1) = the hop distance from the source; "infinity" for an
 *              unreachable vertex, stored as -1 (BASELINE.json; reading R1).
 *   far[s]   = sum over reachable v of level_s[v]                       (Eq. 7)
 *   cc[s]    = (reach_s - 1) / far[s], 0.0 when far = 0                 (Eq. 8 with the
 *              "normalization using component sizes" for disconnected graphs; reading R14)
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms (path, cycle, grid = Manhattan,
 * complete, star, binary tree, disjoint unions, isolated source), invariants on random graphs,
 * literal Eq. 1 Boolean-matrix-power brute force for n <= 64, scipy.sparse.csgraph on larger graphs,
 * farness closed forms; the same on directed graphs (one-way path / cycle / stars, Eq. 1 with
 * A[v][u] = 1 for u -> v, scipy directed shortest paths).  No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* FIFO-queue BFS.  queue: caller scratch of n uint32. Returns #reached (incl. src). */
static uint32_t bfs_core(uint32_t n, const uint32_t *rowptr, const uint32_t *colidx, uint32_t src,
                         int32_t *level, uint32_t *queue) {
  for (uint32_t i = 0; i < n; ++i) level[i] = -1; /* "level[i] = infinity" */
  uint32_t head = 0, tail = 0;
  level[src] = 0; /* x_s^(0) = 1 */
  queue[tail++] = src;
  while (head < tail) {
    uint32_t u = queue[head++];
    for (uint32_t e = rowptr[u]; e < rowptr[u + 1]; ++e) {
      uint32_t v = colidx[e];
      if (level[v] < 0) { /* not visited at any earlier level */
        level[v] = level[u] + 1;
        queue[tail++] = v;
      }
    }
  }
  return tail;
}

/* Single-source BFS.  level: int32[n], -1 = unreachable.  Returns 0, or -1 on bad arguments. */
int oracle_bfs(uint32_t n, const uint32_t *rowptr, const uint32_t *colidx, uint32_t src, int32_t *level) {
  if (!rowptr || !level || src >= n) return -1;
  uint32_t *queue = (uint32_t *)malloc((size_t)n * sizeof(uint32_t));
  if (!queue) return -2;
  bfs_core(n, rowptr, colidx, src, level, queue);
  free(queue);
  return 0;
}

/* Multi-source BFS = k independent single-source runs (kappa concurrent BFS instances).
 * levels: int32[k*n], row b belongs to srcs[b]. */
int oracle_msbfs(uint32_t n, const uint32_t *rowptr, const uint32_t *colidx, const uint32_t *srcs,
                 uint32_t k, int32_t *levels) {
  for (uint32_t b = 0; b < k; ++b) {
    int rc = oracle_bfs(n, rowptr, colidx, srcs[b], levels + (size_t)b * n);
    if (rc) return rc;
  }
  return 0;
}

/* Farness and reach of one level array (Eq. 7): far = sum of levels of reachable vertices,
 * reach = number of reachable vertices including the source. */
void oracle_farness(uint32_t n, const int32_t *level, uint64_t *far, uint32_t *reach) {
  uint64_t f = 0;
  uint32_t r = 0;
  for (uint32_t i = 0; i < n; ++i)
    if (level[i] >= 0) { f += (uint64_t)level[i]; ++r; }
  *far = f;
  *reach = r;
}

/* cc = (reach-1)/far in fp64, one IEEE division; 0.0 for an isolated source (far = 0). */
double oracle_closeness_value(uint32_t reach, uint64_t far) {
  return far == 0 ? 0.0 : (double)(reach - 1) / (double)far;
}

/* Farness / reach / closeness of each source in srcs (srcs == NULL: all vertices 0..nsrcs-1).
 * Each source is one plain BFS; sources are spread over OpenMP threads (nthreads <= 0: all).
 * Any of far / reach / cc may be NULL.  Returns the number of threads used (> 0) or < 0 on error. */
int oracle_closeness(uint32_t n, const uint32_t *rowptr, const uint32_t *colidx, const uint32_t *srcs,
                     uint64_t nsrcs, uint64_t *far, uint32_t *reach, double *cc, int nthreads) {
  int used = 1, err = 0;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel num_threads(nthreads)
#endif
  {
    int32_t *level = (int32_t *)malloc((size_t)n * sizeof(int32_t));
    uint32_t *queue = (uint32_t *)malloc((size_t)n * sizeof(uint32_t));
#ifdef _OPENMP
#pragma omp single
    used = omp_get_num_threads();
#pragma omp for schedule(dynamic, 4)
#endif
    for (int64_t i = 0; i < (int64_t)nsrcs; ++i) {
      uint32_t s = srcs ? srcs[i] : (uint32_t)i;
      if (!level || !queue || s >= n) { err = 1; continue; }
      bfs_core(n, rowptr, colidx, s, level, queue);
      uint64_t f; uint32_t r;
      oracle_farness(n, level, &f, &r);
      if (far) far[i] = f;
      if (reach) reach[i] = r;
      if (cc) cc[i] = oracle_closeness_value(r, f);
    }
    free(level);
    free(queue);
  }
  return err ? -1 : used;
}

/* Edges of the source's connected component, each undirected edge once (BASELINE.json's TEPS
 * numerator): (sum of degrees of reachable vertices) / 2. */
uint64_t oracle_component_edges(uint32_t n, const uint32_t *rowptr, const int32_t *level) {
  uint64_t s = 0;
  for (uint32_t i = 0; i < n; ++i)
    if (level[i] >= 0) s += rowptr[i + 1] - rowptr[i];
  return s / 2;
}
