/*
 * polfed_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, scalar fp64 CPU statement of what POLFED's hot path computes
 * (arxiv/paper_2605_10191; citations are PAPER.md line numbers).  It shares no
 * code with the CUDA library and may be imported only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * Contents (DESIGN.md section "Oracle"):
 *   O1  orc_basis_enumerate / orc_basis_rank   fixed-popcount basis, ascending integers
 *   O2  orc_build_csr                          scalar CSR assembly from a term list
 *   O3  orc_spmm                               Y = H X on an n x s row-major block (Eq. 8)
 *   O4  orc_rescale                            H~X = (HX - aX)/b               (Eq. 31)
 *   O6  orc_clenshaw                           W = sum_k c_k T_k(H~) V          (Eq. 51)
 *
 * The only parallelism is an OpenMP "parallel for" over rows; each row's
 * arithmetic is sequential in stored order, so results do not depend on the
 * thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
  int32_t kind;
  int32_t i;
  int32_t j;
  double amp;
} orc_term;

enum { ORC_ZZ = 0, ORC_Z = 1, ORC_NN = 2, ORC_N = 3, ORC_EXCH = 4, ORC_HOPJW = 5, ORC_XX = 6 };

/* ---- O1: basis ---------------------------------------------------------- */

/* All x in [0, 2^n_sites) with popcount(x) == n_up, ascending (n_up < 0: all x).
 * Brute force over every integer.  states == NULL: count only.  Returns the count. */
int64_t orc_basis_enumerate(int n_sites, int n_up, uint64_t *states) {
  int64_t count = 0;
  uint64_t top = 1ull << n_sites;
  for (uint64_t x = 0; x < top; ++x) {
    if (n_up < 0 || __builtin_popcountll(x) == n_up) {
      if (states) states[count] = x;
      ++count;
    }
  }
  return count;
}

/* Position of x in the ascending list (binary search); -1 if absent. */
int64_t orc_basis_rank(const uint64_t *states, int64_t dim, uint64_t x) {
  int64_t lo = 0, hi = dim - 1;
  while (lo <= hi) {
    int64_t mid = lo + (hi - lo) / 2;
    if (states[mid] == x) return mid;
    if (states[mid] < x) lo = mid + 1; else hi = mid - 1;
  }
  return -1;
}

/* ---- O2: CSR assembly --------------------------------------------------- */

typedef struct { int64_t col; double val; int32_t seq; } orc_entry;

static int entry_cmp(const void *pa, const void *pb) {
  const orc_entry *a = (const orc_entry *)pa, *b = (const orc_entry *)pb;
  if (a->col != b->col) return a->col < b->col ? -1 : 1;
  return a->seq - b->seq;            /* keep term order among equal columns */
}

/* Entries of row r (state x) before merging.  The diagonal is entry 0 (always
 * present); dot-block off-diagonals next; then one entry per term that acts
 * non-trivially, in term order.  Returns the entry count or -1 when a term
 * leaves the basis. */
static int row_entries(const uint64_t *states, int64_t dim, int64_t r,
                       const orc_term *terms, int n_terms, int dot_bits,
                       const double *dot_dense, orc_entry *e) {
  uint64_t x = states[r];
  int n = 0;
  double diag = 0.0;
  e[n].col = r; e[n].val = 0.0; e[n].seq = n; ++n;
  if (dot_bits > 0) {
    uint64_t dd = 1ull << dot_bits, mask = dd - 1, d = x & mask;
    diag += dot_dense[d * dd + d];
    for (uint64_t d2 = 0; d2 < dd; ++d2) {
      if (d2 == d) continue;
      int64_t c = orc_basis_rank(states, dim, (x & ~mask) | d2);
      if (c < 0) return -1;
      e[n].col = c; e[n].val = dot_dense[d * dd + d2]; e[n].seq = n; ++n;
    }
  }
  for (int t = 0; t < n_terms; ++t) {
    int i = terms[t].i, j = terms[t].j;
    double amp = terms[t].amp;
    int bi = (int)((x >> i) & 1), bj = (int)((x >> j) & 1);
    switch (terms[t].kind) {
      case ORC_ZZ: diag += amp * ((bi ? 0.5 : -0.5) * (bj ? 0.5 : -0.5)); break;
      case ORC_Z:  diag += amp * (bi ? 0.5 : -0.5); break;
      case ORC_NN: diag += amp * (double)(bi * bj); break;
      case ORC_N:  diag += amp * (double)bi; break;
      case ORC_EXCH:
      case ORC_HOPJW:
        if (bi != bj) {
          uint64_t y = x ^ (1ull << i) ^ (1ull << j);
          double v = amp;
          if (terms[t].kind == ORC_HOPJW) {
            int lo = i < j ? i : j, hi = i < j ? j : i, between = 0;
            for (int l = lo + 1; l < hi; ++l) between += (int)((x >> l) & 1);
            if (between & 1) v = -amp;
          }
          int64_t c = orc_basis_rank(states, dim, y);
          if (c < 0) return -1;
          e[n].col = c; e[n].val = v; e[n].seq = n; ++n;
        }
        break;
      case ORC_XX: {
        uint64_t y = x ^ (1ull << i) ^ (1ull << j);
        int64_t c = orc_basis_rank(states, dim, y);
        if (c < 0) return -1;
        e[n].col = c; e[n].val = amp; e[n].seq = n; ++n;
        break;
      }
      default: return -1;
    }
  }
  e[0].val = diag;
  return n;
}

/* Sort by column (stable in term order) and sum duplicates left to right. */
static int merge_entries(orc_entry *e, int n) {
  qsort(e, (size_t)n, sizeof(orc_entry), entry_cmp);
  int m = 0;
  for (int k = 0; k < n; ++k) {
    if (m > 0 && e[m - 1].col == e[k].col) e[m - 1].val += e[k].val;
    else e[m++] = e[k];
  }
  return m;
}

/* Two calls: col == NULL fills row_ptr (int32[dim+1]) and returns nnz;
 * otherwise fills col/val using row_ptr.  Returns -1 on error. */
int64_t orc_build_csr(const uint64_t *states, int64_t dim, const orc_term *terms,
                      int n_terms, int dot_bits, const double *dot_dense,
                      int32_t *row_ptr, int32_t *col, double *val) {
  int cap = n_terms + (dot_bits > 0 ? (1 << dot_bits) : 0) + 1;
  int err = 0;
  if (!col) {
    int32_t *cnt = (int32_t *)malloc(sizeof(int32_t) * (size_t)(dim + 1));
    if (!cnt) return -1;
#pragma omp parallel
    {
      orc_entry *e = (orc_entry *)malloc(sizeof(orc_entry) * (size_t)cap);
#pragma omp for schedule(static)
      for (int64_t r = 0; r < dim; ++r) {
        int n = row_entries(states, dim, r, terms, n_terms, dot_bits, dot_dense, e);
        if (n < 0) { err = 1; cnt[r] = 0; } else cnt[r] = merge_entries(e, n);
      }
      free(e);
    }
    int64_t total = 0;
    for (int64_t r = 0; r < dim; ++r) { row_ptr[r] = (int32_t)total; total += cnt[r]; }
    free(cnt);
    if (err || total > 2147483647ll) return -1;
    row_ptr[dim] = (int32_t)total;
    return total;
  }
#pragma omp parallel
  {
    orc_entry *e = (orc_entry *)malloc(sizeof(orc_entry) * (size_t)cap);
#pragma omp for schedule(static)
    for (int64_t r = 0; r < dim; ++r) {
      int n = row_entries(states, dim, r, terms, n_terms, dot_bits, dot_dense, e);
      if (n < 0) { err = 1; continue; }
      int m = merge_entries(e, n);
      for (int k = 0; k < m; ++k) {
        col[row_ptr[r] + k] = (int32_t)e[k].col;
        val[row_ptr[r] + k] = e[k].val;
      }
    }
    free(e);
  }
  return err ? -1 : (int64_t)row_ptr[dim];
}

/* The same assembly for a chosen subset of rows (spot checks at sizes where the full
 * matrix is too slow to build on the CPU).  rows[k] in [0, dim); output row k of the
 * mini-CSR holds matrix row rows[k], columns still index the full dimension.
 * Two calls as above: col == NULL counts (row_ptr: int32[n_rows+1]), else fills. */
int64_t orc_build_csr_rows(const uint64_t *states, int64_t dim, const int64_t *rows,
                           int64_t n_rows, const orc_term *terms, int n_terms, int dot_bits,
                           const double *dot_dense, int32_t *row_ptr, int32_t *col, double *val) {
  int cap = n_terms + (dot_bits > 0 ? (1 << dot_bits) : 0) + 1;
  orc_entry *e = (orc_entry *)malloc(sizeof(orc_entry) * (size_t)cap);
  if (!e) return -1;
  int64_t total = 0;
  for (int64_t k = 0; k < n_rows; ++k) {
    int n = row_entries(states, dim, rows[k], terms, n_terms, dot_bits, dot_dense, e);
    if (n < 0) { free(e); return -1; }
    int m = merge_entries(e, n);
    if (!col) {
      row_ptr[k] = (int32_t)total;
    } else {
      for (int q = 0; q < m; ++q) {
        col[row_ptr[k] + q] = (int32_t)e[q].col;
        val[row_ptr[k] + q] = e[q].val;
      }
    }
    total += m;
  }
  if (!col) row_ptr[n_rows] = (int32_t)total;
  free(e);
  return total;
}

/* ---- O3: sparse matrix x block ------------------------------------------ */

/* Y[i,:] = sum_{e in row i} val[e] * X[col[e],:], sequential in stored order
 * (Eq. 8).  X, Y: n x s row-major. */
void orc_spmm(int64_t n, const int32_t *row_ptr, const int32_t *col, const double *val,
              int s, const double *X, double *Y) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double *y = Y + i * s;
    for (int c = 0; c < s; ++c) y[c] = 0.0;
    for (int32_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
      const double *x = X + (int64_t)col[e] * s;
      double v = val[e];
      for (int c = 0; c < s; ++c) y[c] += v * x[c];
    }
  }
}

/* ---- O4: rescaling ------------------------------------------------------- */

/* T <- (T - a X)/b with T = H X on entry: H~ X (Eq. 31). */
void orc_rescale(int64_t n, int s, double a, double b, const double *X, double *T) {
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < n * (int64_t)s; ++k) T[k] = (T[k] - a * X[k]) / b;
}

/* ---- O6: Clenshaw on a block --------------------------------------------- */

/* PAPER.md:420-429 (Eq. 50-51), coefficients c[0..K] already divided by chi:
 *   B1 = B2 = 0
 *   for k = K..1:  (B1, B2) <- (c_k V + 2 H~ B1 - B2, B1)
 *   W = c_0 V + H~ B1 - B2
 * work: 3*n*s doubles.  Returns the number of sparse products (== K). */
int orc_clenshaw(int64_t n, const int32_t *row_ptr, const int32_t *col, const double *val,
                 int s, double a, double b, int K, const double *c, const double *V,
                 double *W, double *work) {
  int64_t len = n * (int64_t)s;
  double *B1 = work, *B2 = work + len, *T = work + 2 * len;
  int products = 0;
  memset(B1, 0, sizeof(double) * (size_t)len);
  memset(B2, 0, sizeof(double) * (size_t)len);
  for (int k = K; k >= 1; --k) {
    if (k == K) {                                      /* b_{K+1} = 0: H~ b_{K+1} = 0 */
      memset(T, 0, sizeof(double) * (size_t)len);
    } else {
      orc_spmm(n, row_ptr, col, val, s, B1, T);        /* T = H B1      */
      orc_rescale(n, s, a, b, B1, T);                  /* T = H~ B1     */
      ++products;
    }
    double ck = c[k];
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < len; ++q) {
      double bnew = ck * V[q] + 2.0 * T[q] - B2[q];
      B2[q] = B1[q];
      B1[q] = bnew;
    }
  }
  if (K >= 1) {                                        /* the K-th product: H~ b_1 */
    orc_spmm(n, row_ptr, col, val, s, B1, T);
    orc_rescale(n, s, a, b, B1, T);
    ++products;
  } else {
    memset(T, 0, sizeof(double) * (size_t)len);        /* K = 0: W = c_0 V */
  }
  {
    double c0 = c[0];
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < len; ++q) W[q] = c0 * V[q] + T[q] - B2[q];
  }
  return products;
}

/* One recurrence step for timing the cpu_baseline on big workloads:
 * B2 <- c_k V + 2 H~ B1 - B2 (caller swaps). T: n*s scratch. */
void orc_clenshaw_step(int64_t n, const int32_t *row_ptr, const int32_t *col, const double *val,
                       int s, double a, double b, double ck, const double *V,
                       const double *B1, double *B2, double *T) {
  int64_t len = n * (int64_t)s;
  orc_spmm(n, row_ptr, col, val, s, B1, T);
  orc_rescale(n, s, a, b, B1, T);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < len; ++q) B2[q] = ck * V[q] + 2.0 * T[q] - B2[q];
}

int orc_num_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}
