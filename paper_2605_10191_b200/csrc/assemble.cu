// Device-side CSR assembly of a many-body Hamiltonian from a term list.
// Models: XXZ chain Eq. (54); quantum sun Eq. (67) PAPER.md:939-946;
// spinless fermions of BASELINE.json config 5 (R15).  Conventions R12-R14.
//
// One thread builds one row in registers/local memory: it walks the term list, ranks every
// state the row connects to, sorts the (few dozen) entries by column and merges duplicates.
// Pass 1 counts, a device scan turns counts into row_ptr, pass 2 writes col/val.
#include <cub/device/device_reduce.cuh>
#include <cub/device/device_scan.cuh>
#include <thrust/iterator/transform_iterator.h>

#include <new>
#include <vector>

#include "combinadic.cuh"

namespace polfed {
namespace {

constexpr int kMaxRowEntries = 128;

struct ToI64 {
  __host__ __device__ long long operator()(int v) const { return (long long)v; }
};

struct RowBuilder {
  int32_t cols[kMaxRowEntries];
  double vals[kMaxRowEntries];
  int n;
  bool bad;

  __device__ void push(int64_t c, double v) {
    if (c < 0) {
      bad = true;
      return;
    }
    cols[n] = (int32_t)c;
    vals[n] = v;
    ++n;
  }
};

// Entries of the row of state x before sorting; entry 0 is the diagonal.
__device__ void generate_row(RowBuilder& rb, int64_t row, uint64_t x, int n_sites, int n_up,
                             const DevTerm* __restrict__ terms, int n_terms, int dot_bits,
                             const double* __restrict__ dot) {
  rb.n = 0;
  rb.bad = false;
  rb.push(row, 0.0);
  double diag = 0.0;
  if (dot_bits > 0) {
    const uint64_t dd = 1ull << dot_bits, mask = dd - 1, d = x & mask;
    diag = dot[d * dd + d];
    for (uint64_t d2 = 0; d2 < dd; ++d2)
      if (d2 != d) rb.push(rank_state((x & ~mask) | d2, n_sites, n_up), dot[d * dd + d2]);
  }
  for (int t = 0; t < n_terms; ++t) {
    const DevTerm tm = terms[t];
    const int bi = (int)((x >> tm.i) & 1ull), bj = (int)((x >> tm.j) & 1ull);
    switch (tm.kind) {
      case POLFED_TERM_ZZ:
        diag = __dadd_rn(diag, __dmul_rn(tm.amp, (bi == bj) ? 0.25 : -0.25));
        break;
      case POLFED_TERM_Z:
        diag = __dadd_rn(diag, __dmul_rn(tm.amp, bi ? 0.5 : -0.5));
        break;
      case POLFED_TERM_NN:
        if (bi & bj) diag = __dadd_rn(diag, tm.amp);
        break;
      case POLFED_TERM_N:
        if (bi) diag = __dadd_rn(diag, tm.amp);
        break;
      case POLFED_TERM_EXCH:
      case POLFED_TERM_HOPJW:
        if (bi != bj) {
          const uint64_t y = x ^ (1ull << tm.i) ^ (1ull << tm.j);
          double v = tm.amp;
          if (tm.kind == POLFED_TERM_HOPJW) {
            const int lo = min(tm.i, tm.j), hi = max(tm.i, tm.j);
            const uint64_t between = ((1ull << hi) - 1ull) & ~((2ull << lo) - 1ull);
            if (__popcll(x & between) & 1) v = -v;
          }
          rb.push(rank_state(y, n_sites, n_up), v);
        }
        break;
      case POLFED_TERM_XX:
        rb.push(rank_state(x ^ (1ull << tm.i) ^ (1ull << tm.j), n_sites, n_up), tm.amp);
        break;
      default:
        rb.bad = true;
    }
  }
  rb.vals[0] = diag;
}

// Stable insertion sort by column, then sum runs of equal columns left to right.
__device__ int sort_and_merge(RowBuilder& rb) {
  for (int a = 1; a < rb.n; ++a) {
    const int32_t kc = rb.cols[a];
    const double kv = rb.vals[a];
    int b = a - 1;
    while (b >= 0 && rb.cols[b] > kc) {
      rb.cols[b + 1] = rb.cols[b];
      rb.vals[b + 1] = rb.vals[b];
      --b;
    }
    rb.cols[b + 1] = kc;
    rb.vals[b + 1] = kv;
  }
  int m = 0;
  for (int k = 0; k < rb.n; ++k) {
    if (m > 0 && rb.cols[m - 1] == rb.cols[k]) {
      rb.vals[m - 1] = __dadd_rn(rb.vals[m - 1], rb.vals[k]);
    } else {
      rb.cols[m] = rb.cols[k];
      rb.vals[m] = rb.vals[k];
      ++m;
    }
  }
  return m;
}

template <bool FILL>
__global__ void __launch_bounds__(128)
assemble_kernel(int64_t dim, int n_sites, int n_up, const uint64_t* __restrict__ states,
                const DevTerm* __restrict__ terms, int n_terms, int dot_bits,
                const double* __restrict__ dot, int32_t* __restrict__ counts,
                const int32_t* __restrict__ row_ptr, int32_t* __restrict__ col,
                double* __restrict__ val, int* __restrict__ error_flag) {
  const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= dim) return;
  const uint64_t x = states ? states[row] : (uint64_t)row;
  RowBuilder rb;
  generate_row(rb, row, x, n_sites, n_up, terms, n_terms, dot_bits, dot);
  if (rb.bad) {
    *error_flag = 1;
    if (!FILL) counts[row] = 0;
    return;
  }
  const int m = sort_and_merge(rb);
  if (!FILL) {
    counts[row] = m;
  } else {
    const int32_t at = row_ptr[row];
    for (int k = 0; k < m; ++k) {
      col[at + k] = rb.cols[k];
      val[at + k] = rb.vals[k];
    }
  }
}

struct Scratch {  // frees device temporaries on every exit path
  void* p[8] = {nullptr};
  int n = 0;
  ~Scratch() {
    for (int k = 0; k < n; ++k) cudaFree(p[k]);
  }
  template <class T>
  cudaError_t alloc(T** out, size_t bytes) {
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(out), bytes ? bytes : 1);
    if (e == cudaSuccess) p[n++] = *out;
    return e;
  }
};

}  // namespace

// CSR of the term list over the basis (the work of polfed_build_hamiltonian; also used for the
// diagonal + cross-cut parts of the tiled format, tiled_plan.cu).  Arrays are cudaMalloc'ed;
// the caller owns them.  Synchronises `st`.
int assemble_csr(const polfed_basis* basis, const std::vector<DevTerm>& terms, int dot_bits,
                 const double* h_dot, cudaStream_t st, int32_t** out_row_ptr, int32_t** out_col,
                 double** out_val, long long* out_nnz) {
  const int n_terms = (int)terms.size();
  int rc = ensure_binomials();
  if (rc) return rc;
  const int64_t dim = basis->dim;

  Scratch tmp;
  DevTerm* d_terms = nullptr;
  double* d_dot = nullptr;
  int32_t* d_counts = nullptr;
  int* d_flag = nullptr;
  long long* d_total = nullptr;
  POLFED_CUDA(tmp.alloc(&d_terms, sizeof(DevTerm) * terms.size()));
  POLFED_CUDA(tmp.alloc(&d_flag, sizeof(int)));
  POLFED_CUDA(tmp.alloc(&d_total, sizeof(long long)));
  POLFED_CUDA(tmp.alloc(&d_counts, sizeof(int32_t) * (size_t)(dim + 1)));
  if (n_terms)
    POLFED_CUDA(cudaMemcpyAsync(d_terms, terms.data(), sizeof(DevTerm) * terms.size(),
                                cudaMemcpyHostToDevice, st));
  if (dot_bits) {
    const size_t dd = (size_t)1 << dot_bits;
    POLFED_CUDA(tmp.alloc(&d_dot, sizeof(double) * dd * dd));
    POLFED_CUDA(cudaMemcpyAsync(d_dot, h_dot, sizeof(double) * dd * dd, cudaMemcpyHostToDevice, st));
  }
  POLFED_CUDA(cudaMemsetAsync(d_flag, 0, sizeof(int), st));
  POLFED_CUDA(cudaMemsetAsync(d_counts, 0, sizeof(int32_t) * (size_t)(dim + 1), st));

  int32_t* d_row_ptr = nullptr;
  POLFED_CUDA(cudaMalloc(&d_row_ptr, sizeof(int32_t) * (size_t)(dim + 1)));
  struct Guard {  // releases the result arrays unless ownership moved to the caller
    int32_t* a = nullptr;
    int32_t* b = nullptr;
    double* c = nullptr;
    bool armed = true;
    ~Guard() {
      if (armed) { cudaFree(a); cudaFree(b); cudaFree(c); }
    }
  } guard;
  guard.a = d_row_ptr;

  const unsigned grid = (unsigned)((dim + 127) / 128);
  if (dim > 0) {
    assemble_kernel<false><<<grid, 128, 0, st>>>(dim, basis->n_sites, basis->n_up,
                                                 basis->n_up < 0 ? nullptr : basis->d_states,
                                                 d_terms, n_terms, dot_bits, d_dot, d_counts,
                                                 nullptr, nullptr, nullptr, d_flag);
    POLFED_LAUNCH_CHECK("assemble_kernel<count>");
  }
  // total in 64 bits (overflow check), row_ptr by exclusive scan over dim+1 counts
  auto wide = thrust::make_transform_iterator(d_counts, ToI64());
  size_t bytes_a = 0, bytes_b = 0;
  POLFED_CUDA(cub::DeviceReduce::Sum(nullptr, bytes_a, wide, d_total, (int)(dim + 1), st));
  POLFED_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, bytes_b, d_counts, d_row_ptr, (int)(dim + 1), st));
  void* d_cub = nullptr;
  POLFED_CUDA(tmp.alloc(&d_cub, bytes_a > bytes_b ? bytes_a : bytes_b));
  POLFED_CUDA(cub::DeviceReduce::Sum(d_cub, bytes_a, wide, d_total, (int)(dim + 1), st));
  POLFED_CUDA(cub::DeviceScan::ExclusiveSum(d_cub, bytes_b, d_counts, d_row_ptr, (int)(dim + 1), st));
  long long total = 0;
  int flag = 0;
  POLFED_CUDA(cudaMemcpyAsync(&total, d_total, sizeof total, cudaMemcpyDeviceToHost, st));
  POLFED_CUDA(cudaMemcpyAsync(&flag, d_flag, sizeof flag, cudaMemcpyDeviceToHost, st));
  POLFED_CUDA(cudaStreamSynchronize(st));
  if (flag) return fail(POLFED_EINVAL, "polfed_build_hamiltonian: a term leaves the basis");
  if (total >= (1ll << 31))
    return fail(POLFED_ERANGE, "polfed_build_hamiltonian: nnz=%lld does not fit int32", total);

  int32_t* d_col = nullptr;
  double* d_val = nullptr;
  POLFED_CUDA(cudaMalloc(&d_col, sizeof(int32_t) * (size_t)(total ? total : 1)));
  guard.b = d_col;
  POLFED_CUDA(cudaMalloc(&d_val, sizeof(double) * (size_t)(total ? total : 1)));
  guard.c = d_val;
  if (dim > 0) {
    assemble_kernel<true><<<grid, 128, 0, st>>>(dim, basis->n_sites, basis->n_up,
                                                basis->n_up < 0 ? nullptr : basis->d_states,
                                                d_terms, n_terms, dot_bits, d_dot, nullptr,
                                                d_row_ptr, d_col, d_val, d_flag);
    POLFED_LAUNCH_CHECK("assemble_kernel<fill>");
  }
  POLFED_CUDA(cudaStreamSynchronize(st));
  guard.armed = false;
  *out_row_ptr = d_row_ptr;
  *out_col = d_col;
  *out_val = d_val;
  *out_nnz = total;
  return POLFED_OK;
}

}  // namespace polfed

using polfed::fail;

extern "C" int polfed_build_hamiltonian(const polfed_basis* basis, const polfed_term* h_terms,
                                        int n_terms, const polfed_dense_block* dot, int format,
                                        void* stream, polfed_ham** out) {
  using namespace polfed;
  if (!out) return fail(POLFED_EINVAL, "polfed_build_hamiltonian: out is NULL");
  *out = nullptr;
  if (!basis) return fail(POLFED_EINVAL, "polfed_build_hamiltonian: basis is NULL");
  if (format != POLFED_FORMAT_CSR && (format < POLFED_FORMAT_TILED || format > POLFED_FORMAT_SECTOR))
    return fail(POLFED_EINVAL, "polfed_build_hamiltonian: format must be POLFED_FORMAT_CSR, "
                               "_TILED, _FLIP or _SECTOR");
  if (n_terms < 0 || (n_terms > 0 && !h_terms))
    return fail(POLFED_EINVAL, "polfed_build_hamiltonian: bad term list");
  int dot_bits = 0;
  if (dot && dot->n_bits > 0) {
    dot_bits = dot->n_bits;
    if (basis->n_up >= 0)
      return fail(POLFED_EINVAL, "polfed_build_hamiltonian: a dense block needs the full space");
    if (dot_bits > 6 || dot_bits > basis->n_sites || !dot->h_dense)
      return fail(POLFED_EINVAL, "polfed_build_hamiltonian: bad dense block");
  }
  std::vector<DevTerm> terms((size_t)n_terms);
  int n_offdiag = dot_bits ? (1 << dot_bits) - 1 : 0;
  for (int t = 0; t < n_terms; ++t) {
    const polfed_term& s = h_terms[t];
    if (s.kind < POLFED_TERM_ZZ || s.kind > POLFED_TERM_XX)
      return fail(POLFED_EINVAL, "polfed_build_hamiltonian: term %d has unknown kind %d", t, s.kind);
    const bool one_site = (s.kind == POLFED_TERM_Z || s.kind == POLFED_TERM_N);
    const int j = one_site ? s.i : s.j;
    if (s.i < 0 || s.i >= basis->n_sites || j < 0 || j >= basis->n_sites)
      return fail(POLFED_EINVAL, "polfed_build_hamiltonian: term %d acts outside the lattice", t);
    if (s.kind >= POLFED_TERM_EXCH) {
      if (s.i == j)
        return fail(POLFED_EINVAL, "polfed_build_hamiltonian: term %d needs two distinct sites", t);
      ++n_offdiag;
    }
    terms[t] = DevTerm{s.i, j, s.kind, 0, s.amp};
  }
  if (n_offdiag + 1 > kMaxRowEntries)
    return fail(POLFED_EINVAL, "polfed_build_hamiltonian: more than %d entries per row",
                kMaxRowEntries);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int32_t* d_row_ptr = nullptr;
  int32_t* d_col = nullptr;
  double* d_val = nullptr;
  long long total = 0;
  int rc = assemble_csr(basis, terms, dot_bits, dot_bits ? dot->h_dense : nullptr, st, &d_row_ptr,
                        &d_col, &d_val, &total);
  if (rc) return rc;
  polfed_ham* h = nullptr;
  // the tiled, sector and flip plans carry their own copy of the matrix: their handles keep the
  // CSR for the steps those plans do not take (s below the plan's sizes) and skip the packed copy
  rc = polfed_ham_from_csr_ex(basis->dim, total, d_row_ptr, d_col, d_val,
                              format == POLFED_FORMAT_CSR ? 0u : (unsigned)POLFED_HAM_NO_SNAPSHOT, stream, &h);
  if (rc) {
    cudaFree(d_row_ptr); cudaFree(d_col); cudaFree(d_val);
    return rc;
  }
  h->owns = true;
  if (format == POLFED_FORMAT_TILED || format == POLFED_FORMAT_SECTOR) {
    rc = build_tiled_plan(basis, terms, format == POLFED_FORMAT_SECTOR, st, &h->tiled);
    if (rc) {
      polfed_ham_destroy(h);
      return rc;
    }
  }
  if (format == POLFED_FORMAT_FLIP) {
    rc = build_flip_plan(basis, terms, dot_bits, dot_bits ? dot->h_dense : nullptr, h, st, &h->flip);
    if (rc) {
      polfed_ham_destroy(h);
      return rc;
    }
  }
  *out = h;
  return POLFED_OK;
}
