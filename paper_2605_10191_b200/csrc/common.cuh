// Internal declarations shared by the translation units of libpolfed (sm_100a only).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <string>
#include <vector>

#include "polfed.h"

namespace polfed {

// Thread-local error text behind polfed_last_error().
void set_error(const char* fmt, ...);
int fail(int code, const char* fmt, ...);

#define POLFED_CUDA(expr)                                                                  \
  do {                                                                                     \
    cudaError_t err__ = (expr);                                                            \
    if (err__ != cudaSuccess)                                                              \
      return ::polfed::fail(err__ == cudaErrorMemoryAllocation ? POLFED_ENOMEM : POLFED_ECUDA, \
                            "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(err__),     \
                            __FILE__, __LINE__);                                           \
  } while (0)

#define POLFED_LAUNCH_CHECK(what)                                                          \
  do {                                                                                     \
    cudaError_t err__ = cudaGetLastError();                                                \
    if (err__ != cudaSuccess)                                                              \
      return ::polfed::fail(POLFED_ECUDA, "launch of %s failed: %s", what,                 \
                            cudaGetErrorString(err__));                                    \
  } while (0)

constexpr int kMaxSites = 62;
constexpr int kBinomDim = 64;  // table holds C(n, k) for 0 <= n, k < 64

inline bool valid_block_size(int s) {
  return s == 1 || s == 2 || s == 4 || s == 8 || s == 16 || s == 32;
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// One term of the Hamiltonian as the device kernels read it (polfed_term with j filled in).
struct DevTerm {
  int32_t i, j, kind, pad;
  double amp;
};

struct TiledPlan;  // tiled.cuh
struct FlipPlan;   // flip.cuh
struct PackedPlan; // packed.cuh

// assemble.cu: CSR of a term list over a basis; arrays cudaMalloc'ed, owned by the caller.
int assemble_csr(const polfed_basis* basis, const std::vector<DevTerm>& terms, int dot_bits,
                 const double* h_dot, cudaStream_t st, int32_t** out_row_ptr, int32_t** out_col,
                 double** out_val, long long* out_nnz);
// tiled_plan.cu / tiled_sweep.cu: the tiled (matrix-free inside a tile) format, see tiled.cuh.
int build_tiled_plan(const polfed_basis* basis, const std::vector<DevTerm>& terms, bool sector,
                     cudaStream_t st, TiledPlan** out);
void destroy_tiled_plan(TiledPlan* plan);
bool tiled_supports(const polfed_ham* ham, int s);
size_t tiled_workspace_bytes(const polfed_ham* ham, int s);
int tiled_filter_apply(const polfed_ham* ham, double a, double b, int K, const double* h_coeffs,
                       int s, const double* d_V, double* d_W, void* d_work, cudaStream_t st);

// flip.cu: the flip (matrix-free, full-space) format, see flip.cuh.
int build_flip_plan(const polfed_basis* basis, const std::vector<DevTerm>& terms, int dot_bits,
                    const double* h_dot, const polfed_ham* ham, cudaStream_t st, FlipPlan** out);
void destroy_flip_plan(FlipPlan* plan);
bool flip_supports(const polfed_ham* ham, int s);
int flip_step(const polfed_ham* ham, int s, double p, double q, double r, double c, const double* X,
              const double* Z, const double* V, double* Y, cudaStream_t st);

// small_filter.cu: the whole recurrence in one persistent kernel (n * s <= 262144).
// small_filter_apply returns POLFED_ERANGE when it cannot take the matrix (caller: single launches).
bool small_filter_supports(const polfed_ham* ham, int s);
int csr_max_row_len(long long n, const int32_t* d_row_ptr, int* out, cudaStream_t st);
int small_filter_apply(const polfed_ham* ham, double a, double b, int K, const double* h_coeffs,
                       int s, const double* d_V, double* d_W, double* cur, double* old,
                       cudaStream_t st);

// api.cu: stream-ordered scratch from the library's own memory pool of the current device (one per
// device, created on first use, never trimmed: after the first call of a given size an
// allocation is a free-list hit, not a mapping).  Free with cudaFreeAsync.
cudaError_t scratch_alloc(void** p, size_t bytes, cudaStream_t st);

// spmm_clenshaw.cu: the fused step without argument validation (flip handles: flip_step).
int dispatch_step(const polfed_ham* ham, int s, double p, double q, double r, double c,
                  const double* X, const double* Z, const double* V, double* Y, cudaStream_t st);

// tallskinny.cu (see there).  d_C is zeroed by ts_gram before accumulation.
int ts_gram(int s, long long n, const double* Q, int n_panels, size_t stride, const double* B,
            double* d_C, int sm_count, cudaStream_t st);
int ts_gram_variant(int s, long long n, const double* Q, int n_panels, size_t stride, const double* B,
                    double* d_C, int sm_count, int variant, cudaStream_t st);
int ts_update(int s, long long n, const double* Q, int n_panels, size_t stride, const double* d_C,
              double alpha, double beta, double* B, cudaStream_t st);
int ts_residual_norms(int s, long long n, const double* A, const double* B, const double* d_e,
                      double* d_out, int sm_count, cudaStream_t st);
int ts_gather_columns(long long n, const double* src, int src_ld, const int* d_cols, int n_cols,
                      double* dst, int dst_ld, int dst_col0, int sm_count, cudaStream_t st);
int csr_moments(const polfed_ham* ham, double* d_out2, cudaStream_t st);

}  // namespace polfed

struct polfed_basis {
  int n_sites = 0;
  int n_up = -1;         // < 0: full space
  int64_t dim = 0;
  uint64_t* d_states = nullptr;  // may be null for the full space until requested
};

struct polfed_ham {
  int64_t n = 0;
  int64_t nnz = 0;
  const int32_t* d_row_ptr = nullptr;
  const int32_t* d_col = nullptr;
  const double* d_val = nullptr;
  bool owns = false;  // arrays allocated by polfed_build_hamiltonian
  int sm_count = 148;
  int max_row_len = 0;   // longest CSR row (small_filter.cu)
  polfed::TiledPlan* tiled = nullptr;  // POLFED_FORMAT_TILED only (owned)
  polfed::FlipPlan* flip = nullptr;    // POLFED_FORMAT_FLIP only (owned)
  polfed::PackedPlan* packed = nullptr;  // every handle whose matrix qualifies (owned)
};
