// Internal declarations shared by the translation units of libpolfed (sm_100a only).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdarg>
#include <cstdio>
#include <string>

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
};
