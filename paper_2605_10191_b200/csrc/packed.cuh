// Packed CSR (packed.cu): off-diagonal entries as column | value class << 28, dense diagonal.
#pragma once

#include <cstring>

#include "common.cuh"

namespace polfed {

constexpr int kPackedMaxVals = 15;  // distinct off-diagonal values (4-bit class, 15 = overflow guard)

struct PackedVals {  // passed to the kernel by value: an indexed constant-bank read per entry
  double v[16];
};

struct PackedPlan {
  int32_t* d_row_ptr = nullptr;  // [n+1] into d_pcol
  uint32_t* d_pcol = nullptr;    // [nnz_off]
  double* d_diag = nullptr;      // [n]
  long long nnz_off = 0;
  int n_vals = 0;                // distinct off-diagonal values (table entries in use)
  double vals[16] = {};
};

int build_packed_plan(const polfed_ham* ham, cudaStream_t st, PackedPlan** out);
void destroy_packed_plan(PackedPlan* plan);

}  // namespace polfed
