// SELL-C-sigma (north_star: "CSR or SELL-C-sigma"; SURVEY 8(b) `format`): rows are sorted by
// falling length inside windows of sigma rows, cut into slices of C = 8 rows, and every slice is
// stored column-major and padded to its longest row.  With four lanes per row a warp owns one
// slice: entry j of the eight rows is one contiguous 32-byte (columns) / 64-byte (values) segment,
// so the lanes read their row's entry directly -- no shuffle broadcast as in the CSR kernel, whose
// three quad shuffles per entry cost more LSU cycles than the gather itself
// (profiles/r01_flip_config4.md).
#pragma once

#include "common.cuh"

namespace polfed {

constexpr int kSellC = 8;          // rows per slice = rows per warp
constexpr int kSellSigma = 128;    // sorting window (a multiple of kSellC)

struct SellPlan {
  long long n_slices = 0;
  long long padded = 0;              // stored entries including padding
  int32_t* d_perm = nullptr;         // [n_slices * C] row of a position, -1 past the end
  int32_t* d_len = nullptr;          // [n_slices * C] entries of that row
  long long* d_slice_ptr = nullptr;  // [n_slices + 1] first entry of a slice
  int32_t* d_col = nullptr;          // [padded], entry j of slice i, lane r: slice_ptr[i] + j*C + r
  double* d_val = nullptr;
};

}  // namespace polfed
