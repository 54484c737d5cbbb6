// Packed CSR: the CSR of a Hamiltonian whose off-diagonal entries take at most two distinct values
// (north_star: "exploits constant off-diagonal values (J/2, t)").  Off-diagonal
// entries become one 32-bit word, column | value class << 28; the diagonal is a dense array.  A
// stored entry then costs 4 bytes of stream instead of 12 and ONE quad shuffle in the fused
// kernel instead of three (the kernel is bound by the LSU pipe that shuffles share with the
// gathers, profiles/r03_flip_config4.md).  Built for every handle whose matrix qualifies
// (dimension below 2^28, one or two off-diagonal values: XXZ chains); the kernels are in
// spmm_clenshaw.cu.
#include <cub/cub.cuh>

#include "packed.cuh"

namespace polfed {
namespace {

// Distinct off-diagonal values -> table[0..kPackedMaxVals) (bit patterns; 0 = free slot, so an
// explicit off-diagonal zero is stored as value class of +0.0 = pattern 0 -> remapped below).
__global__ void __launch_bounds__(256) packed_values_kernel(long long n, const int32_t* __restrict__ rp,
                                                            const int32_t* __restrict__ col,
                                                            const double* __restrict__ val,
                                                            unsigned long long* table, int* overflow,
                                                            int32_t* __restrict__ counts) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  int off = 0;
  for (int e = rp[r]; e < rp[r + 1]; ++e) {
    if (col[e] == (int32_t)r) continue;
    ++off;
    // +0.0 has the bit pattern of a free slot: store zeros as -0.0 (same product)
    unsigned long long bits = (unsigned long long)__double_as_longlong(val[e]);
    if (bits == 0ull) bits = 0x8000000000000000ull;
    int c = 0;
    for (; c < kPackedMaxVals; ++c) {
      unsigned long long cur = table[c];
      if (cur == 0ull) cur = atomicCAS(table + c, 0ull, bits);
      if (cur == 0ull || cur == bits) break;
    }
    if (c == kPackedMaxVals) *overflow = 1;
  }
  counts[r] = off;
  if (r == 0) counts[n] = 0;
}

__global__ void __launch_bounds__(256) packed_fill_kernel(long long n, const int32_t* __restrict__ rp,
                                                          const int32_t* __restrict__ col,
                                                          const double* __restrict__ val,
                                                          const unsigned long long* __restrict__ table,
                                                          const int32_t* __restrict__ rp_off,
                                                          uint32_t* __restrict__ pcol,
                                                          double* __restrict__ diag) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  double d = 0.0;
  int at = rp_off[r];
  for (int e = rp[r]; e < rp[r + 1]; ++e) {
    if (col[e] == (int32_t)r) {
      d += val[e];
      continue;
    }
    unsigned long long bits = (unsigned long long)__double_as_longlong(val[e]);
    if (bits == 0ull) bits = 0x8000000000000000ull;
    uint32_t cls = 0;
    while (cls < (uint32_t)kPackedMaxVals - 1 && table[cls] != bits) ++cls;
    pcol[at++] = (uint32_t)col[e] | (cls << 28);
  }
  diag[r] = d;
}

}  // namespace

void destroy_packed_plan(PackedPlan* p) {
  if (!p) return;
  cudaFree(p->d_row_ptr);
  cudaFree(p->d_pcol);
  cudaFree(p->d_diag);
  delete p;
}

// *out stays NULL (and POLFED_OK is returned) when the matrix does not qualify.
int build_packed_plan(const polfed_ham* ham, cudaStream_t st, PackedPlan** out) {
  *out = nullptr;
  const long long n = ham->n;
  if (n < 1 || n >= (1LL << 28) || ham->nnz < 1) return POLFED_OK;
  struct Temp {
    std::vector<void*> p;
    ~Temp() {
      for (void* q : p) cudaFree(q);
    }
  } tmp;
  unsigned long long* d_table = nullptr;
  int* d_flag = nullptr;
  int32_t* d_counts = nullptr;
  POLFED_CUDA(cudaMalloc(&d_table, sizeof(unsigned long long) * kPackedMaxVals));
  tmp.p.push_back(d_table);
  POLFED_CUDA(cudaMalloc(&d_flag, sizeof(int)));
  tmp.p.push_back(d_flag);
  POLFED_CUDA(cudaMalloc(&d_counts, sizeof(int32_t) * (size_t)(n + 1)));
  tmp.p.push_back(d_counts);
  POLFED_CUDA(cudaMemsetAsync(d_table, 0, sizeof(unsigned long long) * kPackedMaxVals, st));
  POLFED_CUDA(cudaMemsetAsync(d_flag, 0, sizeof(int), st));
  const unsigned grid = (unsigned)((n + 255) / 256);
  packed_values_kernel<<<grid, 256, 0, st>>>(n, ham->d_row_ptr, ham->d_col, ham->d_val, d_table, d_flag,
                                             d_counts);
  POLFED_LAUNCH_CHECK("packed_values_kernel");
  int overflow = 0;
  unsigned long long table[kPackedMaxVals];
  POLFED_CUDA(cudaMemcpyAsync(&overflow, d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
  POLFED_CUDA(cudaMemcpyAsync(table, d_table, sizeof table, cudaMemcpyDeviceToHost, st));
  POLFED_CUDA(cudaStreamSynchronize(st));
  if (overflow) return POLFED_OK;  // too many distinct values: plain CSR only

  PackedPlan* p = new (std::nothrow) PackedPlan;
  if (!p) return fail(POLFED_ENOMEM, "packed CSR: host allocation failed");
  struct Guard {
    PackedPlan* p;
    ~Guard() { destroy_packed_plan(p); }
  } guard{p};
  for (int c = 0; c < kPackedMaxVals; ++c) {
    memcpy(&p->vals[c], &table[c], sizeof(double));
    if (table[c]) p->n_vals = c + 1;
  }
  // measured: with one or two values (a register select) the packed kernel wins (config 3:
  // 32.7 -> 26.6 us per step); with three or more (config 5: 6.3 -> 6.7 ms) it loses
  if (p->n_vals == 0 || p->n_vals > 2) return POLFED_OK;
  POLFED_CUDA(cudaMalloc(&p->d_row_ptr, sizeof(int32_t) * (size_t)(n + 1)));
  size_t bytes = 0;
  POLFED_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, bytes, d_counts, p->d_row_ptr, (int)(n + 1), st));
  void* d_cub = nullptr;
  POLFED_CUDA(cudaMalloc(&d_cub, bytes ? bytes : 1));
  tmp.p.push_back(d_cub);
  POLFED_CUDA(cub::DeviceScan::ExclusiveSum(d_cub, bytes, d_counts, p->d_row_ptr, (int)(n + 1), st));
  int32_t total = 0;
  POLFED_CUDA(cudaMemcpyAsync(&total, p->d_row_ptr + n, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  POLFED_CUDA(cudaStreamSynchronize(st));
  p->nnz_off = total;
  POLFED_CUDA(cudaMalloc(&p->d_pcol, sizeof(uint32_t) * (size_t)(total > 0 ? total : 1)));
  POLFED_CUDA(cudaMalloc(&p->d_diag, sizeof(double) * (size_t)n));
  packed_fill_kernel<<<grid, 256, 0, st>>>(n, ham->d_row_ptr, ham->d_col, ham->d_val, d_table,
                                           p->d_row_ptr, p->d_pcol, p->d_diag);
  POLFED_LAUNCH_CHECK("packed_fill_kernel");
  POLFED_CUDA(cudaStreamSynchronize(st));
  guard.p = nullptr;
  *out = p;
  return POLFED_OK;
}

}  // namespace polfed
