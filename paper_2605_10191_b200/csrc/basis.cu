// Device-side enumeration and ranking of the fixed-popcount basis (combinatorial number
// system).  The paper uses U(1) sectors without saying how they are
// indexed; reading R12: ascending integers, rank(x) = sum_j C(p_j, j).
#include <new>

#include "combinadic.cuh"

namespace polfed {
namespace {

__global__ void __launch_bounds__(256) enumerate_kernel(int64_t dim, int n_sites, int n_up,
                                                        uint64_t* __restrict__ states) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= dim) return;
  states[r] = n_up < 0 ? (uint64_t)r : unrank_state((uint64_t)r, n_sites, n_up);
}

__global__ void __launch_bounds__(256) rank_kernel(int64_t n, int n_sites, int n_up,
                                                   const uint64_t* __restrict__ states,
                                                   int64_t* __restrict__ out) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  out[t] = rank_state(states[t], n_sites, n_up);
}

int materialise(polfed_basis* b, cudaStream_t st) {
  if (b->d_states || b->dim == 0) return POLFED_OK;
  POLFED_CUDA(cudaMalloc(&b->d_states, (size_t)b->dim * sizeof(uint64_t)));
  const unsigned grid = (unsigned)((b->dim + 255) / 256);
  enumerate_kernel<<<grid, 256, 0, st>>>(b->dim, b->n_sites, b->n_up, b->d_states);
  POLFED_LAUNCH_CHECK("enumerate_kernel");
  POLFED_CUDA(cudaStreamSynchronize(st));
  return POLFED_OK;
}

}  // namespace
}  // namespace polfed

using polfed::fail;

extern "C" {

int polfed_build_basis(int n_sites, int n_up, void* stream, polfed_basis** out) {
  if (!out) return fail(POLFED_EINVAL, "polfed_build_basis: out is NULL");
  *out = nullptr;
  if (n_sites < 1 || n_sites > polfed::kMaxSites)
    return fail(POLFED_EINVAL, "polfed_build_basis: n_sites=%d not in [1,%d]", n_sites,
                polfed::kMaxSites);
  if (n_up > n_sites)
    return fail(POLFED_EINVAL, "polfed_build_basis: n_up=%d > n_sites=%d", n_up, n_sites);
  int rc = polfed::ensure_binomials();
  if (rc) return rc;
  const uint64_t dim = n_up < 0 ? (n_sites >= 31 ? UINT64_MAX : (1ull << n_sites))
                                : polfed::host_binom(n_sites, n_up);
  if (dim >= (1ull << 31))
    return fail(POLFED_ERANGE, "polfed_build_basis: dimension does not fit int32 indices");
  polfed_basis* b = new (std::nothrow) polfed_basis;
  if (!b) return fail(POLFED_ENOMEM, "polfed_build_basis: host allocation failed");
  b->n_sites = n_sites;
  b->n_up = n_up < 0 ? -1 : n_up;
  b->dim = (int64_t)dim;
  if (n_up >= 0) {
    rc = polfed::materialise(b, static_cast<cudaStream_t>(stream));
    if (rc) {
      cudaFree(b->d_states);
      delete b;
      return rc;
    }
  }
  *out = b;
  return POLFED_OK;
}

int polfed_basis_destroy(polfed_basis* basis) {
  if (!basis) return POLFED_OK;
  cudaFree(basis->d_states);
  delete basis;
  return POLFED_OK;
}

int polfed_basis_dim(const polfed_basis* basis, int64_t* dim) {
  if (!basis || !dim) return fail(POLFED_EINVAL, "polfed_basis_dim: NULL argument");
  *dim = basis->dim;
  return POLFED_OK;
}

int polfed_basis_states(const polfed_basis* basis, const uint64_t** d_states) {
  if (!basis || !d_states) return fail(POLFED_EINVAL, "polfed_basis_states: NULL argument");
  int rc = polfed::materialise(const_cast<polfed_basis*>(basis), nullptr);
  if (rc) return rc;
  *d_states = basis->d_states;
  return POLFED_OK;
}

int polfed_basis_rank(const polfed_basis* basis, const uint64_t* d_states, int64_t n,
                      int64_t* d_rank, void* stream) {
  if (!basis) return fail(POLFED_EINVAL, "polfed_basis_rank: basis is NULL");
  if (n < 0) return fail(POLFED_EINVAL, "polfed_basis_rank: n < 0");
  if (n == 0) return POLFED_OK;
  if (!d_states || !d_rank) return fail(POLFED_EINVAL, "polfed_basis_rank: NULL array");
  const unsigned grid = (unsigned)((n + 255) / 256);
  polfed::rank_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(
      n, basis->n_sites, basis->n_up, d_states, d_rank);
  POLFED_LAUNCH_CHECK("rank_kernel");
  return POLFED_OK;
}

}  // extern "C"
