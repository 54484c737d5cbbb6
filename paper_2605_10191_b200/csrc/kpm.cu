// Kernel polynomial method: Chebyshev moments of the density of states on the device and the
// Jackson-damped series on the host (Eq. 35-39).  The
// Chebyshev recurrence T_{n+1} = 2 H~ T_n - T_{n-1} (Eq. 28-30) is the fused step of the filter
// with c = 0, so the moments cost one sparse product + one block dot product each.
#include <cmath>
#include <vector>

#include "common.cuh"

namespace polfed {
namespace {

constexpr int kDotThreads = 256;

// partial[b] = sum over this block's grid-stride share of A[i] * B[i]   (fixed order)
__global__ void __launch_bounds__(kDotThreads) block_dot_partial_kernel(long long len,
                                                                       const double* __restrict__ A,
                                                                       const double* __restrict__ B,
                                                                       double* __restrict__ partial) {
  __shared__ double warp_sum[kDotThreads / 32];
  double acc = 0.0;
  for (long long i = (long long)blockIdx.x * kDotThreads + threadIdx.x; i < len;
       i += (long long)gridDim.x * kDotThreads)
    acc = fma(A[i], B[i], acc);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < kDotThreads / 32; ++w) t += warp_sum[w];
    partial[blockIdx.x] = t;
  }
}

// out[0] = scale * sum of partial[0..count)   (one thread: count is a few hundred)
__global__ void block_dot_final_kernel(int count, const double* __restrict__ partial, double scale,
                                       double* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double t = 0.0;
  for (int i = 0; i < count; ++i) t += partial[i];
  out[0] = scale * t;
}

}  // namespace
}  // namespace polfed

using polfed::fail;

extern "C" {

size_t polfed_kpm_workspace_bytes(int64_t n, int s, int n_moments) {
  if (n < 0 || s <= 0 || n_moments < 0) return 0;
  // two Chebyshev blocks, the per-block partial sums, the moments
  return ((size_t)2 * (size_t)n * s + 4096 + (size_t)n_moments + 2) * sizeof(double);
}

int polfed_kpm_moments(const polfed_ham* ham, double a, double b, int n_moments, int s,
                       const double* d_R, void* d_work, double* h_moments, void* stream) {
  if (!ham || !h_moments) return fail(POLFED_EINVAL, "polfed_kpm_moments: NULL argument");
  if (n_moments < 1) return fail(POLFED_EINVAL, "polfed_kpm_moments: n_moments must be >= 1");
  if (!polfed::valid_block_size(s))
    return fail(POLFED_EINVAL, "polfed_kpm_moments: s must be 1, 2, 4, 8, 16 or 32");
  if (!(b > 0.0) || !std::isfinite(a) || !std::isfinite(b))
    return fail(POLFED_ERANGE, "polfed_kpm_moments: need finite a and b > 0");
  const long long n = ham->n;
  if (n == 0) {
    for (int m = 0; m < n_moments; ++m) h_moments[m] = 0.0;
    return POLFED_OK;
  }
  if (!d_R || !d_work) return fail(POLFED_EINVAL, "polfed_kpm_moments: NULL device buffer");
  if (!polfed::aligned16(d_R) || !polfed::aligned16(d_work))
    return fail(POLFED_EINVAL, "polfed_kpm_moments: buffers must be 16-byte aligned");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t len = (size_t)n * s;
  double* T[2] = {static_cast<double*>(d_work), static_cast<double*>(d_work) + len};
  double* partial = T[1] + len;
  double* d_mu = partial + 4096;
  int blocks = ham->sm_count * 4;
  if (blocks > 4096) blocks = 4096;
  const long long want = (long long)((len + polfed::kDotThreads - 1) / polfed::kDotThreads);
  if (blocks > want) blocks = (int)want;
  const double inv_r = 1.0 / s;

  auto dot = [&](const double* X, int m) -> int {
    polfed::block_dot_partial_kernel<<<blocks, polfed::kDotThreads, 0, st>>>((long long)len, d_R, X,
                                                                             partial);
    POLFED_LAUNCH_CHECK("block_dot_partial_kernel");
    polfed::block_dot_final_kernel<<<1, 32, 0, st>>>(blocks, partial, inv_r, d_mu + m);
    POLFED_LAUNCH_CHECK("block_dot_final_kernel");
    return POLFED_OK;
  };

  int rc = dot(d_R, 0);  // mu_0 = <r|r> averaged: the dimension for unit-variance entries
  if (rc) return rc;
  const double* Tm = d_R;   // T_{n-2}|r>
  const double* Tc = d_R;   // T_{n-1}|r>
  for (int m = 1; m < n_moments; ++m) {
    double* Tn;
    if (m == 1) {  // T_1 = H~ T_0
      Tn = T[0];
      rc = polfed::dispatch_step(ham, s, 1.0 / b, -a / b, 0.0, 0.0, Tc, nullptr, nullptr, Tn, st);
    } else {       // T_n = 2 H~ T_{n-1} - T_{n-2}; written over T_{n-2} except when that is d_R
      Tn = (Tm == d_R) ? T[1] : const_cast<double*>(Tm);
      rc = polfed::dispatch_step(ham, s, 2.0 / b, -2.0 * a / b, -1.0, 0.0, Tc, Tm, nullptr, Tn, st);
    }
    if (rc) return rc;
    rc = dot(Tn, m);
    if (rc) return rc;
    Tm = Tc;
    Tc = Tn;
  }
  POLFED_CUDA(cudaMemcpyAsync(h_moments, d_mu, sizeof(double) * n_moments, cudaMemcpyDeviceToHost,
                              st));
  POLFED_CUDA(cudaStreamSynchronize(st));
  return POLFED_OK;
}

int polfed_kpm_dos(const double* h_moments, int n_moments, const double* e_rescaled, int n_points,
                   double* rho) {
  if (!h_moments || n_moments < 1 || n_points < 0 || (n_points > 0 && (!e_rescaled || !rho)))
    return fail(POLFED_EINVAL, "polfed_kpm_dos: bad argument");
  const int N = n_moments;
  std::vector<double> w(N);
  const double q = M_PI / (N + 1);
  for (int m = 0; m < N; ++m) {  // Jackson kernel, Eq. (39)
    const double g = ((N - m + 1) * std::cos(q * m) + std::sin(q * m) / std::tan(q)) / (N + 1);
    w[m] = h_moments[m] * g;
  }
  for (int p = 0; p < n_points; ++p) {
    const double e = e_rescaled[p];
    if (!(e > -1.0 && e < 1.0))
      return fail(POLFED_ERANGE, "polfed_kpm_dos: rescaled energy %g outside (-1, 1)", e);
    const double th = std::acos(e);
    double series = w[0];
    for (int m = 1; m < N; ++m) series += 2.0 * w[m] * std::cos(m * th);
    rho[p] = series / (M_PI * std::sqrt(1.0 - e * e));  // Eq. (36)
  }
  return POLFED_OK;
}

}  // extern "C"
