// Spectral bounds (scalar Lanczos) and the POLFED eigen-solver driver: block Lanczos on P(H~)
// with full reorthogonalisation, CholeskyQR2, periodic Rayleigh-Ritz.
// PAPER.md:86-182 (Sec. 2.1-2.2), 364-382 (Sec. 4.3), 458-469 (Sec. 4.6).  The small dense
// eigenproblems (H_L and the H-projection) are library calls (cuSOLVER syevd); everything that
// touches an n-long vector runs in this library's kernels.
#include <cusolverDn.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <vector>

#include "common.cuh"

namespace polfed {
namespace {

struct DeviceBuf {
  void* p = nullptr;
  ~DeviceBuf() { cudaFree(p); }
  cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 1); }
  double* f64() const { return static_cast<double*>(p); }
};

double now_seconds() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

// ---- small dense helpers on the host (row-major s x s, s <= 32) --------------------------------

// G = R^T R with R upper triangular.  false: G is not numerically positive definite.
bool cholesky_upper(int s, const double* G, double* R) {
  double gmax = 0.0;
  for (int i = 0; i < s; ++i) gmax = std::max(gmax, G[i * s + i]);
  std::fill(R, R + s * s, 0.0);
  for (int i = 0; i < s; ++i) {
    double d = G[i * s + i];
    for (int k = 0; k < i; ++k) d -= R[k * s + i] * R[k * s + i];
    if (!(d > 1e-15 * gmax)) return false;
    const double rii = std::sqrt(d);
    R[i * s + i] = rii;
    for (int j = i + 1; j < s; ++j) {
      double v = G[i * s + j];
      for (int k = 0; k < i; ++k) v -= R[k * s + i] * R[k * s + j];
      R[i * s + j] = v / rii;
    }
  }
  return true;
}

void upper_inverse(int s, const double* R, double* Ri) {
  std::fill(Ri, Ri + s * s, 0.0);
  for (int j = 0; j < s; ++j) {
    Ri[j * s + j] = 1.0 / R[j * s + j];
    for (int i = j - 1; i >= 0; --i) {
      double v = 0.0;
      for (int k = i + 1; k <= j; ++k) v += R[i * s + k] * Ri[k * s + j];
      Ri[i * s + j] = -v / R[i * s + i];
    }
  }
}

void matmul(int s, const double* A, const double* B, double* C) {
  for (int i = 0; i < s; ++i)
    for (int j = 0; j < s; ++j) {
      double v = 0.0;
      for (int k = 0; k < s; ++k) v += A[i * s + k] * B[k * s + j];
      C[i * s + j] = v;
    }
}

// ---- dense symmetric eigen-decomposition on the device (library call) --------------------------
struct DenseEigh {
  cusolverDnHandle_t handle = nullptr;
  DeviceBuf A, w, work, info;
  size_t cap_m = 0;
  int lwork = 0;
  ~DenseEigh() {
    if (handle) cusolverDnDestroy(handle);
  }
  // Device buffers for problems up to m x m.  Allocated once per solve of the library (cudaMalloc
  // and cudaFree between the block steps cost up to a second each on a busy context).
  int reserve(int m) {
    if (!handle) {
      if (cusolverDnCreate(&handle) != CUSOLVER_STATUS_SUCCESS)
        return fail(POLFED_ECUDA, "cusolverDnCreate failed");
    }
    if ((size_t)m <= cap_m) return POLFED_OK;
    cudaFree(A.p); cudaFree(w.p); cudaFree(work.p); cudaFree(info.p);
    A.p = w.p = work.p = info.p = nullptr;
    cap_m = 0;
    POLFED_CUDA(A.alloc(sizeof(double) * (size_t)m * m));
    POLFED_CUDA(w.alloc(sizeof(double) * (size_t)m));
    POLFED_CUDA(info.alloc(sizeof(int)));
    if (cusolverDnDsyevd_bufferSize(handle, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, m,
                                    A.f64(), m, w.f64(), &lwork) != CUSOLVER_STATUS_SUCCESS)
      return fail(POLFED_ECUDA, "cusolverDnDsyevd_bufferSize failed");
    POLFED_CUDA(work.alloc(sizeof(double) * (size_t)lwork));
    cap_m = (size_t)m;
    return POLFED_OK;
  }
  // h_A: m x m symmetric (row- or column-major alike).  On return h_w ascending, h_Z column j =
  // eigenvector j, stored contiguously (h_Z[j*m + i]).
  int solve(int m, const double* h_A, double* h_w, double* h_Z, cudaStream_t st) {
    int rc = reserve(m);
    if (rc) return rc;
    cusolverDnSetStream(handle, st);
    POLFED_CUDA(cudaMemcpyAsync(A.p, h_A, sizeof(double) * (size_t)m * m, cudaMemcpyHostToDevice, st));
    if (cusolverDnDsyevd(handle, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, m, A.f64(), m,
                         w.f64(), work.f64(), lwork, static_cast<int*>(info.p)) != CUSOLVER_STATUS_SUCCESS)
      return fail(POLFED_ECUDA, "cusolverDnDsyevd failed");
    int h_info = 0;
    POLFED_CUDA(cudaMemcpyAsync(&h_info, info.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaMemcpyAsync(h_w, w.p, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaMemcpyAsync(h_Z, A.p, sizeof(double) * (size_t)m * m, cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaStreamSynchronize(st));
    if (h_info != 0) return fail(POLFED_ECUDA, "cusolverDnDsyevd did not converge (info=%d)", h_info);
    return POLFED_OK;
  }
};

// P(x) = sum_k c_k T_k(x) by the scalar Clenshaw recurrence (Eq. 50-51 with H~ -> x).
// Outside [-1, 1] the series is not the filter any more (it grows without bound): 0 there, so that an
// out-of-interval level never passes a main-lobe test.
double filter_value(const std::vector<double>& c, double x) {
  if (!(std::fabs(x) <= 1.0)) return 0.0;
  double b1 = 0.0, b2 = 0.0;
  for (size_t k = c.size() - 1; k >= 1; --k) {
    const double t = c[k] + 2.0 * x * b1 - b2;
    b2 = b1;
    b1 = t;
  }
  return c[0] + x * b1 - b2;
}
constexpr double kOmega = 0.17613;  // sin(2.655)/2.655, the cutoff implied by Eq. (42) (R4)

// ---- CholeskyQR on one n x s panel, in place ----------------------------------------------------
struct PanelQR {
  int s;
  long long n;
  int sm_count;
  cudaStream_t st;
  DeviceBuf small;  // 2 * s*s doubles
  std::vector<double> G, R, Ri, R1, tmp;
  int init() {
    G.resize(s * s); R.resize(s * s); Ri.resize(s * s); R1.resize(s * s); tmp.resize(s * s);
    POLFED_CUDA(small.alloc(sizeof(double) * 2 * s * s));
    return POLFED_OK;
  }
  // W <- W R^-1 with W^T W = R^T R; R (host, s x s upper) returned in R.
  int once(double* W) {
    double* dG = small.f64();
    double* dRi = dG + s * s;
    int rc = ts_gram(s, n, W, 1, 0, W, dG, sm_count, st);
    if (rc) return rc;
    POLFED_CUDA(cudaMemcpyAsync(G.data(), dG, sizeof(double) * s * s, cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaStreamSynchronize(st));
    for (int i = 0; i < s; ++i)
      for (int j = i + 1; j < s; ++j) G[i * s + j] = G[j * s + i] = 0.5 * (G[i * s + j] + G[j * s + i]);
    if (!cholesky_upper(s, G.data(), R.data()))
      return fail(POLFED_EBREAKDOWN, "rank-deficient block in CholeskyQR");
    upper_inverse(s, R.data(), Ri.data());
    POLFED_CUDA(cudaMemcpyAsync(dRi, Ri.data(), sizeof(double) * s * s, cudaMemcpyHostToDevice, st));
    return ts_update(s, n, W, 1, 0, dRi, 1.0, 0.0, W, st);
  }
  // CholeskyQR2: W = Q B with B = R2 R1 (host, row-major upper triangular) in `B`.
  int twice(double* W, double* B) {
    int rc = once(W);
    if (rc) return rc;
    R1 = R;
    rc = once(W);
    if (rc) return rc;
    matmul(s, R.data(), R1.data(), B);
    return POLFED_OK;
  }
};

}  // namespace
}  // namespace polfed

using polfed::fail;

extern "C" {

int polfed_spectrum_bounds(const polfed_ham* ham, int n_steps, const double* d_v0, double margin,
                           void* stream, double* emin, double* emax, double* a, double* b) {
  using namespace polfed;
  if (!ham) return fail(POLFED_EINVAL, "polfed_spectrum_bounds: ham is NULL");
  if (ham->n < 1) return fail(POLFED_EINVAL, "polfed_spectrum_bounds: empty matrix");
  if (!d_v0) return fail(POLFED_EINVAL, "polfed_spectrum_bounds: d_v0 is NULL");
  if (n_steps <= 0) n_steps = 60;
  if (margin < 0.0) margin = 0.01;
  const long long n = ham->n;
  const int m_max = (int)std::min<long long>(n_steps, n);
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  DeviceBuf basis, coef;
  POLFED_CUDA(basis.alloc(sizeof(double) * (size_t)n * (m_max + 1)));
  POLFED_CUDA(coef.alloc(sizeof(double) * (size_t)(m_max + 2)));
  double* Phi = basis.f64();
  double* dC = coef.f64();
  std::vector<double> hC(m_max + 2), alpha, beta;
  double b_last = 0.0;  // norm of the last residual vector

  // phi_1 = v0 / ||v0||
  POLFED_CUDA(cudaMemcpyAsync(Phi, d_v0, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, st));
  int rc = ts_gram(1, n, Phi, 1, 0, Phi, dC, ham->sm_count, st);
  if (rc) return rc;
  POLFED_CUDA(cudaMemcpyAsync(hC.data(), dC, sizeof(double), cudaMemcpyDeviceToHost, st));
  POLFED_CUDA(cudaStreamSynchronize(st));
  if (!(hC[0] > 0.0) || !std::isfinite(hC[0]))
    return fail(POLFED_EINVAL, "polfed_spectrum_bounds: start vector is zero or not finite");
  double scale = 1.0 / std::sqrt(hC[0]);
  POLFED_CUDA(cudaMemcpyAsync(dC, &scale, sizeof(double), cudaMemcpyHostToDevice, st));
  rc = ts_update(1, n, Phi, 1, 0, dC, 1.0, 0.0, Phi, st);
  if (rc) return rc;

  for (int i = 0; i < m_max; ++i) {  // Eq. (2)-(4) with full reorthogonalisation
    double* w = Phi + (size_t)(i + 1) * n;
    rc = dispatch_step(ham, 1, 1.0, 0.0, 0.0, 0.0, Phi + (size_t)i * n, nullptr, nullptr, w, st);
    if (rc) return rc;
    for (int pass = 0; pass < 2; ++pass) {
      rc = ts_gram(1, n, Phi, i + 1, (size_t)n, w, dC, ham->sm_count, st);
      if (rc) return rc;
      if (pass == 0) {
        POLFED_CUDA(cudaMemcpyAsync(hC.data(), dC + i, sizeof(double), cudaMemcpyDeviceToHost, st));
        POLFED_CUDA(cudaStreamSynchronize(st));
        alpha.push_back(hC[0]);  // a_i = <phi_i|H|phi_i>
      }
      rc = ts_update(1, n, Phi, i + 1, (size_t)n, dC, -1.0, 1.0, w, st);
      if (rc) return rc;
    }
    rc = ts_gram(1, n, w, 1, 0, w, dC, ham->sm_count, st);
    if (rc) return rc;
    POLFED_CUDA(cudaMemcpyAsync(hC.data(), dC, sizeof(double), cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaStreamSynchronize(st));
    const double bnext = std::sqrt(std::max(hC[0], 0.0));
    b_last = bnext;
    if (i + 1 == m_max || !(bnext > 1e-14 * std::max(1.0, std::fabs(alpha.back())))) break;
    beta.push_back(bnext);
    scale = 1.0 / bnext;
    POLFED_CUDA(cudaMemcpyAsync(dC, &scale, sizeof(double), cudaMemcpyHostToDevice, st));
    POLFED_CUDA(cudaStreamSynchronize(st));
    rc = ts_update(1, n, w, 1, 0, dC, 1.0, 0.0, w, st);
    if (rc) return rc;
  }
  const int m = (int)alpha.size();
  std::vector<double> T((size_t)m * m, 0.0), ev(m), Z((size_t)m * m);
  for (int i = 0; i < m; ++i) {
    T[(size_t)i * m + i] = alpha[i];
    if (i + 1 < m && i < (int)beta.size()) T[(size_t)i * m + i + 1] = T[(size_t)(i + 1) * m + i] = beta[i];
  }
  DenseEigh eig;
  rc = eig.solve(m, T.data(), ev.data(), Z.data(), st);
  if (rc) return rc;
  // Ritz values lie inside the spectrum: for a and b the extremal ones are moved outwards by
  // their residual norms beta_{m+1} |last eigenvector component| (Eq. 6 / 16; reading R5)
  if (emin) *emin = ev.front();
  if (emax) *emax = ev.back();
  const double lo = ev.front() - b_last * std::fabs(Z[(size_t)0 * m + (m - 1)]);
  const double hi = ev.back() + b_last * std::fabs(Z[(size_t)(m - 1) * m + (m - 1)]);
  if (a) *a = 0.5 * (hi + lo);
  if (b) *b = 0.5 * (hi - lo) * (1.0 + margin);
  return POLFED_OK;
}

int polfed_block_lanczos_eigs(const polfed_ham* ham, double sigma, int nev, int s, const double* d_V0,
                              const polfed_options* options, double* h_evals, double* d_evecs,
                              double* h_residuals, polfed_report* report, void* stream) {
  using namespace polfed;
  if (!ham) return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: ham is NULL");
  if (!valid_block_size(s)) return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: bad block size s=%d", s);
  if (nev < 1 || nev > ham->n) return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: nev=%d out of range", nev);
  if (!d_V0 || !h_evals || !d_evecs || !h_residuals)
    return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: NULL argument");
  if (!aligned16(d_V0)) return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: d_V0 must be 16-byte aligned");
  polfed_options opt;
  std::memset(&opt, 0, sizeof opt);
  opt.bounds_margin = -1.0;
  if (options) opt = *options;
  polfed_report rep;
  std::memset(&rep, 0, sizeof rep);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const long long n = ham->n;
  const size_t panel = ((size_t)n * s + 1) & ~(size_t)1;  // doubles per panel, kept 16-byte aligned
  const double t_start = now_seconds();

  // -- step 1: rescaling parameters (Eq. 31)
  double a_ = opt.a, b_ = opt.b, e_min, e_max;
  if (b_ > 0.0) {
    e_min = a_ - b_;
    e_max = a_ + b_;
  } else {
    DeviceBuf v0;
    POLFED_CUDA(v0.alloc(sizeof(double) * (size_t)n));
    POLFED_CUDA(cudaMemcpy2DAsync(v0.p, sizeof(double), d_V0, sizeof(double) * s, sizeof(double),
                                  (size_t)n, cudaMemcpyDeviceToDevice, st));
    const double t0 = now_seconds();
    int rc = polfed_spectrum_bounds(ham, opt.bounds_steps, v0.f64(), opt.bounds_margin, stream, &e_min,
                                    &e_max, &a_, &b_);
    if (rc) return rc;
    rep.seconds_bounds = now_seconds() - t0;
    if (!(b_ > 0.0)) return fail(POLFED_ERANGE, "polfed_block_lanczos_eigs: degenerate spectrum bounds");
  }
  const double lam = opt.sigma_is_rescaled ? sigma : (sigma - a_) / b_;
  const double sigma_E = a_ + b_ * lam;
  if (!(lam > -1.0 && lam < 1.0))
    return fail(POLFED_ERANGE, "polfed_block_lanczos_eigs: rescaled target %g outside (-1,1)", lam);
  const double h_norm = std::max(std::fabs(e_min), std::fabs(e_max));
  const double tol = opt.tol > 0.0 ? opt.tol : 1e-8 * h_norm;

  // -- step 2-3: order from the density of states at the target (Eq. 34 or 35-39, then 40-42).
  // The window is sized for 10 % more levels than asked for (at least 2 more): a density estimate
  // that is a few per cent high would otherwise leave fewer than nev levels inside the main lobe
  // and secondary-peak levels would fill the set (reading R4).
  if (opt.window_levels > 0 && opt.window_levels < nev)
    return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: window_levels=%d < nev=%d", opt.window_levels, nev);
  const int nev_window = opt.window_levels > 0 ? opt.window_levels : nev + std::max(2, (nev + 9) / 10);
  rep.nev_window = nev_window;
  int K = opt.K_override;
  double rho = 0.0;
  if (K <= 0) {
    const double t0 = now_seconds();
    DeviceBuf mom;
    POLFED_CUDA(mom.alloc(2 * sizeof(double)));
    int rc = csr_moments(ham, mom.f64(), st);
    if (rc) return rc;
    double h_mom[2];
    POLFED_CUDA(cudaMemcpyAsync(h_mom, mom.p, sizeof h_mom, cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaStreamSynchronize(st));
    const double mu = h_mom[0] / (double)n;
    const double var = h_mom[1] / (double)n - mu * mu;
    if (var > 0.0) {
      const double gam = std::sqrt(var);
      rep.rho_gaussian = b_ * (double)n / (std::sqrt(2.0 * M_PI) * gam) *
                         std::exp(-(sigma_E - mu) * (sigma_E - mu) / (2.0 * var));
      if (rep.rho_gaussian > 0.0)
        polfed_filter_coeffs(a_, b_, sigma_E, nev_window, rep.rho_gaussian, 0, &rep.K_gaussian, nullptr, 0);
    }
    if (opt.dos == POLFED_DOS_KPM) {
      // Eq. (37)-(38): moments averaged over the caller's random vectors, in chunks of at most 32
      const int n_mom = opt.kpm_moments > 0 ? opt.kpm_moments : 75;
      const int n_vec = opt.kpm_vectors;
      if (!opt.d_kpm_block || n_vec < 4 || n_vec % 4 != 0)
        return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: POLFED_DOS_KPM needs d_kpm_block with a "
                                   "positive multiple of 4 columns");
      DeviceBuf chunk, kwork;
      POLFED_CUDA(chunk.alloc(sizeof(double) * (size_t)n * 32));
      POLFED_CUDA(kwork.alloc(polfed_kpm_workspace_bytes(n, 32, n_mom)));
      std::vector<double> mu_avg(n_mom, 0.0), mu_c(n_mom);
      for (int c0 = 0; c0 < n_vec;) {
        const int left = n_vec - c0;
        const int sc = left >= 32 ? 32 : (left >= 16 ? 16 : (left >= 8 ? 8 : 4));
        POLFED_CUDA(cudaMemcpy2DAsync(chunk.p, sizeof(double) * sc, opt.d_kpm_block + c0,
                                      sizeof(double) * n_vec, sizeof(double) * sc, (size_t)n,
                                      cudaMemcpyDeviceToDevice, st));
        rc = polfed_kpm_moments(ham, a_, b_, n_mom, sc, chunk.f64(), kwork.p, mu_c.data(), stream);
        if (rc) return rc;
        for (int i = 0; i < n_mom; ++i) mu_avg[i] += mu_c[i] * sc / n_vec;
        rep.sparse_products += n_mom;
        c0 += sc;
      }
      rc = polfed_kpm_dos(mu_avg.data(), n_mom, &lam, 1, &rep.rho_kpm);
      if (rc) return rc;
      if (rep.rho_kpm > 0.0)
        polfed_filter_coeffs(a_, b_, sigma_E, nev_window, rep.rho_kpm, 0, &rep.K_kpm, nullptr, 0);
      rho = rep.rho_kpm;
    } else {
      rho = rep.rho_gaussian;
    }
    rep.seconds_dos = now_seconds() - t0;
    if (!(rho > 0.0))
      return fail(POLFED_ERANGE, "polfed_block_lanczos_eigs: zero density of states at the target");
  }
  int K_out = 0;
  int rc = polfed_filter_coeffs(a_, b_, sigma_E, nev_window, rho, K, &K_out, nullptr, 0);
  if (rc) return rc;
  K = K_out;
  std::vector<double> coeffs((size_t)K + 1);
  rc = polfed_filter_coeffs(a_, b_, sigma_E, nev_window, 0.0, K, &K_out, coeffs.data(), K + 1);
  if (rc) return rc;

  // -- sizes and device memory
  const int want_cols = (int)std::min<long long>((long long)nev + s, n);
  const int npan = (want_cols + s - 1) / s;
  const int wp = npan * s;  // padded number of Ritz vectors extracted
  long long m_cap = opt.max_krylov_dim;
  if (m_cap <= 0) {
    // R10: 5 nev + 8 s columns, but never more than fits in 85 % of the free device memory
    m_cap = 5LL * nev + 8LL * s;
    size_t free_b = 0, total_b = 0;
    POLFED_CUDA(cudaMemGetInfo(&free_b, &total_b));
    const double panel_bytes = (double)panel * sizeof(double);
    const long long fit = (long long)(0.85 * (double)free_b / panel_bytes) - (2LL * npan + 4);
    m_cap = std::min<long long>(m_cap, std::max<long long>(fit, npan) * s);
  }
  m_cap = std::min<long long>(m_cap, n);
  m_cap = ((m_cap + s - 1) / s) * s;
  if (m_cap > n) m_cap -= s;
  if (m_cap < wp) return fail(POLFED_EINVAL, "polfed_block_lanczos_eigs: max_krylov_dim=%lld < nev + s rounded up (%d), or n too small for this s", m_cap, wp);
  const int k_cap = (int)(m_cap / s);

  DeviceBuf Qb, work, Ub, Xb, T1b, coefb, evb, colsb;
  POLFED_CUDA(Qb.alloc(sizeof(double) * panel * (size_t)(k_cap + 1)));
  POLFED_CUDA(work.alloc(polfed_filter_workspace_bytes_ham(ham, s)));
  POLFED_CUDA(Ub.alloc(sizeof(double) * panel * (size_t)npan));
  POLFED_CUDA(Xb.alloc(sizeof(double) * panel * (size_t)npan));
  POLFED_CUDA(T1b.alloc(sizeof(double) * panel));
  POLFED_CUDA(coefb.alloc(sizeof(double) * (size_t)std::max<long long>(m_cap + s, wp) * s));
  POLFED_CUDA(evb.alloc(sizeof(double) * (size_t)(s + 2)));
  POLFED_CUDA(colsb.alloc(sizeof(int) * (size_t)nev));
  double* Q = Qb.f64();
  double* dC = coefb.f64();
  PanelQR qr{s, n, ham->sm_count, st};
  rc = qr.init();
  if (rc) return rc;
  DenseEigh eig;
  rc = eig.reserve((int)std::max<long long>(m_cap, wp));
  if (rc) return rc;

  std::vector<double> HL((size_t)m_cap * m_cap, 0.0);  // H_L, preallocated
  std::vector<double> hC((size_t)(m_cap + s) * s), Bk(s * s), Bprev(s * s, 0.0);
  std::vector<double> theta, Zl, G((size_t)wp * wp), Eg(wp), Zg((size_t)wp * wp), res(wp), Csel;
  std::vector<double> best_E, best_res;
  std::vector<int> best_cols;
  bool have_best = false;

  // -- V_1 = orthonormalised start block
  POLFED_CUDA(cudaMemcpyAsync(Q, d_V0, sizeof(double) * (size_t)n * s, cudaMemcpyDeviceToDevice, st));
  rc = qr.twice(Q, Bk.data());
  if (rc) return rc;

  // launches of one filter application that skip V: steps k = K-1 .. 0 with c_k == 0 exactly (R22)
  long long zero_coeffs = 0;
  for (int kk = 0; kk < K; ++kk) zero_coeffs += coeffs[kk] == 0.0 ? 1 : 0;
  int next_check = (wp + s - 1) / s;
  int status = POLFED_ENOCONV;
  int k = 0;
  for (k = 1; k <= k_cap; ++k) {
    double* Vk = Q + panel * (size_t)(k - 1);
    double* W = Q + panel * (size_t)k;
    // W = P(H~) V_k  -- the hot path
    double t0 = now_seconds();
    rc = polfed_filter_apply(ham, a_, b_, K, coeffs.data(), s, Vk, W, work.p, stream);
    if (rc) return rc;
    POLFED_CUDA(cudaStreamSynchronize(st));
    rep.seconds_filter += now_seconds() - t0;
    rep.sparse_products += K;
    rep.products_without_v += zero_coeffs;

    // A_k = V_k^T W and full reorthogonalisation against V_1..V_k, twice (Eq. 9, 11)
    t0 = now_seconds();
    for (int pass = 0; pass < 2; ++pass) {
      rc = ts_gram(s, n, Q, k, panel, W, dC, ham->sm_count, st);
      if (rc) return rc;
      if (pass == 0) {
        POLFED_CUDA(cudaMemcpyAsync(hC.data(), dC + (size_t)(k - 1) * s * s, sizeof(double) * s * s,
                                    cudaMemcpyDeviceToHost, st));
      }
      rc = ts_update(s, n, Q, k, panel, dC, -1.0, 1.0, W, st);
      if (rc) return rc;
    }
    POLFED_CUDA(cudaStreamSynchronize(st));
    rep.seconds_reorth += now_seconds() - t0;
    if (k == 1)  // a spectrum that sticks out of [-1, 1] makes the recurrence grow like cosh(K acosh|x|)
      for (int i = 0; i < s * s; ++i)
        if (!std::isfinite(hC[i]))
          return fail(POLFED_ERANGE, "polfed_block_lanczos_eigs: the filtered block is not finite "
                                     "(spectrum outside [a - b, a + b]?)");
    const size_t o = (size_t)(k - 1) * s;
    for (int i = 0; i < s; ++i)
      for (int j = 0; j < s; ++j)
        HL[(o + i) * m_cap + o + j] = 0.5 * (hC[i * s + j] + hC[j * s + i]);  // A_k (Eq. 13)

    // W = V_{k+1} B_{k+1} (Eq. 12)
    t0 = now_seconds();
    rc = qr.twice(W, Bk.data());
    if (rc) return rc;
    POLFED_CUDA(cudaStreamSynchronize(st));
    rep.seconds_qr += now_seconds() - t0;
    if (k < k_cap)
      for (int i = 0; i < s; ++i)
        for (int j = 0; j < s; ++j) {
          HL[(o + s + i) * m_cap + o + j] = Bk[i * s + j];  // B_{k+1} below the diagonal (Eq. 14)
          HL[(o + j) * m_cap + o + s + i] = Bk[i * s + j];
        }
    rep.block_steps = k;
    rep.krylov_dim = k * s;

    const int m = k * s;
    if (m < wp || (k < next_check && k != k_cap)) continue;

    // -- convergence check: Ritz pairs of H_L
    t0 = now_seconds();
    std::vector<double> Hm((size_t)m * m);
    for (int i = 0; i < m; ++i) std::memcpy(&Hm[(size_t)i * m], &HL[(size_t)i * m_cap], sizeof(double) * m);
    theta.resize(m);
    Zl.resize((size_t)m * m);
    rc = eig.solve(m, Hm.data(), theta.data(), Zl.data(), st);
    if (rc) return rc;
    rep.seconds_projected_eig += now_seconds() - t0;
    rep.n_checks += 1;
    // Eq. (16)-(17): ||B_{k+1} tau_j|| for the wp largest Ritz values (eigenvalues ascending)
    int n_small = 0;
    const double theta_top = std::fabs(theta[m - 1]);
    for (int c = 0; c < wp; ++c) {
      const double* z = &Zl[(size_t)(m - 1 - c) * m];
      double e2 = 0.0;
      for (int i = 0; i < s; ++i) {
        double v = 0.0;
        for (int j = 0; j < s; ++j) v += Bk[i * s + j] * z[m - s + j];
        e2 += v * v;
      }
      if (std::sqrt(e2) <= 1e-2 * theta_top) ++n_small;
    }
    if (n_small < nev && k != k_cap) {
      next_check = opt.check_every > 0 ? k + opt.check_every : k + std::max(1, (nev - n_small + 2 * s - 1) / (2 * s));
      continue;
    }

    // -- extraction: u = V_{1:m} t (Eq. 43), Rayleigh-Ritz of H in span(u) (R21), residuals
    t0 = now_seconds();
    double* U = Ub.f64();
    double* X = Xb.f64();
    double* T1 = T1b.f64();
    Csel.resize((size_t)m * s);
    for (int p = 0; p < npan; ++p) {
      for (int r = 0; r < m; ++r)
        for (int c = 0; c < s; ++c) Csel[(size_t)r * s + c] = Zl[(size_t)(m - 1 - (p * s + c)) * m + r];
      POLFED_CUDA(cudaMemcpyAsync(dC, Csel.data(), sizeof(double) * (size_t)m * s, cudaMemcpyHostToDevice, st));
      rc = ts_update(s, n, Q, k, panel, dC, 1.0, 0.0, U + panel * (size_t)p, st);
      if (rc) return rc;
      POLFED_CUDA(cudaStreamSynchronize(st));
    }
    for (int p = 0; p < npan; ++p) {
      rc = dispatch_step(ham, s, 1.0, 0.0, 0.0, 0.0, U + panel * (size_t)p, nullptr, nullptr, T1, st);
      if (rc) return rc;
      rc = ts_gram(s, n, U, npan, panel, T1, dC, ham->sm_count, st);
      if (rc) return rc;
      POLFED_CUDA(cudaMemcpyAsync(hC.data(), dC, sizeof(double) * (size_t)wp * s, cudaMemcpyDeviceToHost, st));
      POLFED_CUDA(cudaStreamSynchronize(st));
      for (int r = 0; r < wp; ++r)
        for (int c = 0; c < s; ++c) G[(size_t)r * wp + p * s + c] = hC[(size_t)r * s + c];
      rep.sparse_products += 1;
    }
    for (int i = 0; i < wp; ++i)
      for (int j = i + 1; j < wp; ++j)
        G[(size_t)i * wp + j] = G[(size_t)j * wp + i] = 0.5 * (G[(size_t)i * wp + j] + G[(size_t)j * wp + i]);
    const double t1 = now_seconds();
    rc = eig.solve(wp, G.data(), Eg.data(), Zg.data(), st);
    if (rc) return rc;
    const double t_eig_inside = now_seconds() - t1;
    rep.seconds_projected_eig += t_eig_inside;
    for (int p = 0; p < npan; ++p) {
      Csel.resize((size_t)wp * s);
      for (int r = 0; r < wp; ++r)
        for (int c = 0; c < s; ++c) Csel[(size_t)r * s + c] = Zg[(size_t)(p * s + c) * wp + r];
      POLFED_CUDA(cudaMemcpyAsync(dC, Csel.data(), sizeof(double) * (size_t)wp * s, cudaMemcpyHostToDevice, st));
      double* Xp = X + panel * (size_t)p;
      rc = ts_update(s, n, U, npan, panel, dC, 1.0, 0.0, Xp, st);
      if (rc) return rc;
      rc = dispatch_step(ham, s, 1.0, 0.0, 0.0, 0.0, Xp, nullptr, nullptr, T1, st);
      if (rc) return rc;
      POLFED_CUDA(cudaMemcpyAsync(evb.p, &Eg[(size_t)p * s], sizeof(double) * s, cudaMemcpyHostToDevice, st));
      rc = ts_residual_norms(s, n, T1, Xp, evb.f64(), dC, ham->sm_count, st);
      if (rc) return rc;
      POLFED_CUDA(cudaMemcpyAsync(&res[(size_t)p * s], dC, sizeof(double) * s, cudaMemcpyDeviceToHost, st));
      POLFED_CUDA(cudaStreamSynchronize(st));
      rep.sparse_products += 1;
    }
    for (int c = 0; c < wp; ++c) res[c] = std::sqrt(std::max(res[c], 0.0));
    rep.seconds_extraction += now_seconds() - t0 - t_eig_inside;
    // The bounds of step 1 are a heuristic, not an enclosure (R5).  A Rayleigh-Ritz value of H
    // itself never leaves [E_min, E_max], so one outside [a - b, a + b] proves that the spectrum
    // sticks out of the Chebyshev interval: there P grows like cosh(K acosh|x|) and swamps the window.
    for (int c = 0; c < wp; ++c) {
      const double x = (Eg[c] - a_) / b_;
      if (std::fabs(x) > 1.0)
        return fail(POLFED_ERANGE,
                    "polfed_block_lanczos_eigs: Ritz value %.17g of H lies outside [a - b, a + b] = [%.17g, %.17g] "
                    "(rescaled %.6f): the spectral bounds are too tight; raise bounds_steps or bounds_margin, "
                    "or pass a, b", Eg[c], a_ - b_, a_ + b_, x);
    }

    // -- selection (R11): converged pairs nearest sigma
    std::vector<int> order(wp);
    for (int c = 0; c < wp; ++c) order[c] = c;
    std::sort(order.begin(), order.end(), [&](int x, int y) {
      return std::fabs(Eg[x] - sigma_E) < std::fabs(Eg[y] - sigma_E);
    });
    std::vector<int> good;
    for (int c : order)
      if (res[c] <= tol) good.push_back(c);
    // done only when the nev extracted pairs nearest sigma are all converged (a converged pair
    // farther away must not stand in for an unconverged nearer one) and lie inside the main lobe
    // of the filter, P(lambda~_i) > Omega: levels on a secondary peak
    // (P <= 0.128) are true eigenpairs too, but the set would not be contiguous
    int n_lead = 0;
    while (n_lead < wp && res[order[n_lead]] <= tol &&
           filter_value(coeffs, (Eg[order[n_lead]] - a_) / b_) > kOmega)
      ++n_lead;
    rep.n_converged = std::min(n_lead, nev);
    std::vector<int> sel;
    const bool done = n_lead >= nev;
    // Every extracted pair converged, yet fewer than nev of them in the main lobe: the wp levels
    // with the largest P are all known, so the lobe holds fewer than nev levels (density of states
    // overestimated, K too high) and no further block step can change that.  Stop here instead of
    // running to max_krylov_dim; the outputs are the nev converged pairs nearest sigma.
    const bool narrow = !done && (int)good.size() == wp;
    if (done || narrow) {
      sel.assign(good.begin(), good.begin() + nev);
    } else {
      sel.assign(order.begin(), order.begin() + nev);
    }
    std::sort(sel.begin(), sel.end(), [&](int x, int y) { return Eg[x] < Eg[y]; });
    if (done || narrow || k == k_cap || !have_best) {
      // write the outputs (best effort until converged)
      for (int j = 0; j < nev; ++j) {
        h_evals[j] = Eg[sel[j]];
        h_residuals[j] = res[sel[j]];
      }
      // columns grouped by panel: gather from X panels into d_evecs (n x nev row-major)
      for (int j = 0; j < nev; ++j) {
        const int c = sel[j];
        const int pcol = c % s;
        POLFED_CUDA(cudaMemcpyAsync(colsb.p, &pcol, sizeof(int), cudaMemcpyHostToDevice, st));
        rc = ts_gather_columns(n, X + panel * (size_t)(c / s), s, static_cast<int*>(colsb.p), 1, d_evecs,
                               nev, j, ham->sm_count, st);
        if (rc) return rc;
        POLFED_CUDA(cudaStreamSynchronize(st));
      }
      have_best = true;
    }
    if (done) {
      status = POLFED_OK;
      break;
    }
    if (narrow) {
      status = POLFED_EWINDOW;
      break;
    }
    const int missing = nev - std::min(n_lead, nev);
    next_check = opt.check_every > 0 ? k + opt.check_every : k + std::max(1, (missing + 2 * s - 1) / (2 * s));
  }

  POLFED_CUDA(cudaStreamSynchronize(st));
  rep.a = a_;
  rep.b = b_;
  rep.lambda_rescaled = lam;
  rep.e_min = e_min;
  rep.e_max = e_max;
  rep.tol = tol;
  rep.K = K;
  rep.seconds_total = now_seconds() - t_start;
  if (report) *report = rep;
  if (status == POLFED_EWINDOW)
    return fail(POLFED_EWINDOW,
                "polfed_block_lanczos_eigs: all %d extracted pairs are converged eigenpairs but only %d lie in the "
                "main lobe of the filter (K = %d is too high for nev = %d: density of states overestimated); "
                "the outputs hold the nev converged pairs nearest sigma; lower K_override or raise window_levels",
                wp, rep.n_converged, K, nev);
  if (status == POLFED_ENOCONV)
    return fail(POLFED_ENOCONV, "polfed_block_lanczos_eigs: %d of %d pairs converged at Krylov dimension %d",
                rep.n_converged, nev, rep.krylov_dim);
  return POLFED_OK;
}

}  // extern "C"
