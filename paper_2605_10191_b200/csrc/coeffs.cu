// Host-side filter parameters: delta-filter coefficients and the order rule.
// PAPER.md:280-286 (Eq. 32-33), 343-362 (Eq. 40-42).  Readings R1, R4.
#include <cmath>
#include <vector>

#include "common.cuh"

namespace polfed {
namespace {

// T_n(lambda) for n = 0..K by the three-term recurrence Eq. (28)-(30), re-anchored on the
// cosine form every 64 terms so rounding does not accumulate over long orders.
// At lambda = 0 (the middle of the spectrum, where every mid-spectrum solve sits) the values are
// known exactly: T_n(0) = cos(n pi/2) = 0 for odd n, (-1)^(n/2) for even n.  cos(n * acos(0)) would
// give ~1e-16 instead of 0 there, and a non-zero c_n costs the fused step its V read (R22).
void chebyshev_at(double lam, int K, std::vector<double>& T) {
  T.assign((size_t)K + 1, 1.0);
  if (K == 0) return;
  if (lam == 0.0) {
    for (int n = 1; n <= K; ++n) T[n] = (n & 1) ? 0.0 : ((n & 2) ? -1.0 : 1.0);
    return;
  }
  const double theta = std::acos(lam);
  T[1] = lam;
  for (int n = 2; n <= K; ++n) {
    if ((n & 63) <= 1)
      T[n] = std::cos((double)n * theta);
    else
      T[n] = 2.0 * lam * T[n - 1] - T[n - 2];
  }
}

// Unnormalised weights w_0 = 1, w_n = 2 T_n(lambda); chi = sum_n w_n T_n(lambda).
double fill_coeffs(double lam, int K, double* out) {
  std::vector<double> T;
  chebyshev_at(lam, K, T);
  long double chi = 1.0L;
  for (int n = 1; n <= K; ++n) chi += 2.0L * (long double)T[n] * (long double)T[n];
  if (out) {
    out[0] = (double)(1.0L / chi);
    for (int n = 1; n <= K; ++n) out[n] = (double)(2.0L * (long double)T[n] / chi);
  }
  return (double)chi;
}

// P(x) for the order-K filter at lam, evaluated with the cosine form.
double filter_at(double lam, int K, double x) {
  const double th = std::acos(lam), tx = std::acos(x);
  long double chi = 1.0L, sum = 1.0L;
  for (int n = 1; n <= K; ++n) {
    const long double t = std::cos((double)n * th);
    chi += 2.0L * t * t;
    sum += 2.0L * t * (long double)std::cos((double)n * tx);
  }
  return (double)(sum / chi);
}

}  // namespace
}  // namespace polfed

using polfed::fail;

extern "C" int polfed_filter_coeffs(double a, double b, double sigma, int nev, double rho_rescaled,
                                    int K_in, int* K_out, double* h_coeffs, int capacity) {
  if (!K_out) return fail(POLFED_EINVAL, "polfed_filter_coeffs: K_out is NULL");
  *K_out = 0;
  if (!(b > 0.0)) return fail(POLFED_ERANGE, "polfed_filter_coeffs: b=%g must be > 0", b);
  const double lam = (sigma - a) / b;
  if (!(lam > -1.0 && lam < 1.0))
    return fail(POLFED_ERANGE, "polfed_filter_coeffs: rescaled target %g outside (-1,1)", lam);
  int K = K_in;
  if (rho_rescaled > 0.0) {
    if (nev < 1) return fail(POLFED_EINVAL, "polfed_filter_coeffs: nev=%d < 1", nev);
    const double delta = (double)nev / (2.0 * rho_rescaled);                  // Eq. (40)
    const double k42 = std::ceil(2.655 * std::sqrt(1.0 - lam * lam) / delta); // Eq. (42)
    if (!(k42 < 1.0e9)) return fail(POLFED_ERANGE, "polfed_filter_coeffs: order %g too large", k42);
    const int K42 = k42 < 1.0 ? 1 : (int)k42;
    // Eq. (41): smallest K in [K42/2, 2 K42] whose value at both window edges is <= Omega.
    const double omega = std::sin(2.655) / 2.655;
    const double xl = lam - delta, xr = lam + delta;
    auto edge = [&](int k) {
      double e = -1.0;
      if (xl > -1.0) e = std::fmax(e, polfed::filter_at(lam, k, xl));
      if (xr < 1.0) e = std::fmax(e, polfed::filter_at(lam, k, xr));
      return e;
    };
    int lo = K42 / 2 < 1 ? 1 : K42 / 2, hi = 2 * K42;
    if (edge(lo) <= omega) {
      K = lo;
    } else if (edge(hi) > omega) {
      K = hi;
    } else {
      while (hi - lo > 1) {
        const int mid = lo + (hi - lo) / 2;
        if (edge(mid) <= omega) hi = mid; else lo = mid;
      }
      K = hi;
    }
  }
  if (K < 0) return fail(POLFED_EINVAL, "polfed_filter_coeffs: K=%d < 0", K);
  *K_out = K;
  if (!h_coeffs) return POLFED_OK;
  if (capacity < K + 1)
    return fail(POLFED_EINVAL, "polfed_filter_coeffs: capacity %d < K+1 = %d", capacity, K + 1);
  polfed::fill_coeffs(lam, K, h_coeffs);
  return POLFED_OK;
}
