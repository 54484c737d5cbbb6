// Combinatorial number system on the device: binomial table, rank and unrank.
// Each translation unit that includes this header owns a copy of the constant table and
// uploads it through ensure_binomials().  Reading R12.
#pragma once

#include "common.cuh"

namespace polfed {

// C(n, k), 0 <= n, k < 64, filled once per process.  Entries that overflow uint64 are
// saturated; they are never reached because dim < 2^31 is enforced.
static __constant__ uint64_t c_binom[kBinomDim * kBinomDim];
static uint64_t h_binom[kBinomDim * kBinomDim];
static bool g_binom_host_ready = false;
static unsigned long long g_binom_device_mask = 0;  // devices (ordinal < 64) that hold the table

// The host table is filled once; the constant-memory copy is per device, so it is uploaded on
// the first use on every device.
static int ensure_binomials() {
  int dev = 0;
  POLFED_CUDA(cudaGetDevice(&dev));
  if (g_binom_host_ready && dev < 64 && ((g_binom_device_mask >> dev) & 1ull)) return POLFED_OK;
  for (int n = 0; n < kBinomDim && !g_binom_host_ready; ++n)
    for (int k = 0; k < kBinomDim; ++k) {
      uint64_t v;
      if (k == 0) v = 1;
      else if (n == 0) v = 0;
      else {
        const uint64_t x = h_binom[(n - 1) * kBinomDim + k - 1], y = h_binom[(n - 1) * kBinomDim + k];
        v = (x > UINT64_MAX - y) ? UINT64_MAX : x + y;  // Pascal's rule
      }
      h_binom[n * kBinomDim + k] = v;
    }
  g_binom_host_ready = true;
  POLFED_CUDA(cudaMemcpyToSymbol(c_binom, h_binom, sizeof h_binom));
  if (dev < 64) g_binom_device_mask |= 1ull << dev;
  return POLFED_OK;
}

static inline uint64_t host_binom(int n, int k) {
  if (k < 0 || n < 0 || k > n) return 0;
  return h_binom[n * kBinomDim + k];
}

// rank -> state: choose the set bits from the top; bit p_j is the largest p with C(p, j) <= r.
__device__ __forceinline__ uint64_t unrank_state(uint64_t r, int n_sites, int n_up) {
  uint64_t x = 0;
  int p = n_sites - 1;
  for (int j = n_up; j >= 1; --j) {
    while (c_binom[p * kBinomDim + j] > r) --p;
    x |= 1ull << p;
    r -= c_binom[p * kBinomDim + j];
    --p;
  }
  return x;
}

__device__ __forceinline__ int64_t rank_state(uint64_t x, int n_sites, int n_up) {
  if (n_up < 0) return (n_sites < 64 && (x >> n_sites)) ? -1 : (int64_t)x;
  if ((x >> n_sites) != 0 || __popcll(x) != n_up) return -1;
  uint64_t r = 0;
  int j = 0;
  while (x) {
    const int p = __ffsll((long long)x) - 1;
    x &= x - 1;
    ++j;
    r += c_binom[p * kBinomDim + j];
  }
  return (int64_t)r;
}

}  // namespace polfed
