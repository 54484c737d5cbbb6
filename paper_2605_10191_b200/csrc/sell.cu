// SELL-8-sigma (sell.cuh): construction from the handle's CSR and the fused step
//   Y = p H X + q X + r Z + c V        (Eq. 51 PAPER.md:427-431 with the rescaling of Eq. 31).
#include <cub/device/device_scan.cuh>

#include <new>

#include "sell.cuh"

namespace polfed {
namespace {

// One CTA per window of sigma positions: rows sorted by (falling length, rising row) with a
// bitonic network in shared memory -- deterministic, unlike a counting sort with atomics.
__global__ void __launch_bounds__(kSellSigma / 2) sell_sort_kernel(long long n,
                                                                  const int32_t* __restrict__ row_ptr,
                                                                  int32_t* __restrict__ perm,
                                                                  int32_t* __restrict__ len) {
  __shared__ unsigned long long key[kSellSigma];
  const long long w0 = (long long)blockIdx.x * kSellSigma;
  for (int i = threadIdx.x; i < kSellSigma; i += blockDim.x) {
    const long long r = w0 + i;
    unsigned long long k = ~0ull;  // past the end: sorts last
    if (r < n) {
      const unsigned l = (unsigned)(row_ptr[r + 1] - row_ptr[r]);
      k = ((unsigned long long)(0xffffffffu - l) << 32) | (unsigned)i;
    }
    key[i] = k;
  }
  __syncthreads();
  for (int size = 2; size <= kSellSigma; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int t = threadIdx.x; t < kSellSigma / 2; t += blockDim.x) {
        const int lo = 2 * t - (t & (stride - 1));
        const int hi = lo + stride;
        const bool up = (lo & size) == 0;
        const unsigned long long a = key[lo], b = key[hi];
        if ((a > b) == up) {
          key[lo] = b;
          key[hi] = a;
        }
      }
      __syncthreads();
    }
  for (int i = threadIdx.x; i < kSellSigma; i += blockDim.x) {
    const unsigned long long k = key[i];
    const bool real = k != ~0ull;
    perm[w0 + i] = real ? (int32_t)(w0 + (unsigned)(k & 0xffffffffu)) : -1;
    len[w0 + i] = real ? (int32_t)(0xffffffffu - (unsigned)(k >> 32)) : 0;
  }
}

// entries of a slice = C * (length of its first, i.e. longest, row)
__global__ void __launch_bounds__(256) sell_width_kernel(long long n_slices,
                                                         const int32_t* __restrict__ len,
                                                         long long* __restrict__ entries) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_slices) entries[i] = (long long)kSellC * len[i * kSellC];
  if (i == n_slices) entries[i] = 0;
}

__global__ void __launch_bounds__(256) sell_fill_kernel(long long n_pos,
                                                        const int32_t* __restrict__ perm,
                                                        const int32_t* __restrict__ len,
                                                        const long long* __restrict__ slice_ptr,
                                                        const int32_t* __restrict__ row_ptr,
                                                        const int32_t* __restrict__ col,
                                                        const double* __restrict__ val,
                                                        int32_t* __restrict__ s_col,
                                                        double* __restrict__ s_val) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_pos) return;
  const long long slice = p / kSellC;
  const int lane = (int)(p % kSellC);
  const long long base = slice_ptr[slice] + lane;
  const int width = (int)((slice_ptr[slice + 1] - slice_ptr[slice]) / kSellC);
  const int row = perm[p], l = len[p];
  const int e0 = row >= 0 ? row_ptr[row] : 0;
  for (int j = 0; j < width; ++j) {
    const bool real = j < l;
    s_col[base + (long long)j * kSellC] = real ? col[e0 + j] : (row >= 0 ? row : 0);
    s_val[base + (long long)j * kSellC] = real ? val[e0 + j] : 0.0;
  }
}


constexpr int kSellThreads = 256;
constexpr int kSellLpr = 4;  // lanes per row

template <int VEC>
struct Vec {
  double v[VEC];
};

template <int VEC, bool STREAM>
__device__ __forceinline__ Vec<VEC> vec_load(const double* p) {
  Vec<VEC> a;
  if constexpr (VEC == 2) {
    const double2 t = STREAM ? __ldcs(reinterpret_cast<const double2*>(p))
                             : __ldg(reinterpret_cast<const double2*>(p));
    a.v[0] = t.x;
    a.v[1] = t.y;
  } else {
#pragma unroll
    for (int h = 0; h < VEC; h += 4) {
      if (STREAM)
        asm volatile("ld.global.cs.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "=d"(a.v[h]), "=d"(a.v[h + 1]), "=d"(a.v[h + 2]), "=d"(a.v[h + 3])
                     : "l"(p + h));
      else
        asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "=d"(a.v[h]), "=d"(a.v[h + 1]), "=d"(a.v[h + 2]), "=d"(a.v[h + 3])
                     : "l"(p + h));
    }
  }
  return a;
}

template <int VEC>
__device__ __forceinline__ void vec_store(double* p, const Vec<VEC>& a) {
  if constexpr (VEC == 2) {
    __stcs(reinterpret_cast<double2*>(p), make_double2(a.v[0], a.v[1]));
  } else {
#pragma unroll
    for (int h = 0; h < VEC; h += 4)
      asm volatile("st.global.cs.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p + h), "d"(a.v[h]),
                   "d"(a.v[h + 1]), "d"(a.v[h + 2]), "d"(a.v[h + 3])
                   : "memory");
  }
}

// A warp owns a slice: lane = 4 * (row of the slice) + quarter of the row (S/4 doubles).
template <int S, bool USE_Z, bool USE_V>
__global__ void __launch_bounds__(kSellThreads)
    sell_step_kernel(long long n_slices, const int32_t* __restrict__ perm,
                     const int32_t* __restrict__ len, const long long* __restrict__ slice_ptr,
                     const int32_t* __restrict__ col, const double* __restrict__ val,
                     const double* __restrict__ X, const double* Z, const double* V, double* Y,
                     double p, double q, double r, double c) {
  constexpr int VEC = S / kSellLpr;
  const int lane = threadIdx.x & 31;
  const int rl = lane / kSellLpr, ql = lane % kSellLpr;
  const long long warps = (long long)gridDim.x * (kSellThreads / 32);
  for (long long slice = (long long)blockIdx.x * (kSellThreads / 32) + (threadIdx.x >> 5);
       slice < n_slices; slice += warps) {
    const long long pos = slice * kSellC + rl;
    const int row = __ldg(perm + pos);
    const int mine = __ldg(len + pos);
    const long long e0 = __ldg(slice_ptr + slice);
    const int width = (int)((__ldg(slice_ptr + slice + 1) - e0) / kSellC);
    const int32_t* cp = col + e0 + rl;
    const double* vp = val + e0 + rl;
    Vec<VEC> acc;
#pragma unroll
    for (int t = 0; t < VEC; ++t) acc.v[t] = 0.0;
    for (int j0 = 0; j0 < width; j0 += 4) {  // four entries of every row in flight
      int cj[4];
      double vj[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        cj[u] = 0;
        vj[u] = 0.0;
        if (j0 + u < mine) {
          cj[u] = __ldcs(cp + (long long)(j0 + u) * kSellC);
          vj[u] = __ldcs(vp + (long long)(j0 + u) * kSellC);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (j0 + u < mine) {
          const Vec<VEC> x = vec_load<VEC, false>(X + (size_t)cj[u] * S + ql * VEC);
#pragma unroll
          for (int t = 0; t < VEC; ++t) acc.v[t] = fma(vj[u], x.v[t], acc.v[t]);
        }
    }
    if (row >= 0) {
      const size_t at = (size_t)row * S + ql * VEC;
      const Vec<VEC> xi = vec_load<VEC, false>(X + at);
      Vec<VEC> y;
#pragma unroll
      for (int t = 0; t < VEC; ++t) y.v[t] = fma(p, acc.v[t], q * xi.v[t]);
      if constexpr (USE_Z) {
        const Vec<VEC> z = vec_load<VEC, true>(Z + at);
#pragma unroll
        for (int t = 0; t < VEC; ++t) y.v[t] = fma(r, z.v[t], y.v[t]);
      }
      if constexpr (USE_V) {
        const Vec<VEC> v = vec_load<VEC, true>(V + at);
#pragma unroll
        for (int t = 0; t < VEC; ++t) y.v[t] = fma(c, v.v[t], y.v[t]);
      }
      vec_store<VEC>(Y + at, y);
    }
  }
}

template <int S>
int launch_sell(const polfed_ham* ham, double p, double q, double r, double c, const double* X,
                const double* Z, const double* V, double* Y, cudaStream_t st) {
  const SellPlan* sp = ham->sell;
  const long long per_cta = kSellThreads / 32;
  const long long want = (sp->n_slices + per_cta - 1) / per_cta;
  const long long cap = (long long)ham->sm_count * 8 * 8;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  const bool uz = r != 0.0, uv = c != 0.0;
#define POLFED_SELL_GO(UZ, UV)                                                                  \
  sell_step_kernel<S, UZ, UV><<<grid, kSellThreads, 0, st>>>(sp->n_slices, sp->d_perm, sp->d_len, \
                                                             sp->d_slice_ptr, sp->d_col, sp->d_val, \
                                                             X, Z, V, Y, p, q, r, c)
  if (uz && uv) POLFED_SELL_GO(true, true);
  else if (uz) POLFED_SELL_GO(true, false);
  else if (uv) POLFED_SELL_GO(false, true);
  else POLFED_SELL_GO(false, false);
#undef POLFED_SELL_GO
  POLFED_LAUNCH_CHECK("sell_step_kernel");
  return POLFED_OK;
}

inline bool aligned32(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) == 0; }

}  // namespace

void destroy_sell_plan(SellPlan* p) {
  if (!p) return;
  cudaFree(p->d_perm);
  cudaFree(p->d_len);
  cudaFree(p->d_slice_ptr);
  cudaFree(p->d_col);
  cudaFree(p->d_val);
  delete p;
}

// s in {8, 16, 32}; the 256-bit accesses of s >= 16 need 32-byte aligned blocks
bool sell_supports(const polfed_ham* ham, int s, const void* X, const void* Z, const void* V,
                   const void* Y) {
  if (!ham || !ham->sell || ham->n == 0 || !(s == 8 || s == 16 || s == 32)) return false;
  return s == 8 || (aligned32(X) && aligned32(Y) && (!Z || aligned32(Z)) && (!V || aligned32(V)));
}

int sell_step(const polfed_ham* ham, int s, double p, double q, double r, double c, const double* X,
              const double* Z, const double* V, double* Y, cudaStream_t st) {
  switch (s) {
    case 8: return launch_sell<8>(ham, p, q, r, c, X, Z, V, Y, st);
    case 16: return launch_sell<16>(ham, p, q, r, c, X, Z, V, Y, st);
    case 32: return launch_sell<32>(ham, p, q, r, c, X, Z, V, Y, st);
  }
  return fail(POLFED_EINVAL, "SELL format: block size s=%d not in {8,16,32}", s);
}

// SELL-8-sigma arrays from the CSR of the handle (any matrix: also polfed_ham_from_csr handles).
int build_sell_plan(const polfed_ham* ham, cudaStream_t st, SellPlan** out) {
  *out = nullptr;
  SellPlan* p = new (std::nothrow) SellPlan;
  if (!p) return fail(POLFED_ENOMEM, "SELL format: host allocation failed");
  struct Guard {
    SellPlan* p;
    ~Guard() { destroy_sell_plan(p); }
  } guard{p};
  const long long n = ham->n;
  const long long n_windows = (n + kSellSigma - 1) / kSellSigma;
  const long long n_pos = n_windows * kSellSigma;
  p->n_slices = n_pos / kSellC;
  POLFED_CUDA(cudaMalloc(&p->d_perm, sizeof(int32_t) * (size_t)(n_pos ? n_pos : 1)));
  POLFED_CUDA(cudaMalloc(&p->d_len, sizeof(int32_t) * (size_t)(n_pos ? n_pos : 1)));
  POLFED_CUDA(cudaMalloc(&p->d_slice_ptr, sizeof(long long) * (size_t)(p->n_slices + 1)));
  if (n > 0) {
    long long* d_entries = nullptr;
    void* d_cub = nullptr;
    POLFED_CUDA(cudaMalloc(&d_entries, sizeof(long long) * (size_t)(p->n_slices + 1)));
    struct Tmp {
      void* a;
      void* b;
      ~Tmp() {
        cudaFree(a);
        cudaFree(b);
      }
    } tmp{d_entries, nullptr};
    sell_sort_kernel<<<(unsigned)n_windows, kSellSigma / 2, 0, st>>>(n, ham->d_row_ptr, p->d_perm,
                                                                     p->d_len);
    POLFED_LAUNCH_CHECK("sell_sort_kernel");
    sell_width_kernel<<<(unsigned)((p->n_slices + 256) / 256), 256, 0, st>>>(p->n_slices, p->d_len,
                                                                             d_entries);
    POLFED_LAUNCH_CHECK("sell_width_kernel");
    size_t bytes = 0;
    POLFED_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, bytes, d_entries, p->d_slice_ptr,
                                              (int)(p->n_slices + 1), st));
    POLFED_CUDA(cudaMalloc(&d_cub, bytes ? bytes : 1));
    tmp.b = d_cub;
    POLFED_CUDA(cub::DeviceScan::ExclusiveSum(d_cub, bytes, d_entries, p->d_slice_ptr,
                                              (int)(p->n_slices + 1), st));
    POLFED_CUDA(cudaMemcpyAsync(&p->padded, p->d_slice_ptr + p->n_slices, sizeof(long long),
                                cudaMemcpyDeviceToHost, st));
    POLFED_CUDA(cudaStreamSynchronize(st));
    POLFED_CUDA(cudaMalloc(&p->d_col, sizeof(int32_t) * (size_t)(p->padded ? p->padded : 1)));
    POLFED_CUDA(cudaMalloc(&p->d_val, sizeof(double) * (size_t)(p->padded ? p->padded : 1)));
    sell_fill_kernel<<<(unsigned)((n_pos + 255) / 256), 256, 0, st>>>(
        n_pos, p->d_perm, p->d_len, p->d_slice_ptr, ham->d_row_ptr, ham->d_col, ham->d_val,
        p->d_col, p->d_val);
    POLFED_LAUNCH_CHECK("sell_fill_kernel");
    POLFED_CUDA(cudaStreamSynchronize(st));
  } else {
    POLFED_CUDA(cudaMemsetAsync(p->d_slice_ptr, 0, sizeof(long long), st));
    POLFED_CUDA(cudaStreamSynchronize(st));
  }
  guard.p = nullptr;
  *out = p;
  return POLFED_OK;
}

}  // namespace polfed
