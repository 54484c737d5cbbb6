// The hot path: fused sparse-matrix x block product + Clenshaw three-term update (sm_100a).
//
//   Y[i,:] = p * sum_j H_ij X[j,:] + q * X[i,:] + r * Z[i,:] + c * V[i,:]
//
// PAPER.md:427-431 (Eq. 51) with the rescaling of Eq. (31) folded into p and q (R18):
//   recurrence step  b_k = 2 H~ b_{k+1} - b_{k+2} + c_k V   ->  p = 2/b, q = -2a/b, r = -1, c = c_k
//   final step       W   =   H~ b_1     - b_2     + c_0 V   ->  p = 1/b, q = -a/b,  r = -1, c = c_0
//
// Layout: CSR (row_ptr int32[N+1], col int32[nnz], val fp64[nnz]); blocks N x S row-major, so
// one nonzero (12 bytes) drives S FMAs and its gather is S*8 contiguous bytes.  A group of
// LPR = S/2 lanes owns one row; every lane keeps two fp64 accumulators and gathers 16 bytes
// per nonzero (128-bit loads).  Column indices and values are read once per row, coalesced
// across the lane group, and handed round by shuffles.  The epilogue reads Z and V and
// writes Y in the same pass -- there is no separate axpy kernel.
#include "common.cuh"
#include "packed.cuh"

namespace polfed {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

// VEC doubles per lane: 2 (128-bit accesses) for S >= 2.  Round 1 used 4 (256-bit accesses, half
// the lanes per row, half the shuffles per entry) for S >= 16; with the packed entries and the
// entry loads one chunk ahead the step is bound by latency, not by the shuffles, and twice the
// entries per chunk win: config 3 24.1 -> 20.9 us, config 4 (CSR) 239 -> 229 us, config 5 (CSR)
// 6.83 -> 6.64 ms; one double per lane loses everywhere (30.1 us, 331 us, 8.0 ms).
template <int S, int VEC_>
struct Shape {
  static constexpr int VEC = VEC_;
  static constexpr int LPR = S / VEC;   // lanes per row
  static constexpr int RPW = 32 / LPR;  // rows per warp
};

template <int VEC>
struct Acc {
  double v[VEC];
};

// 8- or 16-byte loads/stores with cache-operator hints.
template <int VEC>
__device__ __forceinline__ Acc<VEC> load_gather(const double* p) {  // X rows: keep in L1/L2
  Acc<VEC> a;
  if constexpr (VEC == 2) {
    double2 t = __ldg(reinterpret_cast<const double2*>(p));
    a.v[0] = t.x;
    a.v[1] = t.y;
  } else {
    a.v[0] = __ldg(p);
  }
  return a;
}

template <int VEC>
__device__ __forceinline__ Acc<VEC> load_stream(const double* p) {  // Z, V: touched once
  Acc<VEC> a;
  if constexpr (VEC == 2) {
    double2 t = __ldcs(reinterpret_cast<const double2*>(p));
    a.v[0] = t.x;
    a.v[1] = t.y;
  } else {
    a.v[0] = __ldcs(p);
  }
  return a;
}

template <int VEC>
__device__ __forceinline__ void store_stream(double* p, const Acc<VEC>& a) {
  if constexpr (VEC == 2) {
    __stcs(reinterpret_cast<double2*>(p), make_double2(a.v[0], a.v[1]));
  } else {
    __stcs(p, a.v[0]);
  }
}

// NV > 0 (PACKED): row_ptr/col are those of the packed plan (col = column | value class << 28, off-diagonal
// entries only), val is the dense diagonal and vt the value table (packed.cuh).
// Value of class `cls` out of NV table entries: NV = 1 a constant, NV = 2 a register select.
template <int NV>
__device__ __forceinline__ double pick_val(unsigned cls, const PackedVals& vt) {
  if constexpr (NV == 1) {
    return vt.v[0];
  } else {
    return cls ? vt.v[1] : vt.v[0];
  }
}

template <int S, int VEC_, bool USE_Z, bool USE_V, int NV>
__global__ void __launch_bounds__(kThreads)
fused_step_kernel(int n, const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col,
                  const double* __restrict__ val, const double* __restrict__ X, const double* Z,
                  const double* V, double* Y, double p, double q, double r, double c,
                  int rows_per_cta, const PackedVals vt) {
  constexpr bool PACKED = NV > 0;
  using Sh = Shape<S, VEC_>;
  constexpr int VEC = Sh::VEC, LPR = Sh::LPR, RPW = Sh::RPW;
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  const int sl = lane % LPR;   // lane within the row group
  const int sub = lane / LPR;  // row group within the warp
  const long long cta_row0 = (long long)blockIdx.x * rows_per_cta;
  const int cta_row1 = (int)min((long long)n, cta_row0 + rows_per_cta);

  // Programmatic dependent launch: the next step's CTAs may be scheduled while this grid drains;
  // they load their row pointers and first entries (matrix data, never written) and then wait
  // for this grid to complete before they touch a block.
  asm volatile("griddepcontrol.launch_dependents;");
  bool waited = false;
  for (int base = (int)cta_row0 + warp * RPW; base < cta_row1; base += kWarps * RPW) {
    const int row = base + sub;
    const bool active = row < cta_row1;
    int e0 = 0, e1 = 0;
    if (active) {
      e0 = __ldg(row_ptr + row);
      e1 = __ldg(row_ptr + row + 1);
    }
    Acc<VEC> acc;
#pragma unroll
    for (int t = 0; t < VEC; ++t) acc.v[t] = 0.0;

    if constexpr (LPR == 1) {
      // one thread per row (S = 1, 2)
      if (!waited) {
        asm volatile("griddepcontrol.wait;" ::: "memory");
        waited = true;
      }
      for (int e = e0; e < e1; ++e) {
        int cj = __ldcs(col + e);
        double vj;
        if constexpr (PACKED) {
          vj = pick_val<NV>((unsigned)cj >> 28, vt);
          cj &= 0x0fffffff;
        } else {
          vj = __ldcs(val + e);
        }
        const Acc<VEC> x = load_gather<VEC>(X + (size_t)cj * S);
#pragma unroll
        for (int t = 0; t < VEC; ++t) acc.v[t] = fma(vj, x.v[t], acc.v[t]);
      }
    } else {
      const int len = e1 - e0;
      const int maxlen = __reduce_max_sync(0xffffffffu, len);
      // the entries of chunk i + 1 are loaded before the gathers of chunk i
      int cc_n = 0;
      double vv_n = 0.0;
      if (e0 + sl < e1) {
        cc_n = __ldcs(col + e0 + sl);
        if constexpr (!PACKED) vv_n = __ldcs(val + e0 + sl);
      }
      if (!waited) {
        asm volatile("griddepcontrol.wait;" ::: "memory");
        waited = true;
      }
      for (int off = 0; off < maxlen; off += LPR) {
        const int cc = cc_n;
        const double vv = vv_n;
        const int en = e0 + off + LPR + sl;
        cc_n = 0;
        vv_n = 0.0;
        if (en < e1) {
          cc_n = __ldcs(col + en);
          if constexpr (!PACKED) vv_n = __ldcs(val + en);
        }
        const int rem = len - off;  // entries of this row left in the chunk (may be <= 0)
#pragma unroll
        for (int j = 0; j < LPR; ++j) {
          int cj = __shfl_sync(0xffffffffu, cc, j, LPR);
          double vj;
          if constexpr (PACKED) {  // one shuffle per entry; the value is a table read
            vj = pick_val<NV>((unsigned)cj >> 28, vt);
            cj &= 0x0fffffff;
          } else {
            vj = __shfl_sync(0xffffffffu, vv, j, LPR);
          }
          if (j < rem) {
            const Acc<VEC> x = load_gather<VEC>(X + (size_t)cj * S + sl * VEC);
#pragma unroll
            for (int t = 0; t < VEC; ++t) acc.v[t] = fma(vj, x.v[t], acc.v[t]);
          }
        }
      }
    }

    if (active) {
      const size_t at = (size_t)row * S + sl * VEC;
      const Acc<VEC> xi = load_gather<VEC>(X + at);
      Acc<VEC> y;
      double qd = q;
      if constexpr (PACKED) qd = fma(p, __ldg(val + row), q);  // the dense diagonal
#pragma unroll
      for (int t = 0; t < VEC; ++t) y.v[t] = fma(p, acc.v[t], qd * xi.v[t]);
      if constexpr (USE_Z) {
        const Acc<VEC> z = load_stream<VEC>(Z + at);
#pragma unroll
        for (int t = 0; t < VEC; ++t) y.v[t] = fma(r, z.v[t], y.v[t]);
      }
      if constexpr (USE_V) {
        const Acc<VEC> v = load_stream<VEC>(V + at);
#pragma unroll
        for (int t = 0; t < VEC; ++t) y.v[t] = fma(c, v.v[t], y.v[t]);
      }
      store_stream<VEC>(Y + at, y);
    }
  }
}

// b_K = c_K V.
__global__ void __launch_bounds__(256) scale_copy_kernel(size_t len2, const double2* __restrict__ V,
                                                         double2* __restrict__ Y, double c) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < len2; i += stride) {
    double2 v = __ldcs(V + i);
    v.x *= c;
    v.y *= c;
    Y[i] = v;
  }
}

__global__ void scale_copy_tail_kernel(const double* V, double* Y, double c) { Y[0] = c * V[0]; }

template <int S, int VEC>
int launch_step_v(const polfed_ham* ham, double p, double q, double r, double c, const double* X,
                  const double* Z, const double* V, double* Y, cudaStream_t st) {
  using Sh = Shape<S, VEC>;
  const int n = (int)ham->n;
  if (n == 0) return POLFED_OK;
  const int rows_per_pass = kWarps * Sh::RPW;
  // about 4 passes per CTA, but never fewer than 24 CTAs per SM (measured on config 3, 184 756
  // rows: 24.9 us with 1 pass, 26.6 with 2, 30.8 with 3 -- a short kernel ends with a tail of
  // half-empty SMs, and small CTAs keep that tail short)
  int passes = 4;
  while (passes > 1 && (long long)rows_per_pass * passes * ham->sm_count * 24 > n) --passes;
  const int rows_per_cta = rows_per_pass * passes;
  const unsigned grid = (unsigned)((n + (long long)rows_per_cta - 1) / rows_per_cta);
  const bool uz = (r != 0.0), uv = (c != 0.0);
  PackedVals vt{};
  const PackedPlan* pk = ham->packed;
  if (pk)
    for (int i = 0; i < 16; ++i) vt.v[i] = pk->vals[i];
  const int nv = pk ? pk->n_vals : 0;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kThreads);
  cfg.stream = st;
  cudaLaunchAttribute attr{};
  attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr.val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = &attr;
  cfg.numAttrs = 1;
  const int32_t* pk_rp = pk ? pk->d_row_ptr : nullptr;
  const int32_t* pk_col = pk ? reinterpret_cast<const int32_t*>(pk->d_pcol) : nullptr;
  const double* pk_diag = pk ? pk->d_diag : nullptr;
  cudaError_t le = cudaSuccess;
#define POLFED_PK(UZ, UV, NV)                                                                     \
  le = cudaLaunchKernelEx(&cfg, fused_step_kernel<S, VEC, UZ, UV, NV>, n, pk_rp, pk_col, pk_diag, \
                          X, Z, V, Y, p, q, r, c, rows_per_cta, vt)
#define POLFED_GO(UZ, UV)                                                                         \
  if (nv == 1) POLFED_PK(UZ, UV, 1);                                                              \
  else if (nv == 2) POLFED_PK(UZ, UV, 2);                                                         \
  else                                                                                            \
    le = cudaLaunchKernelEx(&cfg, fused_step_kernel<S, VEC, UZ, UV, 0>, n, ham->d_row_ptr,        \
                            ham->d_col, ham->d_val, X, Z, V, Y, p, q, r, c, rows_per_cta, vt)
  if (uz && uv) { POLFED_GO(true, true); }
  else if (uz) { POLFED_GO(true, false); }
  else if (uv) { POLFED_GO(false, true); }
  else { POLFED_GO(false, false); }
#undef POLFED_GO
#undef POLFED_PK
  if (le != cudaSuccess) return fail(POLFED_ECUDA, "fused_step_kernel: %s", cudaGetErrorString(le));
  POLFED_LAUNCH_CHECK("fused_step_kernel");
  return POLFED_OK;
}

template <int S>
int launch_step(const polfed_ham* ham, double p, double q, double r, double c, const double* X,
                const double* Z, const double* V, double* Y, cudaStream_t st) {
  return launch_step_v<S, (S >= 2) ? 2 : 1>(ham, p, q, r, c, X, Z, V, Y, st);
}

}  // namespace

int dispatch_step(const polfed_ham* ham, int s, double p, double q, double r, double c,
                  const double* X, const double* Z, const double* V, double* Y, cudaStream_t st) {
  if (flip_supports(ham, s)) return flip_step(ham, s, p, q, r, c, X, Z, V, Y, st);
  switch (s) {
    case 1: return launch_step<1>(ham, p, q, r, c, X, Z, V, Y, st);
    case 2: return launch_step<2>(ham, p, q, r, c, X, Z, V, Y, st);
    case 4: return launch_step<4>(ham, p, q, r, c, X, Z, V, Y, st);
    case 8: return launch_step<8>(ham, p, q, r, c, X, Z, V, Y, st);
    case 16: return launch_step<16>(ham, p, q, r, c, X, Z, V, Y, st);
    case 32: return launch_step<32>(ham, p, q, r, c, X, Z, V, Y, st);
  }
  return fail(POLFED_EINVAL, "block size s=%d not in {1,2,4,8,16,32}", s);
}

namespace {

int scale_copy(size_t len, const double* V, double* Y, double c, int sm_count, cudaStream_t st) {
  if (len == 0) return POLFED_OK;
  const size_t len2 = len / 2;
  if (len2) {
    size_t want = (len2 + 255) / 256;
    unsigned grid = (unsigned)(want < (size_t)sm_count * 16 ? want : (size_t)sm_count * 16);
    scale_copy_kernel<<<grid, 256, 0, st>>>(len2, reinterpret_cast<const double2*>(V),
                                            reinterpret_cast<double2*>(Y), c);
  }
  if (len & 1) scale_copy_tail_kernel<<<1, 1, 0, st>>>(V + len - 1, Y + len - 1, c);
  POLFED_LAUNCH_CHECK("scale_copy_kernel");
  return POLFED_OK;
}

bool overlap(const void* a, size_t na, const void* b, size_t nb) {
  const char* x = static_cast<const char*>(a);
  const char* y = static_cast<const char*>(b);
  return x < y + nb && y < x + na;
}

}  // namespace
}  // namespace polfed

using polfed::fail;

extern "C" {

int polfed_fused_step(const polfed_ham* ham, int s, double p, double q, double r, double c,
                      const double* d_X, const double* d_Z, const double* d_V, double* d_Y,
                      void* stream) {
  if (!ham) return fail(POLFED_EINVAL, "polfed_fused_step: ham is NULL");
  if (!polfed::valid_block_size(s))
    return fail(POLFED_EINVAL, "polfed_fused_step: block size s=%d not in {1,2,4,8,16,32}", s);
  if (ham->n == 0) return POLFED_OK;
  if (!d_X || !d_Y || (r != 0.0 && !d_Z) || (c != 0.0 && !d_V))
    return fail(POLFED_EINVAL, "polfed_fused_step: NULL block");
  if (!polfed::aligned16(d_X) || !polfed::aligned16(d_Y) || (r != 0.0 && !polfed::aligned16(d_Z)) ||
      (c != 0.0 && !polfed::aligned16(d_V)))
    return fail(POLFED_EINVAL, "polfed_fused_step: blocks must be 16-byte aligned");
  const size_t bytes = (size_t)ham->n * s * sizeof(double);
  if (polfed::overlap(d_X, bytes, d_Y, bytes))
    return fail(POLFED_EINVAL, "polfed_fused_step: Y overlaps X");
  return polfed::dispatch_step(ham, s, p, q, r, c, d_X, d_Z, d_V, d_Y,
                               static_cast<cudaStream_t>(stream));
}

size_t polfed_filter_workspace_bytes(int64_t n, int s) {
  if (n < 0 || s < 1) return 0;
  return (size_t)2 * (size_t)n * (size_t)s * sizeof(double);
}

size_t polfed_filter_workspace_bytes_ham(const polfed_ham* ham, int s) {
  if (!ham || s < 1) return 0;
  if (polfed::tiled_supports(ham, s)) return polfed::tiled_workspace_bytes(ham, s);
  return polfed_filter_workspace_bytes(ham->n, s);
}

int polfed_filter_apply(const polfed_ham* ham, double a, double b, int K, const double* h_coeffs,
                        int s, const double* d_V, double* d_W, void* d_work, void* stream) {
  if (!ham) return fail(POLFED_EINVAL, "polfed_filter_apply: ham is NULL");
  if (!polfed::valid_block_size(s))
    return fail(POLFED_EINVAL, "polfed_filter_apply: block size s=%d not in {1,2,4,8,16,32}", s);
  if (K < 0) return fail(POLFED_EINVAL, "polfed_filter_apply: K=%d < 0", K);
  if (!h_coeffs) return fail(POLFED_EINVAL, "polfed_filter_apply: h_coeffs is NULL");
  if (!(b > 0.0)) return fail(POLFED_ERANGE, "polfed_filter_apply: b=%g must be > 0", b);
  if (ham->n == 0) return POLFED_OK;
  if (!d_V || !d_W || (K >= 1 && !d_work))
    return fail(POLFED_EINVAL, "polfed_filter_apply: NULL block");
  if (!polfed::aligned16(d_V) || !polfed::aligned16(d_W) || !polfed::aligned16(d_work))
    return fail(POLFED_EINVAL, "polfed_filter_apply: blocks must be 16-byte aligned");
  // the tiled sweeps move 32-byte pieces of V and W and bulk-copy 128-byte rows of the workspace
  if (K >= 1 && polfed::tiled_supports(ham, s) &&
      (((reinterpret_cast<uintptr_t>(d_V) | reinterpret_cast<uintptr_t>(d_W)) & 31u) != 0 ||
       (reinterpret_cast<uintptr_t>(d_work) & 127u) != 0))
    return fail(POLFED_EINVAL, "polfed_filter_apply: on a tiled or sector handle d_V and d_W must be "
                               "32-byte and d_work 128-byte aligned");
  const size_t len = (size_t)ham->n * s;
  const size_t bytes = len * sizeof(double);
  const size_t work_bytes = polfed_filter_workspace_bytes_ham(ham, s);
  if (polfed::overlap(d_V, bytes, d_W, bytes) ||
      (K >= 1 && (polfed::overlap(d_work, work_bytes, d_W, bytes) ||
                  polfed::overlap(d_work, work_bytes, d_V, bytes))))
    return fail(POLFED_EINVAL, "polfed_filter_apply: V, W and work must not overlap");
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  if (K == 0)  // W = c_0 V
    return polfed::scale_copy(len, d_V, d_W, h_coeffs[0], ham->sm_count, st);
  if (polfed::tiled_supports(ham, s))  // the alternating-layout pipeline of tiled.cuh
    return polfed::tiled_filter_apply(ham, a, b, K, h_coeffs, s, d_V, d_W, d_work, st);

  double* cur = static_cast<double*>(d_work);  // b_{k+1}
  double* old = cur + len;                     // b_{k+2}, overwritten by b_k
  int rc = polfed::scale_copy(len, d_V, cur, h_coeffs[K], ham->sm_count, st);  // b_K = c_K V
  if (rc) return rc;
  if (polfed::small_filter_supports(ham, s)) {  // one persistent kernel for all K steps
    rc = polfed::small_filter_apply(ham, a, b, K, h_coeffs, s, d_V, d_W, cur, old, st);
    if (rc != POLFED_ERANGE) return rc;
  }
  const double p2 = 2.0 / b, q2 = -2.0 * a / b;
  for (int k = K - 1; k >= 1; --k) {
    // b_k = 2 H~ b_{k+1} - b_{k+2} + c_k V; b_{K+1} = 0 is never read
    const double r = (k == K - 1) ? 0.0 : -1.0;
    rc = polfed::dispatch_step(ham, s, p2, q2, r, h_coeffs[k], cur, old, d_V, old, st);
    if (rc) return rc;
    double* t = cur;  // "Permutation" of Fig. 5: pointer swap only
    cur = old;
    old = t;
  }
  // W = H~ b_1 - b_2 + c_0 V  (b_2 = 0 when K == 1)
  return polfed::dispatch_step(ham, s, 1.0 / b, -a / b, K == 1 ? 0.0 : -1.0, h_coeffs[0], cur, old,
                               d_V, d_W, st);
}

int polfed_filter_apply_host(const polfed_ham* ham, double a, double b, int K,
                             const double* h_coeffs, int s, const double* h_V, double* h_W,
                             void* stream) {
  if (!ham) return fail(POLFED_EINVAL, "polfed_filter_apply_host: ham is NULL");
  if (!polfed::valid_block_size(s))
    return fail(POLFED_EINVAL, "polfed_filter_apply_host: bad block size s=%d", s);
  if (ham->n == 0) return POLFED_OK;
  if (!h_V || !h_W) return fail(POLFED_EINVAL, "polfed_filter_apply_host: NULL block");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t bytes = (size_t)ham->n * s * sizeof(double);
  const size_t pitch = (bytes + 127) / 128 * 128;  // every sub-buffer starts on a 128-byte boundary
  // V | W | work from the library's stream-ordered pool: after the first call the blocks are
  // reused, not allocated
  char* d_all = nullptr;
  POLFED_CUDA(polfed::scratch_alloc(reinterpret_cast<void**>(&d_all),
                                    2 * pitch + polfed_filter_workspace_bytes_ham(ham, s), st));
  double* d_V = reinterpret_cast<double*>(d_all);
  double* d_W = reinterpret_cast<double*>(d_all + pitch);
  void* d_work = d_all + 2 * pitch;
  int rc = POLFED_OK;
  cudaError_t e = cudaMemcpyAsync(d_V, h_V, bytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) {
    rc = polfed_filter_apply(ham, a, b, K, h_coeffs, s, d_V, d_W, d_work, stream);
    if (rc == POLFED_OK) e = cudaMemcpyAsync(h_W, d_W, bytes, cudaMemcpyDeviceToHost, st);
  }
  cudaFreeAsync(d_all, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (rc) return rc;
  if (e != cudaSuccess)
    return fail(POLFED_ECUDA, "polfed_filter_apply_host: %s", cudaGetErrorString(e));
  return POLFED_OK;
}

}  // extern "C"
