// Tall-skinny fp64 kernels for block Lanczos on P(H~):
//   gram    C = Q^T B      full reorthogonalisation coefficients, A_k, Gram matrices
//   update  B = beta B + alpha Q C     W -= Q (Q^T W), Ritz back-map u = V t (Eq. 43), W R^-1
// PAPER.md:136-172 (Eq. 8-14), 364-382.  Q is "panel-blocked": n_panels blocks of n x S
// row-major, panel j at Q + j*panel_stride; B is one n x S block; C is (n_panels*S) x S
// row-major.  Both kernels stream Q exactly once; they are bandwidth-bound like the filter,
// but run once per block step against K filter launches, so they are written for clarity
// (shared-memory tiles, register accumulators, one fp64 atomicAdd per output per CTA).
#include "common.cuh"

namespace polfed {
namespace {

constexpr int kTsThreads = 256;
constexpr int kTileRows = 32;

// ---- C += Q_j^T B over a strided set of row tiles ---------------------------------------------
template <int S>
__global__ void __launch_bounds__(kTsThreads)
gram_kernel(long long n, const double* __restrict__ Q, size_t panel_stride,
            const double* __restrict__ B, double* __restrict__ C) {
  constexpr int OUT = S * S;
  constexpr int PER = (OUT + kTsThreads - 1) / kTsThreads;  // outputs per thread
  __shared__ double As[kTileRows][S];
  __shared__ double Bs[kTileRows][S];
  const int j = blockIdx.y;
  const double* Qj = Q + (size_t)j * panel_stride;
  double acc[PER];
#pragma unroll
  for (int t = 0; t < PER; ++t) acc[t] = 0.0;
  const long long n_tiles = (n + kTileRows - 1) / kTileRows;
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const long long r0 = tile * kTileRows;
    const int rows = (int)min((long long)kTileRows, n - r0);
    for (int e = threadIdx.x; e < kTileRows * S; e += kTsThreads) {
      const int i = e / S, a = e % S;
      const bool ok = i < rows;
      As[i][a] = ok ? Qj[(size_t)(r0 + i) * S + a] : 0.0;
      Bs[i][a] = ok ? B[(size_t)(r0 + i) * S + a] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int t = 0; t < PER; ++t) {
      const int o = threadIdx.x + t * kTsThreads;
      if (o < OUT) {
        const int a = o / S, b = o % S;
        double sum = acc[t];
#pragma unroll 8
        for (int i = 0; i < kTileRows; ++i) sum = fma(As[i][a], Bs[i][b], sum);
        acc[t] = sum;
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int t = 0; t < PER; ++t) {
    const int o = threadIdx.x + t * kTsThreads;
    if (o < OUT) atomicAdd(C + (size_t)j * OUT + o, acc[t]);
  }
}

// ---- B = beta B + alpha sum_j Q_j C_j on one tile of rows per CTA -----------------------------
template <int S>
__global__ void __launch_bounds__(kTsThreads)
update_kernel(long long n, const double* Q, int n_panels, size_t panel_stride,
              const double* __restrict__ C, double alpha, double beta, double* B) {
  constexpr int GROUPS = kTsThreads / S;      // row groups per CTA
  constexpr int RPT = (kTileRows + GROUPS - 1) / GROUPS;  // rows per thread
  constexpr int ROWS = GROUPS * RPT;          // rows per CTA tile
  __shared__ double Qs[ROWS][S + 1];
  __shared__ double Cs[S][S];
  const int b = threadIdx.x % S, g = threadIdx.x / S;
  const long long r0 = (long long)blockIdx.x * ROWS;
  double acc[RPT];
#pragma unroll
  for (int t = 0; t < RPT; ++t) acc[t] = 0.0;
  for (int j = 0; j < n_panels; ++j) {
    const double* Qj = Q + (size_t)j * panel_stride;
    for (int e = threadIdx.x; e < ROWS * S; e += kTsThreads) {
      const int i = e / S, a = e % S;
      Qs[i][a] = (r0 + i < n) ? Qj[(size_t)(r0 + i) * S + a] : 0.0;
    }
    for (int e = threadIdx.x; e < S * S; e += kTsThreads) Cs[e / S][e % S] = C[(size_t)j * S * S + e];
    __syncthreads();
#pragma unroll 4
    for (int a = 0; a < S; ++a) {
      const double c = Cs[a][b];
#pragma unroll
      for (int t = 0; t < RPT; ++t) acc[t] = fma(Qs[g + t * GROUPS][a], c, acc[t]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int t = 0; t < RPT; ++t) {
    const long long row = r0 + g + t * GROUPS;
    if (row < n) {
      double* out = B + (size_t)row * S + b;
      const double old = (beta != 0.0) ? beta * *out : 0.0;
      *out = fma(alpha, acc[t], old);
    }
  }
}

// ---- per-column sum of squares of (A - B diag(e)) ----------------------------------------------
template <int S>
__global__ void __launch_bounds__(kTsThreads)
residual_norm_kernel(long long n, const double* __restrict__ A, const double* __restrict__ B,
                     const double* __restrict__ e, double* __restrict__ out) {
  constexpr int GROUPS = kTsThreads / S;
  __shared__ double red[kTsThreads];
  const int b = threadIdx.x % S, g = threadIdx.x / S;
  const double eb = e[b];
  double sum = 0.0;
  for (long long row = (long long)blockIdx.x * GROUPS + g; row < n; row += (long long)gridDim.x * GROUPS) {
    const double d = A[(size_t)row * S + b] - eb * B[(size_t)row * S + b];
    sum = fma(d, d, sum);
  }
  red[threadIdx.x] = sum;
  __syncthreads();
  if (g == 0) {
    for (int k = 1; k < GROUPS; ++k) sum += red[k * S + b];
    atomicAdd(out + b, sum);
  }
}

// ---- dst[:, dst_col0 + c] = src[:, cols[c]] (row-major, different leading dimensions) ----------
__global__ void __launch_bounds__(256) gather_columns_kernel(long long n, const double* __restrict__ src,
                                                             int src_ld, const int* __restrict__ cols,
                                                             int n_cols, double* __restrict__ dst,
                                                             int dst_ld, int dst_col0) {
  const long long total = n * (long long)n_cols;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const long long row = t / n_cols;
    const int c = (int)(t % n_cols);
    dst[(size_t)row * dst_ld + dst_col0 + c] = src[(size_t)row * src_ld + cols[c]];
  }
}

// ---- Tr H and sum of squared entries (Gaussian DOS, Eq. 34, R7) --------------------------------
__global__ void __launch_bounds__(256) moments_kernel(long long n, const int32_t* __restrict__ row_ptr,
                                                      const int32_t* __restrict__ col,
                                                      const double* __restrict__ val, double* out) {
  __shared__ double red[2][256];
  double tr = 0.0, sq = 0.0;
  for (long long row = (long long)blockIdx.x * blockDim.x + threadIdx.x; row < n;
       row += (long long)gridDim.x * blockDim.x) {
    for (int e = row_ptr[row]; e < row_ptr[row + 1]; ++e) {
      const double v = val[e];
      sq = fma(v, v, sq);
      if (col[e] == row) tr += v;
    }
  }
  red[0][threadIdx.x] = tr;
  red[1][threadIdx.x] = sq;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) {
      red[0][threadIdx.x] += red[0][threadIdx.x + w];
      red[1][threadIdx.x] += red[1][threadIdx.x + w];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    atomicAdd(out, red[0][0]);
    atomicAdd(out + 1, red[1][0]);
  }
}

template <int S>
int gram_launch(long long n, const double* Q, int n_panels, size_t stride, const double* B, double* C,
                int sm_count, cudaStream_t st) {
  const long long n_tiles = (n + kTileRows - 1) / kTileRows;
  long long gx = (long long)sm_count * 8 / (n_panels > 0 ? n_panels : 1);
  if (gx < 1) gx = 1;
  if (gx > n_tiles) gx = n_tiles;
  dim3 grid((unsigned)gx, (unsigned)n_panels);
  gram_kernel<S><<<grid, kTsThreads, 0, st>>>(n, Q, stride, B, C);
  POLFED_LAUNCH_CHECK("gram_kernel");
  return POLFED_OK;
}

template <int S>
int update_launch(long long n, const double* Q, int n_panels, size_t stride, const double* C, double alpha,
                  double beta, double* B, cudaStream_t st) {
  constexpr int GROUPS = kTsThreads / S;
  constexpr int ROWS = GROUPS * ((kTileRows + GROUPS - 1) / GROUPS);
  const unsigned grid = (unsigned)((n + ROWS - 1) / ROWS);
  update_kernel<S><<<grid, kTsThreads, 0, st>>>(n, Q, n_panels, stride, C, alpha, beta, B);
  POLFED_LAUNCH_CHECK("update_kernel");
  return POLFED_OK;
}

template <int S>
int resid_launch(long long n, const double* A, const double* B, const double* e, double* out, int sm_count,
                 cudaStream_t st) {
  constexpr int GROUPS = kTsThreads / S;
  long long want = (n + GROUPS - 1) / GROUPS;
  const unsigned grid = (unsigned)(want < (long long)sm_count * 8 ? want : (long long)sm_count * 8);
  residual_norm_kernel<S><<<grid, kTsThreads, 0, st>>>(n, A, B, e, out);
  POLFED_LAUNCH_CHECK("residual_norm_kernel");
  return POLFED_OK;
}

}  // namespace

#define POLFED_BY_S(s, CALL)                                                     \
  switch (s) {                                                                   \
    case 1: { constexpr int S_ = 1; return CALL; }                               \
    case 2: { constexpr int S_ = 2; return CALL; }                               \
    case 4: { constexpr int S_ = 4; return CALL; }                               \
    case 8: { constexpr int S_ = 8; return CALL; }                               \
    case 16: { constexpr int S_ = 16; return CALL; }                             \
    case 32: { constexpr int S_ = 32; return CALL; }                             \
    default: return fail(POLFED_EINVAL, "block size s=%d not in {1,2,4,8,16,32}", s); \
  }

int ts_gram(int s, long long n, const double* Q, int n_panels, size_t stride, const double* B, double* d_C,
            int sm_count, cudaStream_t st) {
  if (n_panels <= 0 || n <= 0) return POLFED_OK;
  POLFED_CUDA(cudaMemsetAsync(d_C, 0, sizeof(double) * (size_t)n_panels * s * s, st));
  POLFED_BY_S(s, (gram_launch<S_>(n, Q, n_panels, stride, B, d_C, sm_count, st)));
}

int ts_update(int s, long long n, const double* Q, int n_panels, size_t stride, const double* d_C,
              double alpha, double beta, double* B, cudaStream_t st) {
  if (n <= 0) return POLFED_OK;
  POLFED_BY_S(s, (update_launch<S_>(n, Q, n_panels, stride, d_C, alpha, beta, B, st)));
}

int ts_residual_norms(int s, long long n, const double* A, const double* B, const double* d_e, double* d_out,
                      int sm_count, cudaStream_t st) {
  POLFED_CUDA(cudaMemsetAsync(d_out, 0, sizeof(double) * (size_t)s, st));
  if (n <= 0) return POLFED_OK;
  POLFED_BY_S(s, (resid_launch<S_>(n, A, B, d_e, d_out, sm_count, st)));
}

int ts_gather_columns(long long n, const double* src, int src_ld, const int* d_cols, int n_cols, double* dst,
                      int dst_ld, int dst_col0, int sm_count, cudaStream_t st) {
  if (n <= 0 || n_cols <= 0) return POLFED_OK;
  gather_columns_kernel<<<sm_count * 8, 256, 0, st>>>(n, src, src_ld, d_cols, n_cols, dst, dst_ld, dst_col0);
  POLFED_LAUNCH_CHECK("gather_columns_kernel");
  return POLFED_OK;
}

int csr_moments(const polfed_ham* ham, double* d_out2, cudaStream_t st) {
  POLFED_CUDA(cudaMemsetAsync(d_out2, 0, 2 * sizeof(double), st));
  if (ham->n == 0) return POLFED_OK;
  moments_kernel<<<ham->sm_count * 8, 256, 0, st>>>(ham->n, ham->d_row_ptr, ham->d_col, ham->d_val, d_out2);
  POLFED_LAUNCH_CHECK("moments_kernel");
  return POLFED_OK;
}

}  // namespace polfed
