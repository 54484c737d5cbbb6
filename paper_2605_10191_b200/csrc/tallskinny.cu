// Tall-skinny fp64 kernels for block Lanczos on P(H~):
//   gram    C = Q^T B      full reorthogonalisation coefficients, A_k, Gram matrices
//   update  B = beta B + alpha Q C     W -= Q (Q^T W), Ritz back-map u = V t (Eq. 43), W R^-1
// PAPER.md:136-172 (Eq. 8-14), 364-382.  Q is "panel-blocked": n_panels blocks of n x S
// row-major, panel j at Q + j*panel_stride; B is one n x S block; C is (n_panels*S) x S
// row-major.  Both kernels stream Q exactly once.  Every reduction is in a fixed order (per-CTA
// partial results, then one pass that adds them by ascending CTA index), so H_L, the CholeskyQR
// factors and with them the iteration count of the eigen-solver are reproducible run to run.
// For s in {8, 16, 32} the Gram product runs on the fp64 tensor cores (mma.sync m8n8k4, operands
// straight from global memory into fragments); the shared-memory FMA kernel serves s < 8 and is
// the measured alternative (profiles/r02_reorth.md); with 4 panels or more one warp takes one panel and
// the warps of a CTA share the rows of B through L1 (gram_dmma_panels_kernel, profiles/r03_gram_panels.md).
#include <mutex>

#include "common.cuh"

namespace polfed {
namespace {

constexpr int kTsThreads = 256;
constexpr int kTileRows = 32;

// ---- C += Q_j^T B over a strided set of row tiles ---------------------------------------------
template <int S>
__global__ void __launch_bounds__(kTsThreads)
gram_kernel(long long n, const double* __restrict__ Q, size_t panel_stride,
            const double* __restrict__ B, double* __restrict__ partial) {
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
    if (o < OUT) partial[((size_t)blockIdx.x * gridDim.y + j) * OUT + o] = acc[t];
  }
}

// ---- the same product on the fp64 tensor cores ------------------------------------------------
// mma.sync.aligned.m8n8k4 (D = A B + C, A 8x4 row-major, B 4x8 column-major): lane l holds
// A[l/4][l%4], B[l%4][l/4] and C[l/4][2(l%4) + {0,1}].  With A = Q_j^T and B = B over four rows r,
// both fragments are element (r0 + l%4, tile * 8 + l/4) of their row-major blocks, so a warp
// instruction reads four 64-byte row pieces.  A warp owns all (S/8)^2 output tiles and walks
// over rows; the CTA adds its warps in warp order.
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

constexpr int kDmmaThreads = 128;

template <int S>
__global__ void __launch_bounds__(kDmmaThreads)
gram_dmma_kernel(long long n, const double* __restrict__ Q, size_t panel_stride,
                 const double* __restrict__ B, double* __restrict__ partial) {
  constexpr int T = S / 8, OUT = S * S, WARPS = kDmmaThreads / 32;
  __shared__ double red[WARPS][OUT];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int j = blockIdx.y;
  const double* Qj = Q + (size_t)j * panel_stride + (lane & 3) * S + (lane >> 2);
  const double* Bl = B + (lane & 3) * S + (lane >> 2);
  double acc[T][T][2];
#pragma unroll
  for (int m = 0; m < T; ++m)
#pragma unroll
    for (int c = 0; c < T; ++c) acc[m][c][0] = acc[m][c][1] = 0.0;
  // rows in groups of 4; group g -> warp (g mod all warps of this panel), ascending
  const long long groups = n / 4;
  const long long stride = (long long)gridDim.x * WARPS;
  for (long long g = (long long)blockIdx.x * WARPS + warp; g < groups; g += stride) {
    const size_t at = (size_t)g * 4 * S;
    double a[T], b[T];
#pragma unroll
    for (int m = 0; m < T; ++m) {
      a[m] = __ldg(Qj + at + m * 8);
      b[m] = __ldg(Bl + at + m * 8);
    }
#pragma unroll
    for (int m = 0; m < T; ++m)
#pragma unroll
      for (int c = 0; c < T; ++c) dmma(acc[m][c][0], acc[m][c][1], a[m], b[c]);
  }
  // the last n mod 4 rows: warp 0 of CTA 0, lanes of the missing rows feed zeros
  if (blockIdx.x == 0 && warp == 0 && groups * 4 < n) {
    const size_t at = (size_t)groups * 4 * S;
    const bool ok = groups * 4 + (lane & 3) < n;
    double a[T], b[T];
#pragma unroll
    for (int m = 0; m < T; ++m) {
      a[m] = ok ? __ldg(Qj + at + m * 8) : 0.0;
      b[m] = ok ? __ldg(Bl + at + m * 8) : 0.0;
    }
#pragma unroll
    for (int m = 0; m < T; ++m)
#pragma unroll
      for (int c = 0; c < T; ++c) dmma(acc[m][c][0], acc[m][c][1], a[m], b[c]);
  }
#pragma unroll
  for (int m = 0; m < T; ++m)
#pragma unroll
    for (int c = 0; c < T; ++c) {
      const int row = m * 8 + (lane >> 2), col = c * 8 + 2 * (lane & 3);
      red[warp][row * S + col] = acc[m][c][0];
      red[warp][row * S + col + 1] = acc[m][c][1];
    }
  __syncthreads();
  for (int o = threadIdx.x; o < OUT; o += kDmmaThreads) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) t += red[w][o];
    partial[((size_t)blockIdx.x * gridDim.y + j) * OUT + o] = t;
  }
}

// The same product for several panels at once, W read once per CTA (round 3; with one
// panel per CTA the rows of B were fetched once per panel, 1.6 x the algorithmic DRAM traffic at 8
// panels).  The four warps of a CTA take four DIFFERENT panels and walk the SAME row groups, so the
// 64-byte row pieces of B that the first warp brings into L1 serve the other three; each warp owns
// its panel's accumulators, so there is no reduction inside the CTA: partial sum (x, j) is written
// straight from the fragments.  Row group g -> CTA column (g mod gridDim.x), ascending: fixed order.
template <int S>
__global__ void __launch_bounds__(kDmmaThreads)
gram_dmma_panels_kernel(long long n, const double* __restrict__ Q, int n_panels, size_t panel_stride,
                        const double* __restrict__ B, double* __restrict__ partial) {
  constexpr int T = S / 8, OUT = S * S, WARPS = kDmmaThreads / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int j = blockIdx.y * WARPS + warp;
  if (j >= n_panels) return;
  const double* Qj = Q + (size_t)j * panel_stride + (lane & 3) * S + (lane >> 2);
  const double* Bl = B + (lane & 3) * S + (lane >> 2);
  double acc[T][T][2];
#pragma unroll
  for (int m = 0; m < T; ++m)
#pragma unroll
    for (int c = 0; c < T; ++c) acc[m][c][0] = acc[m][c][1] = 0.0;
  const long long groups = n / 4;
  for (long long g = blockIdx.x; g < groups; g += gridDim.x) {
    const size_t at = (size_t)g * 4 * S;
    double a[T], b[T];
#pragma unroll
    for (int m = 0; m < T; ++m) {
      a[m] = __ldg(Qj + at + m * 8);
      b[m] = __ldg(Bl + at + m * 8);
    }
#pragma unroll
    for (int m = 0; m < T; ++m)
#pragma unroll
      for (int c = 0; c < T; ++c) dmma(acc[m][c][0], acc[m][c][1], a[m], b[c]);
  }
  if (blockIdx.x == 0 && groups * 4 < n) {  // the last n mod 4 rows: missing rows feed zeros
    const size_t at = (size_t)groups * 4 * S;
    const bool ok = groups * 4 + (lane & 3) < n;
    double a[T], b[T];
#pragma unroll
    for (int m = 0; m < T; ++m) {
      a[m] = ok ? __ldg(Qj + at + m * 8) : 0.0;
      b[m] = ok ? __ldg(Bl + at + m * 8) : 0.0;
    }
#pragma unroll
    for (int m = 0; m < T; ++m)
#pragma unroll
      for (int c = 0; c < T; ++c) dmma(acc[m][c][0], acc[m][c][1], a[m], b[c]);
  }
  double* out = partial + ((size_t)blockIdx.x * n_panels + j) * OUT;
#pragma unroll
  for (int m = 0; m < T; ++m)
#pragma unroll
    for (int c = 0; c < T; ++c) {
      const int row = m * 8 + (lane >> 2), col = c * 8 + 2 * (lane & 3);
      *reinterpret_cast<double2*>(out + row * S + col) = make_double2(acc[m][c][0], acc[m][c][1]);
    }
}

// out[i] = sum over p = 0..count-1 (ascending) of partial[p * len + i]
__global__ void __launch_bounds__(256) sum_partials_kernel(int count, size_t len,
                                                           const double* __restrict__ partial,
                                                           double* __restrict__ out) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= len) return;
  double t = 0.0;
  for (int p = 0; p < count; ++p) t += partial[(size_t)p * len + i];
  out[i] = t;
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

// ---- the same update on the fp64 tensor cores --------------------------------------------------
// D (8 rows x 8 columns) += Q_j[8 rows][4 columns k0..k0+3] C_j[k0..k0+3][8 columns]: the A fragment
// of lane l is Q_j[r0 + l/4][k0 + l%4], the B fragment C_j[k0 + l%4][8c + l/4].  A warp owns
// kUpdGroups groups of 8 rows, so every C fragment (read through L1) feeds kUpdGroups mma.
constexpr int kUpdGroups = 4;

template <int S>
__global__ void __launch_bounds__(kDmmaThreads)
update_dmma_kernel(long long n, const double* __restrict__ Q, int n_panels, size_t panel_stride,
                   const double* __restrict__ C, double alpha, double beta, double* B) {
  constexpr int T = S / 8;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long base = ((long long)blockIdx.x * (kDmmaThreads / 32) + warp) * (8 * kUpdGroups);
  if (base >= n) return;
  double acc[kUpdGroups][T][2];
#pragma unroll
  for (int g = 0; g < kUpdGroups; ++g)
#pragma unroll
    for (int c = 0; c < T; ++c) acc[g][c][0] = acc[g][c][1] = 0.0;
  long long row[kUpdGroups];
#pragma unroll
  for (int g = 0; g < kUpdGroups; ++g) row[g] = base + g * 8 + (lane >> 2);
  for (int j = 0; j < n_panels; ++j) {
    const double* Qj = Q + (size_t)j * panel_stride + (lane & 3);
    const double* Cj = C + (size_t)j * S * S + (lane & 3) * S + (lane >> 2);
#pragma unroll 2
    for (int k0 = 0; k0 < S; k0 += 4) {
      double a[kUpdGroups], cf[T];
#pragma unroll
      for (int g = 0; g < kUpdGroups; ++g)
        a[g] = row[g] < n ? __ldg(Qj + (size_t)row[g] * S + k0) : 0.0;
#pragma unroll
      for (int c = 0; c < T; ++c) cf[c] = __ldg(Cj + k0 * S + c * 8);
#pragma unroll
      for (int g = 0; g < kUpdGroups; ++g)
#pragma unroll
        for (int c = 0; c < T; ++c) dmma(acc[g][c][0], acc[g][c][1], a[g], cf[c]);
    }
  }
#pragma unroll
  for (int g = 0; g < kUpdGroups; ++g) {
    if (row[g] >= n) continue;
#pragma unroll
    for (int c = 0; c < T; ++c) {
      double2* out = reinterpret_cast<double2*>(B + (size_t)row[g] * S + c * 8 + 2 * (lane & 3));
      double2 o = make_double2(0.0, 0.0);
      if (beta != 0.0) {
        o = *out;
        o.x *= beta;
        o.y *= beta;
      }
      o.x = fma(alpha, acc[g][c][0], o.x);
      o.y = fma(alpha, acc[g][c][1], o.y);
      *out = o;
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
    out[(size_t)blockIdx.x * S + b] = sum;  // per-CTA partial, added up in CTA order afterwards
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
  if (threadIdx.x == 0) {  // per-CTA partials, added up in CTA order afterwards
    out[2 * blockIdx.x] = red[0][0];
    out[2 * blockIdx.x + 1] = red[1][0];
  }
}

// Scratch for per-CTA partial results from the library's stream-ordered pool (common.cuh).
struct PoolBuf {
  double* p = nullptr;
  cudaStream_t st;
  explicit PoolBuf(cudaStream_t s) : st(s) {}
  cudaError_t alloc(size_t doubles) {
    return scratch_alloc(reinterpret_cast<void**>(&p), sizeof(double) * doubles, st);
  }
  ~PoolBuf() {
    if (p) cudaFreeAsync(p, st);
  }
};

int sum_partials(int count, size_t len, const double* partial, double* out, cudaStream_t st) {
  sum_partials_kernel<<<(unsigned)((len + 255) / 256), 256, 0, st>>>(count, len, partial, out);
  POLFED_LAUNCH_CHECK("sum_partials_kernel");
  return POLFED_OK;
}

// variant: 0 = automatic (tensor cores for S >= 8), 1 = shared-memory FMA kernel, 2 = tensor cores
template <int S>
int gram_launch(long long n, const double* Q, int n_panels, size_t stride, const double* B, double* C,
                int sm_count, int variant, cudaStream_t st) {
  const bool dmma_ok = S >= 8;
  const bool use_dmma = dmma_ok && variant != 1;
  if constexpr (S >= 8) {
    if (use_dmma && n_panels >= 4) {  // one warp per panel, B read once per CTA
      constexpr int WARPS = kDmmaThreads / 32;
      const int gy = (n_panels + WARPS - 1) / WARPS;
      int occ = 0;
      POLFED_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, gram_dmma_panels_kernel<S>,
                                                                kDmmaThreads, 0));
      const long long groups = n / 4;
      long long gxp = (long long)sm_count * (occ > 0 ? occ : 4) / gy;  // one wave of resident CTAs
      if (gxp > groups) gxp = groups;
      if (gxp < 1) gxp = 1;
      const size_t lenp = (size_t)n_panels * S * S;
      PoolBuf part(st);
      POLFED_CUDA(part.alloc((size_t)gxp * lenp));
      gram_dmma_panels_kernel<S><<<dim3((unsigned)gxp, (unsigned)gy), kDmmaThreads, 0, st>>>(
          n, Q, n_panels, stride, B, part.p);
      POLFED_LAUNCH_CHECK("gram_dmma_panels_kernel");
      return sum_partials((int)gxp, lenp, part.p, C, st);
    }
  }
  long long gx;
  if (use_dmma) {
    const long long groups = (n / 4 + kDmmaThreads / 32 - 1) / (kDmmaThreads / 32);
    gx = (long long)sm_count * 8 / n_panels;
    if (gx < 1) gx = 1;
    if (gx > groups) gx = groups > 0 ? groups : 1;
  } else {
    const long long n_tiles = (n + kTileRows - 1) / kTileRows;
    gx = (long long)sm_count * 8 / n_panels;
    if (gx < 1) gx = 1;
    if (gx > n_tiles) gx = n_tiles;
  }
  const size_t len = (size_t)n_panels * S * S;
  PoolBuf partial(st);
  POLFED_CUDA(partial.alloc((size_t)gx * len));
  dim3 grid((unsigned)gx, (unsigned)n_panels);
  if constexpr (S >= 8) {
    if (use_dmma) gram_dmma_kernel<S><<<grid, kDmmaThreads, 0, st>>>(n, Q, stride, B, partial.p);
  }
  if (!use_dmma) gram_kernel<S><<<grid, kTsThreads, 0, st>>>(n, Q, stride, B, partial.p);
  POLFED_LAUNCH_CHECK("gram_kernel");
  return sum_partials((int)gx, len, partial.p, C, st);
}

template <int S>
int update_launch(long long n, const double* Q, int n_panels, size_t stride, const double* C, double alpha,
                  double beta, double* B, cudaStream_t st) {
  if constexpr (S >= 8) {  // tensor cores, unless B is one of the panels (in-place W R^-1): the
                           // shared-memory kernel stages its rows before it writes them
    if (n_panels > 0 && (B + (size_t)n * S <= Q || B >= Q + (size_t)(n_panels - 1) * stride + (size_t)n * S)) {
      constexpr int ROWS_D = (kDmmaThreads / 32) * 8 * kUpdGroups;
      update_dmma_kernel<S><<<(unsigned)((n + ROWS_D - 1) / ROWS_D), kDmmaThreads, 0, st>>>(
          n, Q, n_panels, stride, C, alpha, beta, B);
      POLFED_LAUNCH_CHECK("update_dmma_kernel");
      return POLFED_OK;
    }
  }
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
  PoolBuf partial(st);
  POLFED_CUDA(partial.alloc((size_t)grid * S));
  residual_norm_kernel<S><<<grid, kTsThreads, 0, st>>>(n, A, B, e, partial.p);
  POLFED_LAUNCH_CHECK("residual_norm_kernel");
  return sum_partials((int)grid, S, partial.p, out, st);
}

// ---- the Gram product for callers that must not allocate (polfed_block_gram_static) ------------
// The per-CTA partial sums of gram_kernel / gram_dmma_kernel normally sit in a block taken from
// the library's stream-ordered pool.  Some callers cannot afford that: a solver that has already
// handed every free byte of HBM to its Krylov basis (any further cudaMalloc or pool growth then
// fails), a process running under a fixed device-memory budget (an MPS or scheduler limit), or a
// latency-bound loop that must not hit the implicit device-wide synchronisation of the CUDA
// allocator.  For them the partial sums go into this fixed array in the library's own device
// image.  It costs kStaticGramDoubles * 8 bytes = 4 MiB on every GPU that loads libpolfed.so, from
// load until the process exits.
//
// In host code `g_gram_static` is only a handle for the symbol, never a device address (a kernel
// given `g_gram_static` from the host would fault, or quietly use host memory where the GPU can
// reach it); static_gram_scratch() asks the runtime for the real address once per device, with
// that device current, and the launches below get that pointer.
constexpr size_t kStaticGramDoubles = POLFED_STATIC_GRAM_DOUBLES;
static __device__ __align__(256) double g_gram_static[kStaticGramDoubles];

std::mutex g_static_mu;
double* g_static_ptr[64] = {};  // by device ordinal; filled on the first call on that device

int static_gram_scratch(double** out) {
  int dev = 0;
  POLFED_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(POLFED_EINVAL, "polfed_block_gram_static: device ordinal %d", dev);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    double* ptr = nullptr;
    POLFED_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_gram_static));
    if (!ptr) return fail(POLFED_ECUDA, "polfed_block_gram_static: no device address for the static scratch");
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return POLFED_OK;
}

// gram_launch with the partial sums in `scratch` (kStaticGramDoubles doubles).  The grid is the one
// gram_launch would take, cut down until gx * n_panels * S * S partial sums fit; every slot that
// sum_partials reads is written by this call's own CTAs first (a CTA without rows writes zeros),
// so what an earlier call left in the array is never read and nothing has to be cleared.
template <int S>
int gram_launch_static(long long n, const double* Q, int n_panels, size_t stride, const double* B, double* C,
                       int sm_count, int variant, double* scratch, cudaStream_t st) {
  const size_t len = (size_t)n_panels * S * S;
  const bool use_dmma = S >= 8 && variant != 1;
  const long long work = use_dmma ? (n / 4 + kDmmaThreads / 32 - 1) / (kDmmaThreads / 32)
                                  : (n + kTileRows - 1) / kTileRows;
  long long gx = (long long)sm_count * 8 / n_panels;
  if (gx > work) gx = work;
  if (gx > (long long)(kStaticGramDoubles / len)) gx = (long long)(kStaticGramDoubles / len);
  if (gx < 1) gx = 1;
  dim3 grid((unsigned)gx, (unsigned)n_panels);
  if constexpr (S >= 8) {
    if (use_dmma) gram_dmma_kernel<S><<<grid, kDmmaThreads, 0, st>>>(n, Q, stride, B, scratch);
  }
  if (!use_dmma) gram_kernel<S><<<grid, kTsThreads, 0, st>>>(n, Q, stride, B, scratch);
  POLFED_LAUNCH_CHECK("gram_kernel (static scratch)");
  return sum_partials((int)gx, len, scratch, C, st);
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

constexpr int g_gram_variant = 0;

int ts_gram(int s, long long n, const double* Q, int n_panels, size_t stride, const double* B, double* d_C,
            int sm_count, cudaStream_t st) {
  if (n_panels <= 0 || n <= 0) return POLFED_OK;
  POLFED_BY_S(s, (gram_launch<S_>(n, Q, n_panels, stride, B, d_C, sm_count, g_gram_variant, st)));
}

int ts_gram_variant(int s, long long n, const double* Q, int n_panels, size_t stride, const double* B,
                    double* d_C, int sm_count, int variant, cudaStream_t st) {
  if (n_panels <= 0 || n <= 0) return POLFED_OK;
  POLFED_BY_S(s, (gram_launch<S_>(n, Q, n_panels, stride, B, d_C, sm_count, variant, st)));
}

int ts_gram_static(int s, long long n, const double* Q, int n_panels, size_t stride, const double* B,
                   double* d_C, int sm_count, int variant, double* scratch, cudaStream_t st) {
  POLFED_BY_S(s, (gram_launch_static<S_>(n, Q, n_panels, stride, B, d_C, sm_count, variant, scratch, st)));
}

int ts_update(int s, long long n, const double* Q, int n_panels, size_t stride, const double* d_C,
              double alpha, double beta, double* B, cudaStream_t st) {
  if (n <= 0) return POLFED_OK;
  POLFED_BY_S(s, (update_launch<S_>(n, Q, n_panels, stride, d_C, alpha, beta, B, st)));
}

int ts_residual_norms(int s, long long n, const double* A, const double* B, const double* d_e, double* d_out,
                      int sm_count, cudaStream_t st) {
  if (n <= 0) {
    POLFED_CUDA(cudaMemsetAsync(d_out, 0, sizeof(double) * (size_t)s, st));
    return POLFED_OK;
  }
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
  if (ham->n == 0) {
    POLFED_CUDA(cudaMemsetAsync(d_out2, 0, 2 * sizeof(double), st));
    return POLFED_OK;
  }
  const int grid = ham->sm_count * 8;
  PoolBuf partial(st);
  POLFED_CUDA(partial.alloc((size_t)grid * 2));
  moments_kernel<<<grid, 256, 0, st>>>(ham->n, ham->d_row_ptr, ham->d_col, ham->d_val, partial.p);
  POLFED_LAUNCH_CHECK("moments_kernel");
  return sum_partials(grid, 2, partial.p, d_out2, st);
}

}  // namespace polfed

using polfed::fail;

extern "C" {

int polfed_block_gram(int s, int64_t n, const double* d_Q, int n_panels, int64_t panel_stride,
                      const double* d_B, double* d_C, int variant, void* stream) {
  if (!polfed::valid_block_size(s)) return fail(POLFED_EINVAL, "polfed_block_gram: bad block size s=%d", s);
  if (n < 0 || n_panels < 0 || panel_stride < 0 || variant < 0 || variant > 2)
    return fail(POLFED_EINVAL, "polfed_block_gram: bad argument");
  if (n == 0 || n_panels == 0) return POLFED_OK;
  if (!d_Q || !d_B || !d_C || !polfed::aligned16(d_Q) || !polfed::aligned16(d_B) || !polfed::aligned16(d_C))
    return fail(POLFED_EINVAL, "polfed_block_gram: NULL or misaligned block");
  if (n_panels > 1 && panel_stride < n * s)
    return fail(POLFED_EINVAL, "polfed_block_gram: panel_stride %lld < n*s, the panels overlap",
                (long long)panel_stride);
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  return polfed::ts_gram_variant(s, n, d_Q, n_panels, (size_t)panel_stride, d_B, d_C, sms, variant,
                                 static_cast<cudaStream_t>(stream));
}

int polfed_block_gram_static(int s, int64_t n, const double* d_Q, int n_panels, int64_t panel_stride,
                             const double* d_B, double* d_C, int variant, void* stream) {
  if (!polfed::valid_block_size(s))
    return fail(POLFED_EINVAL, "polfed_block_gram_static: bad block size s=%d", s);
  if (n < 0 || n_panels < 0 || panel_stride < 0 || variant < 0 || variant > 2)
    return fail(POLFED_EINVAL, "polfed_block_gram_static: bad argument");
  if (n == 0 || n_panels == 0) return POLFED_OK;
  if ((long long)n_panels * s * s > (long long)POLFED_STATIC_GRAM_DOUBLES)
    return fail(POLFED_ERANGE,
                "polfed_block_gram_static: n_panels*s*s = %lld partial sums per CTA row exceed the static "
                "scratch of %d doubles (POLFED_STATIC_GRAM_DOUBLES); split the panels over several calls "
                "or use polfed_block_gram",
                (long long)n_panels * s * s, (int)POLFED_STATIC_GRAM_DOUBLES);
  if (!d_Q || !d_B || !d_C || !polfed::aligned16(d_Q) || !polfed::aligned16(d_B) || !polfed::aligned16(d_C))
    return fail(POLFED_EINVAL, "polfed_block_gram_static: NULL or misaligned block");
  if (n_panels > 1 && panel_stride < n * s)
    return fail(POLFED_EINVAL, "polfed_block_gram_static: panel_stride %lld < n*s, the panels overlap",
                (long long)panel_stride);
  double* scratch = nullptr;
  if (int rc = polfed::static_gram_scratch(&scratch)) return rc;
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  return polfed::ts_gram_static(s, n, d_Q, n_panels, (size_t)panel_stride, d_B, d_C, sms, variant, scratch,
                                static_cast<cudaStream_t>(stream));
}

int polfed_block_update(int s, int64_t n, const double* d_Q, int n_panels, int64_t panel_stride,
                        const double* d_C, double alpha, double beta, double* d_B, void* stream) {
  if (!polfed::valid_block_size(s)) return fail(POLFED_EINVAL, "polfed_block_update: bad block size s=%d", s);
  if (n < 0 || n_panels < 0 || panel_stride < 0) return fail(POLFED_EINVAL, "polfed_block_update: bad argument");
  if (n == 0) return POLFED_OK;
  if (!d_B || (n_panels > 0 && (!d_Q || !d_C)))
    return fail(POLFED_EINVAL, "polfed_block_update: NULL block");
  // the tensor-core kernel moves B in 16-byte pieces: a misaligned B would fault on the device
  if (!polfed::aligned16(d_B) || (n_panels > 0 && (!polfed::aligned16(d_Q) || !polfed::aligned16(d_C))))
    return fail(POLFED_EINVAL, "polfed_block_update: blocks must be 16-byte aligned");
  if (n_panels > 1 && panel_stride < n * s)
    return fail(POLFED_EINVAL, "polfed_block_update: panel_stride %lld < n*s, the panels overlap",
                (long long)panel_stride);
  return polfed::ts_update(s, n, d_Q, n_panels, (size_t)panel_stride, d_C, alpha, beta, d_B,
                           static_cast<cudaStream_t>(stream));
}

}  // extern "C"
