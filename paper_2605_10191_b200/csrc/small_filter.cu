// The whole Clenshaw recurrence of Eq. (51) PAPER.md:427-431 in ONE persistent kernel for small
// matrices (BASELINE configs 1 and 2: a fused launch moves 0.02-0.7 us of memory traffic against
// 5-6 us of launch latency; SURVEY section 7 "tiny configs are latency-bound").  Every thread owns
// a few (row, column) items and keeps its own entries of b_{k+1}, b_{k+2} and V in registers; the
// CSR entries of its rows are staged in shared memory once per launch; the blocks rotate by a
// pointer swap inside the kernel (Fig. 5).  n * s <= 4096: one CTA, both blocks in shared memory,
// __syncthreads between the steps.  n * s <= 262144: a cooperative grid (one CTA per SM), blocks
// in L2, a grid barrier between the steps.  The coefficients travel as kernel parameters, up to
// kSmallChunk recurrence steps per launch, so nothing is allocated and no device buffer beyond the
// caller's two-block workspace is needed.  DESIGN.md section 5e.
#include <cooperative_groups.h>

#include <algorithm>
#include <mutex>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace polfed {
namespace {

constexpr int kSmallChunk = 384;  // recurrence steps per launch (3 KB of kernel parameters)

struct SmallArgs {
  int n, s, n_steps;
  const int32_t* row_ptr;
  const int32_t* col;
  const double* val;
  const double* V;
  double* cur;  // b_{k+1}
  double* old;  // b_{k+2}, overwritten by b_k
  double* W;    // target of the final step (k = 0), if it is in this launch
  double a, b;
  int max_len;      // longest row of the matrix (entries staged per row slot)
  int first_has_z;  // the first step of the whole recurrence has no b_{k+2}
  int last_is_w;    // the last step of this launch is k = 0: factor 1, written to W
  double c[kSmallChunk];  // c[i]: coefficient of step i of this launch
};

constexpr int kSingleItems = 4096;    // single-CTA variant: both blocks in shared memory
constexpr int kSingleThreads = 1024;  // up to 4 items per thread
constexpr int kGridThreads = 512;     // cooperative variant (1024 when that saves a second item per thread)
constexpr int kGridItems = 262144;    // n * s limit of the cooperative variant (config 2: 102 960)

// Every thread owns the items it = tid + j * n_threads for the whole recurrence, so its own
// entries of b_{k+1}, b_{k+2} and V stay in registers, and the CSR entries of its rows are staged
// once per launch in shared memory ([entry][row slot]: the s threads of a row share a slot).  Per
// step it gathers b_{k+1} at its row's columns from shared memory and publishes b_k there.
// SINGLE: one CTA, both blocks in shared memory, __syncthreads between the steps.  Otherwise a
// cooperative grid of at most one CTA per SM: blocks in global memory (L2), a grid barrier
// between the steps.
template <bool SINGLE, int J>
__global__ void __launch_bounds__(SINGLE ? kSingleThreads : 2 * kGridThreads)
    small_filter_kernel(const SmallArgs a) {
  extern __shared__ double s_dyn[];
  const int tid = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_threads = gridDim.x * blockDim.x;
  const int items = a.n * a.s;
  const int rows_per_j = blockDim.x / a.s, slots = J * rows_per_j;
  double* s_blocks = s_dyn;                                      // SINGLE: two blocks
  double* ent_val = s_dyn + (SINGLE ? 2 * items : 0);            // [max_len][slots]
  int* ent_col = reinterpret_cast<int*>(ent_val + a.max_len * slots);
  double x_own[J], z_own[J], v_own[J];
  int len[J], col_j[J];
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const int it = tid + j * n_threads;
    x_own[j] = z_own[j] = v_own[j] = 0.0;
    len[j] = col_j[j] = 0;
    if (it < items) {
      const int row = it / a.s;
      col_j[j] = it - row * a.s;
      const int e0 = __ldg(a.row_ptr + row);
      len[j] = __ldg(a.row_ptr + row + 1) - e0;
      const int slot = j * rows_per_j + threadIdx.x / a.s;
      for (int k = col_j[j]; k < len[j]; k += a.s) {  // the row's threads share the copy
        ent_val[k * slots + slot] = __ldg(a.val + e0 + k);
        ent_col[k * slots + slot] = __ldg(a.col + e0 + k) * a.s;
      }
      x_own[j] = __ldcg(a.cur + it);
      if (a.first_has_z) z_own[j] = __ldcg(a.old + it);
      v_own[j] = __ldg(a.V + it);
    }
  }
  double* cur = a.cur;
  double* old = a.old;
  if (SINGLE) {
    cur = s_blocks;
    old = s_blocks + items;
#pragma unroll
    for (int j = 0; j < J; ++j)
      if (tid + j * n_threads < items) cur[tid + j * n_threads] = x_own[j];
  }
  __syncthreads();
  const double p2 = 2.0 / a.b, q2 = -2.0 * a.a / a.b;
  const int slot0 = threadIdx.x / a.s;
  for (int i = 0; i < a.n_steps; ++i) {
    const bool last = a.last_is_w && i + 1 == a.n_steps;
    const double p = last ? 0.5 * p2 : p2, q = last ? 0.5 * q2 : q2;
    const double r = (i == 0 && !a.first_has_z) ? 0.0 : -1.0;
    const double c = a.c[i];
    double* out = last ? a.W : old;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int it = tid + j * n_threads;
      const double* ev = ent_val + j * rows_per_j + slot0;
      const int* ec = ent_col + j * rows_per_j + slot0;
      const double* xc = cur + col_j[j];
      double acc = 0.0;
      if (SINGLE) {
#pragma unroll 4
        for (int k = 0; k < len[j]; ++k) acc = fma(ev[k * slots], xc[ec[k * slots]], acc);
      } else {
        // gathers from L2: ten independent loads in flight per round
        for (int k0 = 0; k0 < len[j]; k0 += 10) {
          double v[10], x[10];
#pragma unroll
          for (int u = 0; u < 10; ++u) {
            const bool on = k0 + u < len[j];
            v[u] = on ? ev[(k0 + u) * slots] : 0.0;
            x[u] = on ? __ldcg(xc + ec[(k0 + u) * slots]) : 0.0;
          }
#pragma unroll
          for (int u = 0; u < 10; ++u) acc = fma(v[u], x[u], acc);
        }
      }
      if (it < items) {
        double y = fma(p, acc, q * x_own[j]);
        y = fma(r, z_own[j], y);
        y = fma(c, v_own[j], y);
        if (SINGLE && !last) out[it] = y;
        else __stcg(out + it, y);
        z_own[j] = x_own[j];
        x_own[j] = y;
      }
    }
    double* t = cur;  // "Permutation" of Fig. 5
    cur = old;
    old = t;
    if (i + 1 < a.n_steps) {
      if (SINGLE) __syncthreads();
      else cg::this_grid().sync();
    }
  }
  if (SINGLE && !a.last_is_w) {
    // more launches follow: publish b_{k+1} (cur) and b_{k+2} (old) in the caller's blocks, in the
    // places the host expects after n_steps rotations
    double* g_cur = (a.n_steps & 1) ? a.old : a.cur;
    double* g_old = (a.n_steps & 1) ? a.cur : a.old;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int it = tid + j * n_threads;
      if (it < items) {
        g_cur[it] = x_own[j];
        g_old[it] = z_own[j];
      }
    }
  }
}

// Register variant for the smallest matrices (config 1: 924 rows, s = 1): rows of at most ML
// entries, at most J items per thread -- the entries themselves (value and the element offset of
// the gathered entry of b_{k+1}) stay in registers for the whole recurrence, padded with zero
// values, so a step is ML independent shared-memory gathers and two FMA chains per item with no
// loop, no entry loads and no length test.  One CTA, both blocks in shared memory.
constexpr int kRegThreads = 512;
constexpr int kRegMaxLen = 16;

template <int J, int ML>
__global__ void __launch_bounds__(kRegThreads) small_reg_kernel(const SmallArgs a) {
  extern __shared__ double s_dyn[];
  const int tid = threadIdx.x;
  const int items = a.n * a.s;
  double ev[J][ML];
  int ec[J][ML];
  double x_own[J], z_own[J], v_own[J];
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const int it = tid + j * kRegThreads;
    const bool valid = it < items;
    const int safe = valid ? it : 0;
    const int row = safe / a.s, colj = safe - row * a.s;
    const int e0 = __ldg(a.row_ptr + row);
    const int len = valid ? __ldg(a.row_ptr + row + 1) - e0 : 0;
#pragma unroll
    for (int k = 0; k < ML; ++k) {
      const bool on = k < len;
      ev[j][k] = on ? __ldg(a.val + e0 + k) : 0.0;
      ec[j][k] = on ? __ldg(a.col + e0 + k) * a.s + colj : safe;
    }
    x_own[j] = valid ? __ldcg(a.cur + it) : 0.0;
    z_own[j] = (valid && a.first_has_z) ? __ldcg(a.old + it) : 0.0;
    v_own[j] = valid ? __ldg(a.V + it) : 0.0;
  }
  double* cur = s_dyn;
  double* old = s_dyn + items;
#pragma unroll
  for (int j = 0; j < J; ++j)
    if (tid + j * kRegThreads < items) cur[tid + j * kRegThreads] = x_own[j];
  __syncthreads();
  const double p2 = 2.0 / a.b, q2 = -2.0 * a.a / a.b;
  for (int i = 0; i < a.n_steps; ++i) {
    const bool last = a.last_is_w && i + 1 == a.n_steps;
    const double p = last ? 0.5 * p2 : p2, q = last ? 0.5 * q2 : q2;
    const double r = (i == 0 && !a.first_has_z) ? 0.0 : -1.0;
    const double c = a.c[i];
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int it = tid + j * kRegThreads;
      double x[ML];
#pragma unroll
      for (int k = 0; k < ML; ++k) x[k] = cur[ec[j][k]];
      double acc0 = 0.0, acc1 = 0.0;
#pragma unroll
      for (int k = 0; k < ML; k += 2) {
        acc0 = fma(ev[j][k], x[k], acc0);
        acc1 = fma(ev[j][k + 1], x[k + 1], acc1);
      }
      double y = fma(p, acc0 + acc1, q * x_own[j]);
      y = fma(r, z_own[j], y);
      y = fma(c, v_own[j], y);
      if (it < items) {
        if (last) a.W[it] = y;
        else old[it] = y;
      }
      z_own[j] = x_own[j];
      x_own[j] = y;
    }
    double* t = cur;
    cur = old;
    old = t;
    if (i + 1 < a.n_steps) __syncthreads();
  }
  if (!a.last_is_w) {  // more launches follow (see small_filter_kernel)
    double* g_cur = (a.n_steps & 1) ? a.old : a.cur;
    double* g_old = (a.n_steps & 1) ? a.cur : a.old;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int it = tid + j * kRegThreads;
      if (it < items) {
        g_cur[it] = x_own[j];
        g_old[it] = z_own[j];
      }
    }
  }
}

__global__ void __launch_bounds__(256) max_row_len_kernel(long long n, const int32_t* __restrict__ rp,
                                                          int* out) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int v = r < n ? rp[r + 1] - rp[r] : 0;
  v = __reduce_max_sync(0xffffffffu, v);
  if ((threadIdx.x & 31) == 0) atomicMax(out, v);
}

const void* const kKernels[8] = {
    (const void*)small_filter_kernel<true, 1>,  (const void*)small_filter_kernel<true, 2>,
    (const void*)small_filter_kernel<true, 4>,  (const void*)small_filter_kernel<true, 8>,
    (const void*)small_filter_kernel<false, 1>, (const void*)small_filter_kernel<false, 2>,
    (const void*)small_filter_kernel<false, 4>, (const void*)small_filter_kernel<false, 8>};
const void* const kRegKernels[2] = {(const void*)small_reg_kernel<1, kRegMaxLen>,
                                    (const void*)small_reg_kernel<2, kRegMaxLen>};

}  // namespace

// True when the persistent kernel takes the recurrence of this handle and block size.
bool small_filter_supports(const polfed_ham* ham, int s) {
  if (!ham || ham->tiled || ham->flip || ham->max_row_len < 1) return false;
  return ham->n * (long long)s <= kGridItems;
}

// Longest row of a CSR matrix (polfed_ham_from_csr records it in the handle).  Runs on `st` and
// synchronises it.
int csr_max_row_len(long long n, const int32_t* d_row_ptr, int* out, cudaStream_t st) {
  *out = 0;
  if (n < 1) return POLFED_OK;
  int* d_max = nullptr;
  POLFED_CUDA(cudaMalloc(&d_max, sizeof(int)));
  cudaError_t e = cudaMemsetAsync(d_max, 0, sizeof(int), st);
  if (e == cudaSuccess) {
    max_row_len_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, d_row_ptr, d_max);
    e = cudaMemcpyAsync(out, d_max, sizeof(int), cudaMemcpyDeviceToHost, st);
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_max);
  if (e != cudaSuccess) return fail(POLFED_ECUDA, "csr_max_row_len: %s", cudaGetErrorString(e));
  return POLFED_OK;
}

// cur = c_K V has been written by the caller; runs steps k = K-1 .. 0.
int small_filter_apply(const polfed_ham* ham, double a_, double b_, int K, const double* c, int s,
                       const double* d_V, double* d_W, double* cur, double* old, cudaStream_t st) {
  constexpr int kSmemCap = 200 * 1024;
  // The shared-memory opt-in of a kernel and the cooperative-launch capability belong to a device,
  // not to the process: set / query them once per device ordinal (any thread may get here first).
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static int coop_of[kMaxDev];
  static bool ready[kMaxDev] = {};
  int dev = 0, coop = 0;
  POLFED_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) return POLFED_ERANGE;  // caller: single launches
  {
    std::lock_guard<std::mutex> lock(mu);
    if (!ready[dev]) {
      POLFED_CUDA(cudaDeviceGetAttribute(&coop_of[dev], cudaDevAttrCooperativeLaunch, dev));
      for (int v = 0; v < 8; ++v)
        POLFED_CUDA(cudaFuncSetAttribute(kKernels[v], cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         kSmemCap));
      ready[dev] = true;
    }
    coop = coop_of[dev];
  }
  const int items = (int)ham->n * s;
  const bool single = items <= kSingleItems;
  const bool in_regs = items <= 2 * kRegThreads && ham->max_row_len <= kRegMaxLen;
  if (!single && !coop) return POLFED_ERANGE;  // caller: single launches
  // cooperative variant: 1024-thread CTAs when 512-thread CTAs would leave threads with two items
  const int grid_threads = items > kGridThreads * ham->sm_count ? 2 * kGridThreads : kGridThreads;
  const int threads = single ? kSingleThreads : grid_threads;
  const int grid = single ? 1 : std::min((items + grid_threads - 1) / grid_threads, ham->sm_count);
  const int j_used = (items + grid * threads - 1) / (grid * threads);
  int jlog = 0;  // items per thread of the instantiation: 1, 2, 4 or 8
  while ((1 << jlog) < j_used) ++jlog;
  const size_t smem = (single ? 2 * (size_t)items * sizeof(double) : 0) +
                      ((size_t)1 << jlog) * (threads / s) * ham->max_row_len * 12 + 16;
  if (jlog > 3 || smem > (size_t)kSmemCap) return POLFED_ERANGE;  // caller: single launches
  const void* kernel = kKernels[(single ? 0 : 4) + jlog];
  if (in_regs) kernel = kRegKernels[items > kRegThreads];

  SmallArgs args{};
  args.n = (int)ham->n;
  args.s = s;
  args.row_ptr = ham->d_row_ptr;
  args.col = ham->d_col;
  args.val = ham->d_val;
  args.V = d_V;
  args.W = d_W;
  args.a = a_;
  args.b = b_;
  args.max_len = ham->max_row_len;
  for (int k = K - 1; k >= 0;) {  // launches of up to kSmallChunk steps, k descending
    const int n_steps = std::min(k + 1, kSmallChunk);
    args.n_steps = n_steps;
    args.cur = cur;
    args.old = old;
    args.first_has_z = (k != K - 1);
    args.last_is_w = (k - n_steps + 1 == 0);
    for (int i = 0; i < n_steps; ++i) args.c[i] = c[k - i];
    void* params[] = {&args};
    if (in_regs)
      POLFED_CUDA(cudaLaunchKernel(kernel, dim3(1), dim3(kRegThreads), params,
                                   2 * (size_t)items * sizeof(double), st));
    else if (single)
      POLFED_CUDA(cudaLaunchKernel(kernel, dim3(1), dim3(kSingleThreads), params, smem, st));
    else {
      const cudaError_t le = cudaLaunchCooperativeKernel(kernel, dim3((unsigned)grid),
                                                         dim3((unsigned)threads), params, smem, st);
      // a device (or an MPS / green-context share of one) that cannot hold the whole grid at once:
      // nothing has run yet on the first chunk, so the caller can still take the single launches
      if (k == K - 1 && (le == cudaErrorCooperativeLaunchTooLarge || le == cudaErrorInvalidValue ||
                         le == cudaErrorLaunchOutOfResources)) {
        (void)cudaGetLastError();
        return POLFED_ERANGE;
      }
      POLFED_CUDA(le);
    }
    if (n_steps & 1) std::swap(cur, old);  // the kernel's rotation, seen from the host
    k -= n_steps;
  }
  return POLFED_OK;
}

}  // namespace polfed
