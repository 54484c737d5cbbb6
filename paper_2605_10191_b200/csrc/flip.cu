// The flip format (flip.cuh): plan construction and the fused step
//   Y = p H X + q X + r Z + c V        (Eq. 51 PAPER.md:427-431 with the rescaling of Eq. 31)
// for full-space models made of a dense 8 x 8 block on bits 0-2, two-bit flips with uniform
// amplitudes and an arbitrary diagonal.
#include <new>

#include "flip.cuh"

namespace polfed {
namespace {

constexpr int kFlipThreads = 256;

__device__ __forceinline__ double2 ld_keep(const double2* p) {  // X: read many times per step
  return __ldg(p);
}
__device__ __forceinline__ double2 ld_stream(const double2* p) {  // Z, V: read once
  double2 r;
  asm volatile("ld.global.cs.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(double2* p, double2 v) {
  asm volatile("st.global.cs.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// S/2 lanes own one block of 8 rows, 16 bytes (two columns) of every row each.
template <int S, bool USE_Z, bool USE_V>
__global__ void __launch_bounds__(kFlipThreads, 2)
    flip_step_kernel(long long n_blocks, const FlipTerms t, const double* __restrict__ diag,
                     double p, double q, double r, double c, const double2* __restrict__ X,
                     const double2* Z, const double2* __restrict__ V, double2* Y) {
  constexpr int LPB = S / 2;  // lanes per block = double2 per row
  const int li = threadIdx.x % LPB;
  // grid-stride over blocks: the grid sweeps the rows front to back, a moving window of X in L2
  // (a contiguous range per CTA instead was measured slower: 0.257 vs 0.218 ms on config 4)
  const long long groups = (long long)gridDim.x * (kFlipThreads / LPB);
  for (long long blk = (long long)blockIdx.x * (kFlipThreads / LPB) + threadIdx.x / LPB;
       blk < n_blocks; blk += groups) {
    const size_t row0 = (size_t)blk * kFlipBlockRows;
    double2 xo[kFlipBlockRows], acc[kFlipBlockRows];
#pragma unroll
    for (int i = 0; i < kFlipBlockRows; ++i) xo[i] = ld_keep(X + (row0 + i) * LPB + li);
#pragma unroll
    for (int i = 0; i < kFlipBlockRows; ++i) {  // diagonal + the dense block, in registers
      const double dg = __ldg(diag + row0 + i);
      acc[i].x = dg * xo[i].x;
      acc[i].y = dg * xo[i].y;
#pragma unroll
      for (int j = 0; j < kFlipBlockRows; ++j) {
        if (j == i) continue;
        const double m = t.dense[i * kFlipBlockRows + j];
        acc[i].x = fma(m, xo[j].x, acc[i].x);
        acc[i].y = fma(m, xo[j].y, acc[i].y);
      }
    }
    for (int f = 0; f < t.n_flips; ++f) {  // one partner block per flip term
      const size_t prow0 = (size_t)(blk ^ (long long)t.hi[f]) * kFlipBlockRows;
      const uint32_t lo = t.lo[f];
      const double amp = t.amp[f];
      double2 xp[kFlipBlockRows];
#pragma unroll
      for (int i = 0; i < kFlipBlockRows; ++i)
        xp[i] = ld_keep(X + (prow0 + ((uint32_t)i ^ lo)) * LPB + li);
#pragma unroll
      for (int i = 0; i < kFlipBlockRows; ++i) {
        acc[i].x = fma(amp, xp[i].x, acc[i].x);
        acc[i].y = fma(amp, xp[i].y, acc[i].y);
      }
    }
#pragma unroll
    for (int i = 0; i < kFlipBlockRows; ++i) {
      const size_t at = (row0 + i) * LPB + li;
      double2 y;
      y.x = fma(p, acc[i].x, q * xo[i].x);
      y.y = fma(p, acc[i].y, q * xo[i].y);
      if (USE_Z) {
        const double2 z = ld_stream(Z + at);
        y.x = fma(r, z.x, y.x);
        y.y = fma(r, z.y, y.y);
      }
      if (USE_V) {
        const double2 v = ld_stream(V + at);
        y.x = fma(c, v.x, y.x);
        y.y = fma(c, v.y, y.y);
      }
      st_stream(Y + at, y);
    }
  }
}

// diag[r] = the stored diagonal entry of row r of the CSR (always present, assemble.cu)
__global__ void __launch_bounds__(256) csr_diag_kernel(long long n, const int32_t* __restrict__ row_ptr,
                                                       const int32_t* __restrict__ col,
                                                       const double* __restrict__ val,
                                                       double* __restrict__ diag) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  double d = 0.0;
  for (int e = row_ptr[r]; e < row_ptr[r + 1]; ++e)
    if (col[e] == (int32_t)r) d += val[e];
  diag[r] = d;
}

template <int S>
int launch_flip(const polfed_ham* ham, double p, double q, double r, double c, const double* X,
                const double* Z, const double* V, double* Y, cudaStream_t st) {
  const FlipPlan* plan = ham->flip;
  const long long n_blocks = ham->n / kFlipBlockRows;
  const long long per_cta = kFlipThreads / (S / 2);
  long long want = (n_blocks + per_cta - 1) / per_cta;
  const long long cap = (long long)ham->sm_count * 2 * 8;  // a few waves of resident CTAs
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  const double2* X2 = reinterpret_cast<const double2*>(X);
  const double2* Z2 = reinterpret_cast<const double2*>(Z);
  const double2* V2 = reinterpret_cast<const double2*>(V);
  double2* Y2 = reinterpret_cast<double2*>(Y);
  const bool uz = r != 0.0, uv = c != 0.0;
  if (uz && uv)
    flip_step_kernel<S, true, true><<<grid, kFlipThreads, 0, st>>>(n_blocks, plan->terms,
                                                                   plan->d_diag, p, q, r, c, X2, Z2,
                                                                   V2, Y2);
  else if (uz)
    flip_step_kernel<S, true, false><<<grid, kFlipThreads, 0, st>>>(n_blocks, plan->terms,
                                                                    plan->d_diag, p, q, r, c, X2,
                                                                    Z2, V2, Y2);
  else if (uv)
    flip_step_kernel<S, false, true><<<grid, kFlipThreads, 0, st>>>(n_blocks, plan->terms,
                                                                    plan->d_diag, p, q, r, c, X2,
                                                                    Z2, V2, Y2);
  else
    flip_step_kernel<S, false, false><<<grid, kFlipThreads, 0, st>>>(n_blocks, plan->terms,
                                                                     plan->d_diag, p, q, r, c, X2,
                                                                     Z2, V2, Y2);
  POLFED_LAUNCH_CHECK("flip_step_kernel");
  return POLFED_OK;
}

}  // namespace

void destroy_flip_plan(FlipPlan* p) {
  if (!p) return;
  cudaFree(p->d_diag);
  delete p;
}

bool flip_supports(const polfed_ham* ham, int s) {
  return ham && ham->flip && (s == 8 || s == 16 || s == 32) && ham->n > 0;
}

int flip_step(const polfed_ham* ham, int s, double p, double q, double r, double c, const double* X,
              const double* Z, const double* V, double* Y, cudaStream_t st) {
  switch (s) {
    case 8: return launch_flip<8>(ham, p, q, r, c, X, Z, V, Y, st);
    case 16: return launch_flip<16>(ham, p, q, r, c, X, Z, V, Y, st);
    case 32: return launch_flip<32>(ham, p, q, r, c, X, Z, V, Y, st);
  }
  return fail(POLFED_EINVAL, "flip format: block size s=%d not in {8,16,32}", s);
}

// The plan of a handle whose CSR is already assembled (the diagonal is taken from it).
int build_flip_plan(const polfed_basis* basis, const std::vector<DevTerm>& terms, int dot_bits,
                    const double* h_dot, const polfed_ham* ham, cudaStream_t st, FlipPlan** out) {
  *out = nullptr;
  if (basis->n_up >= 0)
    return fail(POLFED_EINVAL, "flip format: needs the full 2^n space (n_up < 0)");
  if (basis->n_sites < kFlipBlockBits || basis->n_sites > 31)
    return fail(POLFED_EINVAL, "flip format: n_sites=%d not in [%d,31]", basis->n_sites,
                kFlipBlockBits);
  if (dot_bits > kFlipBlockBits)
    return fail(POLFED_EINVAL, "flip format: the dense block may act on at most %d bits",
                kFlipBlockBits);
  FlipPlan* p = new (std::nothrow) FlipPlan;
  if (!p) return fail(POLFED_ENOMEM, "flip format: host allocation failed");
  struct Guard {
    FlipPlan* p;
    ~Guard() { destroy_flip_plan(p); }
  } guard{p};
  FlipTerms& t = p->terms;
  t.n_flips = 0;
  for (double& m : t.dense) m = 0.0;
  if (dot_bits > 0) {  // embed the 2^dot_bits block: identity on the other low bits
    const int dd = 1 << dot_bits;
    for (int r = 0; r < kFlipBlockRows; ++r)
      for (int c = 0; c < kFlipBlockRows; ++c)
        if ((r >> dot_bits) == (c >> dot_bits))
          t.dense[r * kFlipBlockRows + c] = h_dot[(size_t)(r & (dd - 1)) * dd + (c & (dd - 1))];
  }
  for (const DevTerm& term : terms) {
    if (term.kind < POLFED_TERM_EXCH) continue;  // diagonal kinds: in the CSR diagonal
    if (term.kind != POLFED_TERM_XX)
      return fail(POLFED_EINVAL, "flip format: only XX off-diagonal terms (uniform amplitudes)");
    const uint32_t mask = (1u << term.i) | (1u << term.j);
    const uint32_t lo = mask & (kFlipBlockRows - 1), hi = mask >> kFlipBlockBits;
    if (hi == 0) {  // both bits inside a block: part of the dense 8 x 8
      for (uint32_t r = 0; r < (uint32_t)kFlipBlockRows; ++r)
        t.dense[r * kFlipBlockRows + (r ^ lo)] += term.amp;
      continue;
    }
    if (t.n_flips == kFlipMaxTerms)
      return fail(POLFED_EINVAL, "flip format: more than %d flip terms", kFlipMaxTerms);
    t.hi[t.n_flips] = hi;
    t.lo[t.n_flips] = lo;
    t.amp[t.n_flips] = term.amp;
    ++t.n_flips;
  }
  for (int r = 0; r < kFlipBlockRows; ++r) t.dense[r * kFlipBlockRows + r] = 0.0;
  for (int f = t.n_flips; f < kFlipMaxTerms; ++f) {
    t.hi[f] = t.lo[f] = 0u;
    t.amp[f] = 0.0;
  }
  const long long n = ham->n;
  POLFED_CUDA(cudaMalloc(&p->d_diag, sizeof(double) * (size_t)(n ? n : 1)));
  if (n > 0) {
    csr_diag_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, ham->d_row_ptr, ham->d_col,
                                                                 ham->d_val, p->d_diag);
    POLFED_LAUNCH_CHECK("csr_diag_kernel");
    POLFED_CUDA(cudaStreamSynchronize(st));
  }
  guard.p = nullptr;
  *out = p;
  return POLFED_OK;
}

}  // namespace polfed
