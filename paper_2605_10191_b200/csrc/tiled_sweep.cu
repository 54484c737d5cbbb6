// The tiled hot path (tiled.cuh): one persistent kernel per Clenshaw step.  A CTA takes a tile
// (a contiguous run of positions that share their high bits), pulls its 16-column panel of
// b_{k+1} into shared memory with one bulk copy, finishes b_k from shared-memory gathers, parks
// b_k in an L2-resident scratch, pulls it back as the new shared tile and starts P_{k-1} from it.
// Eq. (51) PAPER.md:427-431 with the rescaling of Eq. (31); see tiled.cuh for the algebra.
//
// Thread mapping.  Four lanes own one 128-byte panel row, 32 contiguous bytes each, so every
// global access of a row is one 256-bit instruction per lane and one full line per row.  In
// shared memory the same 32 bytes are read as two 16-byte chunks; the rows a warp works on
// alternate the order of the two (even row slots low chunk first, odd slots high chunk first),
// so that the two rows of a quarter-warp always hit disjoint banks whatever rows they gather.
#include "tiled.cuh"

namespace polfed {
namespace {

enum { MODE_STEP = 0, MODE_INIT = 1, MODE_LAST = 2 };

constexpr int kWarps = kTileThreads / 32;
constexpr int kRowsPerIter = 8;  // rows per warp iteration

struct SweepArgs {
  long long n;
  int n_tiles, n_panels, max_tile_rows;
  const int32_t* tile_row0;
  const int32_t* tile_rec0;
  const uint32_t* records;  // kTileRecWords words per class row, position order
  const double* diag;       // [n]
  const int32_t* cc_col;    // [n_cross][n]
  const double* cc_val;     // [n_cross][n]
  int n_cross;
  const int32_t* dst_map;   // position -> output row (other layout, or natural for MODE_LAST)
  double coef[kTileMaxCoef];
  const double* X1;  // b_{k+1}, panel-major, this layout
  const double* Pk;  // partial b_k
  const double* V;   // V in this layout
  double* Bout;      // b_k, other layout
  double* Pout;      // partial b_{k-1}, other layout
  double* W;         // MODE_LAST: row-major n x w_ld output in the caller's row order
  int w_ld;
  double* scratch;   // per CTA: max_tile_rows x 16 doubles
  int* counter;
  double cK;              // MODE_INIT: b_K = cK V
  double pf;              // finishing scalar p_k
  double ps, qs, rs, cs;  // starting scalars of step k-1
  int mode;
};

struct D4 {
  double x, y, z, w;  // x,y = low 16-byte chunk, z,w = high chunk of a lane's 32 bytes
};

__device__ __forceinline__ D4 ldg256(const double* p) {  // read-only data, default caching
  D4 r;
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ D4 ldg256_stream(const double* p) {  // touched once
  D4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void stg256(double* p, const D4& r) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(r.x), "d"(r.y), "d"(r.z),
               "d"(r.w)
               : "memory");
}
__device__ __forceinline__ void stg256_stream(double* p, const D4& r) {
  asm volatile("st.global.L1::no_allocate.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(r.x),
               "d"(r.y), "d"(r.z), "d"(r.w)
               : "memory");
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async;" ::: "memory");
}

// One thread: bulk-copy `bytes` (a multiple of 128) from global to shared in <= 32 KB pieces.
__device__ __forceinline__ void tile_load(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
  mbar_expect_tx(bar, bytes);
  for (unsigned at = 0; at < bytes; at += 32768u) {
    const unsigned len = min(32768u, bytes - at);
    bulk_g2s(static_cast<char*>(dst) + at, static_cast<const char*>(src) + at, len, bar);
  }
}

template <int NC>
__device__ __forceinline__ double pick_coef(uint32_t cls, const double (&coef)[kTileMaxCoef]) {
  double cf = coef[0];
  if (NC == 2) {
    if (cls & 1u) cf = coef[1];
  } else if (NC > 2) {
    if (cls == 1u) cf = coef[1];
    if (cls == 2u) cf = coef[2];
    if (cls == 3u) cf = coef[3];
  }
  return cf;
}

__device__ __forceinline__ void hop_fma(double cf, uint32_t sign_bit31, uint32_t off,
                                        const unsigned char* __restrict__ x_first,
                                        const unsigned char* __restrict__ x_second, double2& acc_f,
                                        double2& acc_s) {
  cf = __hiloint2double(__double2hiint(cf) ^ (int)(sign_bit31 & 0x80000000u), __double2loint(cf));
  const double2 xa = *reinterpret_cast<const double2*>(x_first + off);
  const double2 xb = *reinterpret_cast<const double2*>(x_second + off);
  acc_f.x = fma(cf, xa.x, acc_f.x);
  acc_f.y = fma(cf, xa.y, acc_f.y);
  acc_s.x = fma(cf, xb.x, acc_s.x);
  acc_s.y = fma(cf, xb.y, acc_s.y);
}

// All in-tile neighbours of the row whose record quarter this lane holds (rq); max_deg is
// warp-uniform, shorter rows run into entries that point at the zero row.
template <int NC>
__device__ __forceinline__ void tile_hops(const uint4 rq, int max_deg,
                                          const unsigned char* __restrict__ x_first,
                                          const unsigned char* __restrict__ x_second,
                                          const double (&coef)[kTileMaxCoef], double2& acc_f,
                                          double2& acc_s) {
#pragma unroll
  for (int w = 1; w <= kTileMaxDeg / 2; ++w) {
    if (2 * (w - 1) >= max_deg) break;
    const uint32_t mine = (w & 3) == 0 ? rq.x : (w & 3) == 1 ? rq.y : (w & 3) == 2 ? rq.z : rq.w;
    const uint32_t word = __shfl_sync(0xffffffffu, mine, w >> 2, 4);
    hop_fma(pick_coef<NC>(word & 3u, coef), word << 1, word & 0x3ff80u, x_first, x_second, acc_f,
            acc_s);
    hop_fma(pick_coef<NC>((word >> 2) & 3u, coef), word, (word >> 11) & 0x3ff80u, x_first,
            x_second, acc_f, acc_s);
  }
}

// (first, second) accumulators of a lane -> (low, high) chunk order of its 32 bytes.
__device__ __forceinline__ D4 to_lohi(const double2 f, const double2 s, bool odd) {
  D4 r;
  r.x = odd ? s.x : f.x;
  r.y = odd ? s.y : f.y;
  r.z = odd ? f.x : s.x;
  r.w = odd ? f.y : s.y;
  return r;
}

template <int NC>
__global__ void __launch_bounds__(kTileThreads, 1) tiled_sweep_kernel(const SweepArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];  // (max_tile_rows + 1) x 128 B
  __shared__ uint64_t bar;
  __shared__ int s_tile;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int q = lane & 3, slot = lane >> 2;
  const bool odd = slot & 1;
  const unsigned char* x_first = smem_raw + 32 * q + (odd ? 16 : 0);
  const unsigned char* x_second = smem_raw + 32 * q + (odd ? 0 : 16);
  if (tid == 0) mbar_init(&bar, 1);
  __syncthreads();
  unsigned parity = 0;
  double* scratch = a.scratch + (size_t)blockIdx.x * a.max_tile_rows * kTilePanel;
  const size_t panel_stride = (size_t)a.n * kTilePanel;  // doubles per panel
  const double2 zero2 = make_double2(0.0, 0.0);

  for (;;) {
    if (tid == 0) s_tile = atomicAdd(a.counter, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= a.n_tiles) break;
    const int row0 = __ldg(a.tile_row0 + tile);
    const int nrows = __ldg(a.tile_row0 + tile + 1) - row0;
    const uint4* rec = reinterpret_cast<const uint4*>(a.records) +
                       (size_t)__ldg(a.tile_rec0 + tile) * 4;
    if (tid < 8) reinterpret_cast<double2*>(smem_raw)[nrows * 8 + tid] = zero2;  // the zero row
    const int first_pos = warp * kRowsPerIter + slot;
    __syncthreads();

    for (int panel = 0; panel < a.n_panels; ++panel) {
      const double* X1 = a.X1 + panel * panel_stride;
      const double* Pk = a.Pk + panel * panel_stride;
      const double* V = a.V + panel * panel_stride;
      double* Bout = a.Bout + panel * panel_stride;
      double* Pout = a.Pout + panel * panel_stride;

      uint4 rq_next = make_uint4(0u, 0u, 0u, 0u);
      if (first_pos < nrows) rq_next = __ldg(rec + (size_t)first_pos * 4 + q);
      if (a.mode != MODE_INIT) {
        if (tid == 0) tile_load(smem_raw, X1 + (size_t)row0 * kTilePanel, (unsigned)nrows * 128u, &bar);
        mbar_wait(&bar, parity);
        parity ^= 1u;
      }

      // ---- phase 2: b_k = P_k + p_k (O_l + DM) b_{k+1} -----------------------------------------
      for (int base = warp * kRowsPerIter; base < nrows; base += kWarps * kRowsPerIter) {
        const int pos = base + slot;
        const bool active = pos < nrows;
        const size_t row = (size_t)row0 + pos;
        const uint4 rq = rq_next;
        {
          const int pos_n = pos + kWarps * kRowsPerIter;
          if (pos_n < nrows) rq_next = __ldg(rec + (size_t)pos_n * 4 + q);
        }
        int dst = 0;
        if (active) dst = __ldg(a.dst_map + row);
        D4 b;
        if (a.mode == MODE_INIT) {
          b.x = b.y = b.z = b.w = 0.0;
          if (active) {
            const D4 v = ldg256_stream(V + row * kTilePanel + 4 * q);
            b.x = a.cK * v.x;
            b.y = a.cK * v.y;
            b.z = a.cK * v.z;
            b.w = a.cK * v.w;
          }
        } else {
          D4 pk;
          pk.x = pk.y = pk.z = pk.w = 0.0;
          double dg = 0.0;
          int cc[kTileMaxCross];
          double cv[kTileMaxCross];
#pragma unroll
          for (int j = 0; j < kTileMaxCross; ++j) {
            cc[j] = -1;
            cv[j] = 0.0;
          }
          if (active) {
            pk = ldg256_stream(Pk + row * kTilePanel + 4 * q);
            dg = __ldg(a.diag + row);
#pragma unroll
            for (int j = 0; j < kTileMaxCross; ++j)
              if (j < a.n_cross) {
                cc[j] = __ldg(a.cc_col + (size_t)j * a.n + row);
                cv[j] = __ldg(a.cc_val + (size_t)j * a.n + row);
              }
          }
          const int deg = __shfl_sync(0xffffffffu, (int)rq.x, 0, 4);
          const int max_deg = __reduce_max_sync(0xffffffffu, active ? deg : 0);
          double2 acc_f = zero2, acc_s = zero2;
          tile_hops<NC>(rq, max_deg, x_first, x_second, a.coef, acc_f, acc_s);
          if (active) {  // diagonal: own row of the shared tile
            const double2 oa = *reinterpret_cast<const double2*>(x_first + (size_t)pos * 128);
            const double2 ob = *reinterpret_cast<const double2*>(x_second + (size_t)pos * 128);
            acc_f.x = fma(dg, oa.x, acc_f.x);
            acc_f.y = fma(dg, oa.y, acc_f.y);
            acc_s.x = fma(dg, ob.x, acc_s.x);
            acc_s.y = fma(dg, ob.y, acc_s.y);
          }
          D4 acc = to_lohi(acc_f, acc_s, odd);
#pragma unroll
          for (int j = 0; j < kTileMaxCross; ++j)  // hops across the cut: other tiles, from L2
            if (cc[j] >= 0) {
              const D4 g = ldg256(X1 + (size_t)cc[j] * kTilePanel + 4 * q);
              acc.x = fma(cv[j], g.x, acc.x);
              acc.y = fma(cv[j], g.y, acc.y);
              acc.z = fma(cv[j], g.z, acc.z);
              acc.w = fma(cv[j], g.w, acc.w);
            }
          b.x = fma(a.pf, acc.x, pk.x);
          b.y = fma(a.pf, acc.y, pk.y);
          b.z = fma(a.pf, acc.z, pk.z);
          b.w = fma(a.pf, acc.w, pk.w);
        }
        if (active) {
          if (a.mode == MODE_LAST) {
            stg256_stream(a.W + (size_t)dst * a.w_ld + panel * kTilePanel + 4 * q, b);
          } else {
            stg256_stream(Bout + (size_t)dst * kTilePanel + 4 * q, b);
            stg256(scratch + (size_t)pos * kTilePanel + 4 * q, b);
          }
        }
      }
      if (a.mode == MODE_LAST) {
        __syncthreads();  // the next bulk copy overwrites the tile
        continue;
      }

      // ---- b_k becomes the shared tile ------------------------------------------------------
      if (first_pos < nrows) rq_next = __ldg(rec + (size_t)first_pos * 4 + q);
      __threadfence_block();
      fence_proxy_async();
      __syncthreads();
      if (tid == 0) tile_load(smem_raw, scratch, (unsigned)nrows * 128u, &bar);
      mbar_wait(&bar, parity);
      parity ^= 1u;

      // ---- phase 3: P_{k-1} = c_{k-1} V + p_{k-1} O_l b_k + q_{k-1} b_k + r b_{k+1} ------------
      for (int base = warp * kRowsPerIter; base < nrows; base += kWarps * kRowsPerIter) {
        const int pos = base + slot;
        const bool active = pos < nrows;
        const size_t row = (size_t)row0 + pos;
        const uint4 rq = rq_next;
        {
          const int pos_n = pos + kWarps * kRowsPerIter;
          if (pos_n < nrows) rq_next = __ldg(rec + (size_t)pos_n * 4 + q);
        }
        D4 x1, v;
        x1.x = x1.y = x1.z = x1.w = 0.0;
        v = x1;
        int dst = 0;
        if (active) {
          dst = __ldg(a.dst_map + row);
          if (a.rs != 0.0) x1 = ldg256(X1 + row * kTilePanel + 4 * q);
          if (a.cs != 0.0) v = ldg256_stream(V + row * kTilePanel + 4 * q);
        }
        const int deg = __shfl_sync(0xffffffffu, (int)rq.x, 0, 4);
        const int max_deg = __reduce_max_sync(0xffffffffu, active ? deg : 0);
        double2 acc_f = zero2, acc_s = zero2;
        tile_hops<NC>(rq, max_deg, x_first, x_second, a.coef, acc_f, acc_s);
        if (active) {
          const double2 oa = *reinterpret_cast<const double2*>(x_first + (size_t)pos * 128);
          const double2 ob = *reinterpret_cast<const double2*>(x_second + (size_t)pos * 128);
          acc_f.x = fma(a.ps, acc_f.x, a.qs * oa.x);
          acc_f.y = fma(a.ps, acc_f.y, a.qs * oa.y);
          acc_s.x = fma(a.ps, acc_s.x, a.qs * ob.x);
          acc_s.y = fma(a.ps, acc_s.y, a.qs * ob.y);
          D4 y = to_lohi(acc_f, acc_s, odd);
          y.x = fma(a.cs, v.x, fma(a.rs, x1.x, y.x));
          y.y = fma(a.cs, v.y, fma(a.rs, x1.y, y.y));
          y.z = fma(a.cs, v.z, fma(a.rs, x1.z, y.z));
          y.w = fma(a.cs, v.w, fma(a.rs, x1.w, y.w));
          stg256_stream(Pout + (size_t)dst * kTilePanel + 4 * q, y);
        }
      }
      __syncthreads();  // all reads of the tile done before the next bulk copy
    }
  }
}

// V (row-major n x s, caller's row order) -> panel-major copies at the positions of both layouts.
__global__ void __launch_bounds__(256) tiled_pack_kernel(long long n, int n_panels,
                                                         const double* __restrict__ V,
                                                         const int32_t* __restrict__ from_nat0,
                                                         const int32_t* __restrict__ from_nat1,
                                                         double* __restrict__ V0,
                                                         double* __restrict__ V1) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;  // one 32-byte piece each
  const int per_row = n_panels * 4;
  const long long row = t / per_row;
  if (row >= n) return;
  const int w = (int)(t % per_row), panel = w >> 2, piece = w & 3;
  const D4 v = ldg256_stream(V + t * 4);
  const size_t ps = (size_t)n * kTilePanel;
  stg256(V0 + panel * ps + (size_t)__ldg(from_nat0 + row) * kTilePanel + 4 * piece, v);
  stg256(V1 + panel * ps + (size_t)__ldg(from_nat1 + row) * kTilePanel + 4 * piece, v);
}

template <int NC>
int launch_sweep(const TiledPlan* p, const SweepArgs& a, cudaStream_t st) {
  tiled_sweep_kernel<NC><<<p->grid, kTileThreads, p->smem_bytes, st>>>(a);
  POLFED_LAUNCH_CHECK("tiled_sweep_kernel");
  return POLFED_OK;
}

int sweep(const TiledPlan* p, int layout, SweepArgs a, cudaStream_t st) {
  const TiledLayout& L = p->lay[layout];
  a.records = L.d_records;
  a.diag = L.d_diag;
  a.cc_col = L.d_cc_col;
  a.cc_val = L.d_cc_val;
  a.n_cross = L.n_cross;
  a.dst_map = (a.mode == MODE_LAST) ? L.d_to_natural : L.d_to_other;
  for (int c = 0; c < kTileMaxCoef; ++c) a.coef[c] = L.coef[c];
  POLFED_CUDA(cudaMemsetAsync(p->d_counter, 0, sizeof(int), st));
  return L.n_coef <= 2 ? launch_sweep<2>(p, a, st) : launch_sweep<4>(p, a, st);
}

template <int NC>
int configure_one(TiledPlan* p, int* occ) {
  POLFED_CUDA(cudaFuncSetAttribute(tiled_sweep_kernel<NC>,
                                   cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)p->smem_bytes));
  int o = 0;
  POLFED_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, tiled_sweep_kernel<NC>,
                                                            kTileThreads, p->smem_bytes));
  if (o < 1) return fail(POLFED_ECUDA, "tiled format: sweep kernel does not fit an SM");
  *occ = (*occ == 0 || o < *occ) ? o : *occ;
  return POLFED_OK;
}

}  // namespace

int tiled_configure_launch(TiledPlan* p) {
  p->smem_bytes = (size_t)(p->max_tile_rows + 1) * 128;  // + the zero row
  int occ = 0, rc;
  if ((rc = configure_one<2>(p, &occ))) return rc;
  if ((rc = configure_one<4>(p, &occ))) return rc;
  int dev = 0, sms = 148;
  POLFED_CUDA(cudaGetDevice(&dev));
  POLFED_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const long long want = (long long)occ * sms;
  p->grid = (int)(want < p->n_tiles ? want : p->n_tiles);
  if (p->grid < 1) p->grid = 1;
  return POLFED_OK;
}

bool tiled_supports(const polfed_ham* ham, int s) {
  return ham && ham->tiled && (s == 16 || s == 32) && ham->n > 0;
}

// X/P pairs (4 blocks) + V in both layouts (2 blocks) + the per-CTA scratch
size_t tiled_workspace_bytes(const polfed_ham* ham, int s) {
  const TiledPlan* p = ham->tiled;
  return (size_t)6 * (size_t)ham->n * s * sizeof(double) +
         (size_t)p->grid * p->max_tile_rows * 128;
}

int tiled_filter_apply(const polfed_ham* ham, double a_, double b_, int K, const double* c,
                       int s, const double* d_V, double* d_W, void* d_work, cudaStream_t st) {
  const TiledPlan* p = ham->tiled;
  const size_t len = (size_t)ham->n * s;
  double* base = static_cast<double*>(d_work);
  double* X[2] = {base, base + 2 * len};
  double* P[2] = {base + len, base + 3 * len};
  double* Vl[2] = {base + 4 * len, base + 5 * len};
  double* scratch = base + 6 * len;
  const int n_panels = s / kTilePanel;

  const long long threads = (long long)ham->n * n_panels * 4;
  tiled_pack_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
      ham->n, n_panels, d_V, p->lay[0].d_from_natural, p->lay[1].d_from_natural, Vl[0], Vl[1]);
  POLFED_LAUNCH_CHECK("tiled_pack_kernel");

  SweepArgs a{};
  a.n = ham->n;
  a.n_tiles = p->n_tiles;
  a.n_panels = n_panels;
  a.max_tile_rows = p->max_tile_rows;
  a.tile_row0 = p->d_tile_row0;
  a.tile_rec0 = p->d_tile_rec0;
  a.scratch = scratch;
  a.counter = p->d_counter;
  a.W = d_W;
  a.w_ld = s;
  auto pk = [&](int k) { return (k == 0 ? 1.0 : 2.0) / b_; };
  auto qk = [&](int k) { return (k == 0 ? -1.0 : -2.0) * a_ / b_; };

  // sweep j finishes b_{K-j} in layout j & 1 and starts the partial b_{K-j-1}
  for (int j = 0; j <= K; ++j) {
    const int k = K - j, layout = j & 1;
    const int in = (j + 1) & 1, out = j & 1;  // buffer pairs
    a.X1 = X[in];
    a.Pk = P[in];
    a.V = Vl[layout];
    a.Bout = X[out];
    a.Pout = P[out];
    a.cK = c[K];
    a.pf = pk(k);
    a.mode = (j == 0) ? MODE_INIT : (k == 0 ? MODE_LAST : MODE_STEP);
    if (k > 0) {
      a.ps = pk(k - 1);
      a.qs = qk(k - 1);
      a.cs = c[k - 1];
      a.rs = (j == 0) ? 0.0 : -1.0;
    }
    int rc = sweep(p, layout, a, st);
    if (rc) return rc;
  }
  return POLFED_OK;
}

}  // namespace polfed
