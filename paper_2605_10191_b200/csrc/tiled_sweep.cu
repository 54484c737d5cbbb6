// The tiled hot path (tiled.cuh): one persistent kernel per Clenshaw step.  A CTA takes a tile
// (a contiguous run of rows that share their high bits), pulls its 16-column panel of b_{k+1}
// into shared memory with one bulk copy, finishes b_k from shared-memory gathers, parks b_k in
// an L2-resident scratch, pulls it back as the new shared tile and starts P_{k-1} from it.
// Eq. (51) PAPER.md:427-431 with the rescaling of Eq. (31); see tiled.cuh for the algebra.
#include "tiled.cuh"

namespace polfed {
namespace {

enum { MODE_STEP = 0, MODE_INIT = 1, MODE_LAST = 2 };

struct SweepArgs {
  long long n;
  int n_tiles, n_panels, max_tile_rows;
  const int32_t* tile_row0;
  const int32_t* tile_rec0;
  const uint32_t* records;  // kTileRecWords words per class row
  const int32_t* dm_row_ptr;
  const int32_t* dm_col;
  const double* dm_val;
  const int32_t* pi;
  double coef[kTileMaxCoef];
  const double2* X1;  // b_{k+1}, panel-major, this layout
  const double2* Pk;  // partial b_k
  const double2* V;   // V in this layout
  double2* Bout;      // b_k, other layout
  double2* Pout;      // partial b_{k-1}, other layout
  double* W;          // MODE_LAST: row-major n x w_ld output in the natural layout
  int w_ld;
  double2* scratch;   // per CTA: max_tile_rows x 8 double2
  int* counter;
  double cK;              // MODE_INIT: b_K = cK V
  double pf;              // finishing scalar p_k
  double ps, qs, rs, cs;  // starting scalars of step k-1
  int mode;
  int out_perm;  // outputs go to row pi[row] (else to row)
};

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

// Thread mapping: 4 lanes own one 128-byte panel row (two 16-byte chunks each), a warp works on
// 8 rows at a time.  Even row slots read chunk q first and chunk q+4 second, odd slots the other
// way round, so that the two rows of a quarter-warp always hit disjoint shared-memory banks.

// One in-tile neighbour: entry in bits 16..31 of t = row (11 bits) | class (2) | sign (bit 31).
template <int NC>
__device__ __forceinline__ void hop_entry(uint32_t t, const unsigned char* __restrict__ xs_a,
                                          const unsigned char* __restrict__ xs_b,
                                          const double (&coef)[kTileMaxCoef], double2& acc_a,
                                          double2& acc_b) {
  const uint32_t off = (t >> 9) & 0x3ff80u;  // row * 128
  double cf = coef[0];
  if (NC == 2) {
    if (t & 0x08000000u) cf = coef[1];
  } else if (NC > 2) {
    const uint32_t c = (t >> 27) & 3u;
    if (c == 1) cf = coef[1];
    if (c == 2) cf = coef[2];
    if (NC > 3 && c == 3) cf = coef[3];
  }
  cf = __hiloint2double(__double2hiint(cf) ^ (int)(t & 0x80000000u), __double2loint(cf));
  const double2 xa = *reinterpret_cast<const double2*>(xs_a + off);
  const double2 xb = *reinterpret_cast<const double2*>(xs_b + off);
  acc_a.x = fma(cf, xa.x, acc_a.x);
  acc_a.y = fma(cf, xa.y, acc_a.y);
  acc_b.x = fma(cf, xb.x, acc_b.x);
  acc_b.y = fma(cf, xb.y, acc_b.y);
}

// All in-tile neighbours of the row whose record quarter this lane holds (rq); max_deg is
// warp-uniform, shorter rows run into entries that point at the zero row.
template <int NC>
__device__ __forceinline__ void tile_hops(const uint4 rq, int max_deg,
                                          const unsigned char* __restrict__ xs_a,
                                          const unsigned char* __restrict__ xs_b,
                                          const double (&coef)[kTileMaxCoef], double2& acc_a,
                                          double2& acc_b) {
#pragma unroll
  for (int w = 1; w <= kTileMaxDeg / 2; ++w) {
    if (2 * (w - 1) >= max_deg) break;
    const uint32_t mine = (w & 3) == 0 ? rq.x : (w & 3) == 1 ? rq.y : (w & 3) == 2 ? rq.z : rq.w;
    const uint32_t word = __shfl_sync(0xffffffffu, mine, w >> 2, 4);
    hop_entry<NC>(word << 16, xs_a, xs_b, coef, acc_a, acc_b);
    hop_entry<NC>(word, xs_a, xs_b, coef, acc_a, acc_b);
  }
}

template <int NC>
__global__ void __launch_bounds__(kTileThreads, 1) tiled_sweep_kernel(const SweepArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double2* xs = reinterpret_cast<double2*>(smem_raw);  // (max_tile_rows + 1) x 8 double2
  __shared__ uint64_t bar;
  __shared__ int s_tile;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int q = lane & 3, slot = lane >> 2;
  const int ca = q + 4 * (slot & 1), cb = ca ^ 4;  // the two chunks of this lane
  const unsigned char* xs_a = smem_raw + ca * 16;
  const unsigned char* xs_b = smem_raw + cb * 16;
  if (tid == 0) mbar_init(&bar, 1);
  __syncthreads();
  unsigned parity = 0;
  double2* scratch = a.scratch + (size_t)blockIdx.x * a.max_tile_rows * 8;
  const size_t panel_stride = (size_t)a.n * 8;  // double2 per panel
  constexpr int kRowsPerPass = (kTileThreads / 32) * 8;

  for (;;) {
    if (tid == 0) s_tile = atomicAdd(a.counter, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= a.n_tiles) break;
    const int row0 = __ldg(a.tile_row0 + tile);
    const int nrows = __ldg(a.tile_row0 + tile + 1) - row0;
    const uint4* rec = reinterpret_cast<const uint4*>(a.records) +
                       (size_t)__ldg(a.tile_rec0 + tile) * 4;
    if (tid < 8) xs[nrows * 8 + tid] = make_double2(0.0, 0.0);  // the zero row
    __syncthreads();

    for (int panel = 0; panel < a.n_panels; ++panel) {
      const double2* X1 = a.X1 + panel * panel_stride;
      const double2* Pk = a.Pk + panel * panel_stride;
      const double2* V = a.V + panel * panel_stride;
      double2* Bout = a.Bout + panel * panel_stride;
      double2* Pout = a.Pout + panel * panel_stride;

      if (a.mode != MODE_INIT) {
        if (tid == 0) tile_load(xs, X1 + (size_t)row0 * 8, (unsigned)nrows * 128u, &bar);
        mbar_wait(&bar, parity);
        parity ^= 1u;
      }

      // ---- phase 2: b_k = P_k + p_k (O_l + DM) b_{k+1} -----------------------------------------
      for (int base = warp * 8; base < nrows; base += kRowsPerPass) {
        const int t = base + slot;
        const bool active = t < nrows;
        uint4 rq = make_uint4(0u, 0u, 0u, 0u);
        if (active) rq = __ldg(rec + (size_t)t * 4 + q);
        const uint32_t header = __shfl_sync(0xffffffffu, rq.x, 0, 4);
        const int rid = header & 0x7ff;
        const int row = row0 + rid;
        double2 ba = make_double2(0.0, 0.0), bb = ba;
        if (a.mode == MODE_INIT) {
          if (active) {
            const double2 va = __ldcs(V + (size_t)row * 8 + ca);
            const double2 vb = __ldcs(V + (size_t)row * 8 + cb);
            ba = make_double2(a.cK * va.x, a.cK * va.y);
            bb = make_double2(a.cK * vb.x, a.cK * vb.y);
          }
        } else {
          int e0 = 0, e1 = 0;
          double2 pka = ba, pkb = ba;
          if (active) {
            e0 = __ldg(a.dm_row_ptr + row);
            e1 = __ldg(a.dm_row_ptr + row + 1);
            pka = __ldcs(Pk + (size_t)row * 8 + ca);
            pkb = __ldcs(Pk + (size_t)row * 8 + cb);
          }
          const int max_deg =
              __reduce_max_sync(0xffffffffu, active ? (int)((header >> 16) & 0x1f) : 0);
          double2 acc_a = ba, acc_b = ba;
          // diagonal + cross-cut entries: columns inside the tile come from shared memory
          const int ndm = e1 - e0;
          const int max_dm = __reduce_max_sync(0xffffffffu, ndm);
          for (int off = 0; off < max_dm; off += 4) {
            const int e = e0 + off + q;
            int cc = 0;
            double vv = 0.0;
            if (e < e1) {
              cc = __ldg(a.dm_col + e);
              vv = __ldg(a.dm_val + e);
            }
            const int rem = ndm - off;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              if (off + j >= max_dm) break;
              const int cj = __shfl_sync(0xffffffffu, cc, j, 4);
              const double vj = __shfl_sync(0xffffffffu, vv, j, 4);
              if (j < rem) {
                const unsigned u = (unsigned)(cj - row0);
                double2 xa, xb;
                if (u < (unsigned)nrows) {
                  xa = xs[u * 8 + ca];
                  xb = xs[u * 8 + cb];
                } else {
                  xa = __ldg(X1 + (size_t)cj * 8 + ca);
                  xb = __ldg(X1 + (size_t)cj * 8 + cb);
                }
                acc_a.x = fma(vj, xa.x, acc_a.x);
                acc_a.y = fma(vj, xa.y, acc_a.y);
                acc_b.x = fma(vj, xb.x, acc_b.x);
                acc_b.y = fma(vj, xb.y, acc_b.y);
              }
            }
          }
          tile_hops<NC>(rq, max_deg, xs_a, xs_b, a.coef, acc_a, acc_b);
          ba = make_double2(fma(a.pf, acc_a.x, pka.x), fma(a.pf, acc_a.y, pka.y));
          bb = make_double2(fma(a.pf, acc_b.x, pkb.x), fma(a.pf, acc_b.y, pkb.y));
        }
        if (active) {
          const int dst = a.out_perm ? __ldg(a.pi + row) : row;
          if (a.mode == MODE_LAST) {
            double* w = a.W + (size_t)dst * a.w_ld + panel * kTilePanel;
            *reinterpret_cast<double2*>(w + 2 * ca) = ba;
            *reinterpret_cast<double2*>(w + 2 * cb) = bb;
          } else {
            __stcs(Bout + (size_t)dst * 8 + ca, ba);
            __stcs(Bout + (size_t)dst * 8 + cb, bb);
            scratch[rid * 8 + ca] = ba;
            scratch[rid * 8 + cb] = bb;
          }
        }
      }
      if (a.mode == MODE_LAST) {
        __syncthreads();  // the next bulk copy overwrites xs
        continue;
      }

      // ---- b_k becomes the shared tile ------------------------------------------------------
      __threadfence_block();
      fence_proxy_async();
      __syncthreads();
      if (tid == 0) tile_load(xs, scratch, (unsigned)nrows * 128u, &bar);
      mbar_wait(&bar, parity);
      parity ^= 1u;

      // ---- phase 3: P_{k-1} = c_{k-1} V + p_{k-1} O_l b_k + q_{k-1} b_k + r b_{k+1} -----------------
      for (int base = warp * 8; base < nrows; base += kRowsPerPass) {
        const int t = base + slot;
        const bool active = t < nrows;
        uint4 rq = make_uint4(0u, 0u, 0u, 0u);
        if (active) rq = __ldg(rec + (size_t)t * 4 + q);
        const uint32_t header = __shfl_sync(0xffffffffu, rq.x, 0, 4);
        const int rid = header & 0x7ff;
        const int row = row0 + rid;
        const double2 zero = make_double2(0.0, 0.0);
        double2 x1a = zero, x1b = zero, va = zero, vb = zero;
        int dst = row;
        if (active) {
          if (a.rs != 0.0) {
            x1a = __ldg(X1 + (size_t)row * 8 + ca);
            x1b = __ldg(X1 + (size_t)row * 8 + cb);
          }
          if (a.cs != 0.0) {
            va = __ldcs(V + (size_t)row * 8 + ca);
            vb = __ldcs(V + (size_t)row * 8 + cb);
          }
          if (a.out_perm) dst = __ldg(a.pi + row);
        }
        const int max_deg =
            __reduce_max_sync(0xffffffffu, active ? (int)((header >> 16) & 0x1f) : 0);
        double2 acc_a = zero, acc_b = zero;
        tile_hops<NC>(rq, max_deg, xs_a, xs_b, a.coef, acc_a, acc_b);
        if (active) {
          const double2 oa = xs[rid * 8 + ca], ob = xs[rid * 8 + cb];
          double2 ya, yb;
          ya.x = fma(a.ps, acc_a.x, a.qs * oa.x);
          ya.y = fma(a.ps, acc_a.y, a.qs * oa.y);
          yb.x = fma(a.ps, acc_b.x, a.qs * ob.x);
          yb.y = fma(a.ps, acc_b.y, a.qs * ob.y);
          ya.x = fma(a.rs, x1a.x, ya.x);
          ya.y = fma(a.rs, x1a.y, ya.y);
          yb.x = fma(a.rs, x1b.x, yb.x);
          yb.y = fma(a.rs, x1b.y, yb.y);
          ya.x = fma(a.cs, va.x, ya.x);
          ya.y = fma(a.cs, va.y, ya.y);
          yb.x = fma(a.cs, vb.x, yb.x);
          yb.y = fma(a.cs, vb.y, yb.y);
          __stcs(Pout + (size_t)dst * 8 + ca, ya);
          __stcs(Pout + (size_t)dst * 8 + cb, yb);
        }
      }
      __syncthreads();  // all reads of xs done before the next bulk copy
    }
  }
}

// V (row-major n x s) -> panel-major copies in both layouts.
__global__ void __launch_bounds__(256) tiled_pack_kernel(long long n, int n_panels,
                                                         const double2* __restrict__ V,
                                                         const int32_t* __restrict__ pi,
                                                         double2* __restrict__ V0,
                                                         double2* __restrict__ V1) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long per_row = (long long)n_panels * 8;
  const long long row = t / per_row;
  if (row >= n) return;
  const int w = (int)(t % per_row), panel = w >> 3, l = w & 7;
  const double2 v = __ldcs(V + t);
  const size_t ps = (size_t)n * 8;
  V0[panel * ps + (size_t)row * 8 + l] = v;
  V1[panel * ps + (size_t)__ldg(pi + row) * 8 + l] = v;
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
  a.dm_row_ptr = L.d_dm_row_ptr;
  a.dm_col = L.d_dm_col;
  a.dm_val = L.d_dm_val;
  for (int c = 0; c < kTileMaxCoef; ++c) a.coef[c] = L.coef[c];
  POLFED_CUDA(cudaMemsetAsync(p->d_counter, 0, sizeof(int), st));
  switch (L.n_coef) {
    case 0:
    case 1: return launch_sweep<1>(p, a, st);
    case 2: return launch_sweep<2>(p, a, st);
    case 3: return launch_sweep<3>(p, a, st);
    default: return launch_sweep<4>(p, a, st);
  }
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
  if ((rc = configure_one<1>(p, &occ))) return rc;
  if ((rc = configure_one<2>(p, &occ))) return rc;
  if ((rc = configure_one<3>(p, &occ))) return rc;
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
  double2* scratch = reinterpret_cast<double2*>(base + 6 * len);
  const int n_panels = s / kTilePanel;

  const long long threads = (long long)ham->n * n_panels * 8;
  tiled_pack_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
      ham->n, n_panels, reinterpret_cast<const double2*>(d_V), p->d_pi,
      reinterpret_cast<double2*>(Vl[0]), reinterpret_cast<double2*>(Vl[1]));
  POLFED_LAUNCH_CHECK("tiled_pack_kernel");

  SweepArgs a{};
  a.n = ham->n;
  a.n_tiles = p->n_tiles;
  a.n_panels = n_panels;
  a.max_tile_rows = p->max_tile_rows;
  a.tile_row0 = p->d_tile_row0;
  a.tile_rec0 = p->d_tile_rec0;
  a.pi = p->d_pi;
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
    a.X1 = reinterpret_cast<const double2*>(X[in]);
    a.Pk = reinterpret_cast<const double2*>(P[in]);
    a.V = reinterpret_cast<const double2*>(Vl[layout]);
    a.Bout = reinterpret_cast<double2*>(X[out]);
    a.Pout = reinterpret_cast<double2*>(P[out]);
    a.cK = c[K];
    a.pf = pk(k);
    a.mode = (j == 0) ? MODE_INIT : (k == 0 ? MODE_LAST : MODE_STEP);
    a.out_perm = (k == 0) ? (layout == 1) : 1;
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
