// Host side of the sector sweep (sector.cuh): instantiation table, launch configuration, the V
// pack kernel and the Clenshaw pipeline of Eq. (51) PAPER.md:427-431 as K + 1 sweeps.
#include "sector_kernel.cuh"

namespace polfed {

// One entry per instantiation file sector_m*.cu.
struct SectorImpl {
  int m;
  bool nnn, jw;
  int (*launch)(const sector::SecArgs&, int mode, int grid, size_t smem, cudaStream_t);
  int (*configure)(size_t smem, int* occ);
};
#define POLFED_SECTOR_DECL(M, NNN, JW)                                                        \
  int sector_launch_##M##_##NNN##_##JW(const sector::SecArgs&, int, int, size_t, cudaStream_t); \
  int sector_configure_##M##_##NNN##_##JW(size_t, int*);
#define POLFED_SECTOR_ENTRY(M, NNN, JW) \
  {M, NNN != 0, JW != 0, sector_launch_##M##_##NNN##_##JW, sector_configure_##M##_##NNN##_##JW},
#define POLFED_SECTOR_LIST(X) \
  X(4, 1, 1) X(5, 1, 1) X(6, 1, 1) X(7, 1, 1) X(8, 1, 1) X(9, 1, 1) X(13, 1, 1) \
  X(6, 0, 0) X(7, 0, 0) X(8, 0, 0) X(10, 0, 0)
POLFED_SECTOR_LIST(POLFED_SECTOR_DECL)

namespace {

const SectorImpl kImpls[] = {POLFED_SECTOR_LIST(POLFED_SECTOR_ENTRY)};

const SectorImpl* find_impl(int m, bool nnn, bool jw) {
  for (const SectorImpl& i : kImpls)
    if (i.m == m && i.nnn == nnn && i.jw == (nnn && jw)) return &i;
  return nullptr;
}

// V (row-major n x s, caller's row order) -> panel-major [s/8][n][8] copies at the positions of
// both layouts.  One thread moves one 32-byte piece.
__global__ void __launch_bounds__(256) sector_pack_kernel(long long n, int n_panels,
                                                          const double* __restrict__ V,
                                                          const int32_t* __restrict__ from_nat0,
                                                          const int32_t* __restrict__ from_nat1,
                                                          double* __restrict__ V0,
                                                          double* __restrict__ V1) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int per_row = n_panels * 2;
  const long long row = t / per_row;
  if (row >= n) return;
  const int w = (int)(t % per_row), panel = w >> 1, piece = w & 1;
  double4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w)
               : "l"(V + t * 4));
  const size_t ps = (size_t)n * kSecPanel;
  double* d0 = V0 + panel * ps + (size_t)__ldg(from_nat0 + row) * kSecPanel + 4 * piece;
  double* d1 = V1 + panel * ps + (size_t)__ldg(from_nat1 + row) * kSecPanel + 4 * piece;
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(d0), "d"(v.x), "d"(v.y), "d"(v.z),
               "d"(v.w)
               : "memory");
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(d1), "d"(v.x), "d"(v.y), "d"(v.z),
               "d"(v.w)
               : "memory");
}

}  // namespace

bool sector_m_supported(int m, bool nnn, bool jw) { return find_impl(m, nnn, jw) != nullptr; }

void destroy_sector_plan(SectorPlan* sp) {
  if (!sp) return;
  for (auto& l : sp->lay) cudaFree(l.d_meta);
  cudaFree(sp->d_units);
  cudaFree(sp->d_tile_class);
  delete sp;
}

int sector_configure_launch(const TiledPlan* tp, SectorPlan* sp) {
  const SectorImpl* impl = find_impl(sp->m, sp->nnn, sp->jw);
  if (!impl) return fail(POLFED_EINVAL, "sector sweep: no kernel for m=%d", sp->m);
  const size_t buf = ((size_t)sp->max_rows_p * 64 + 127) / 128 * 128;
  sp->smem_bytes = 2 * buf;
  int occ = 0;
  int rc = impl->configure(sp->smem_bytes, &occ);
  if (rc) return rc;
  int dev = 0, sms = 148;
  POLFED_CUDA(cudaGetDevice(&dev));
  POLFED_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const long long want = (long long)occ * sms;
  sp->grid = (int)(want < 4LL * tp->n_tiles ? want : 4LL * tp->n_tiles);
  if (sp->grid < 1) sp->grid = 1;
  return POLFED_OK;
}

// X/P pairs (4 blocks) + V in both layouts (2 blocks) + two work-item counters
size_t sector_workspace_bytes(const polfed_ham* ham, int s) {
  return (size_t)6 * (size_t)ham->n * s * sizeof(double) + 128;
}

int sector_filter_apply(const polfed_ham* ham, double a_, double b_, int K, const double* c, int s,
                        const double* d_V, double* d_W, void* d_work, cudaStream_t st) {
  const TiledPlan* p = ham->tiled;
  const SectorPlan* sp = p->sector;
  const SectorImpl* impl = find_impl(sp->m, sp->nnn, sp->jw);
  const size_t len = (size_t)ham->n * s;
  double* base = static_cast<double*>(d_work);
  double* X[2] = {base, base + 2 * len};
  double* P[2] = {base + len, base + 3 * len};
  double* Vl[2] = {base + 4 * len, base + 5 * len};
  int* counters = reinterpret_cast<int*>(base + 6 * len);  // one per sweep parity, 64 bytes apart
  const int n_panels = s / kSecPanel;

  POLFED_CUDA(cudaMemsetAsync(counters, 0, 128, st));
  const long long threads = (long long)ham->n * n_panels * 2;
  sector_pack_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
      ham->n, n_panels, d_V, p->lay[0].d_from_natural, p->lay[1].d_from_natural, Vl[0], Vl[1]);
  POLFED_LAUNCH_CHECK("sector_pack_kernel");

  sector::SecArgs a{};
  a.n = ham->n;
  a.n_tiles = p->n_tiles;
  a.n_panels = n_panels;
  a.tile_row0 = p->d_tile_row0;
  a.tile_class = sp->d_tile_class;
  a.units = sp->d_units;
  a.W = d_W;
  a.w_ld = s;
  a.buf_bytes = (unsigned)(sp->smem_bytes / 2);
  a.tab = sp->tab;
  auto pk = [&](int k) { return (k == 0 ? 1.0 : 2.0) / b_; };
  auto qk = [&](int k) { return (k == 0 ? -1.0 : -2.0) * a_ / b_; };

  // sweep j finishes b_{K-j} in layout j & 1 and starts the partial b_{K-j-1}
  for (int j = 0; j <= K; ++j) {
    const int k = K - j, layout = j & 1;
    const int in = (j + 1) & 1, out = j & 1;  // buffer pairs
    const TiledLayout& L = p->lay[layout];
    const SectorLayout& S = sp->lay[layout];
    a.meta = S.d_meta;
    a.dst_nat = L.d_to_natural;
    for (int e = 0; e <= kTileMaxCrossCoef; ++e) a.ccoef[e] = L.ccoef[e];
    a.t1 = S.t1;
    a.t2 = S.t2;
    a.X1 = X[in];
    a.Pk = P[in];
    a.V = Vl[layout];
    a.Bout = X[out];
    a.Pout = P[out];
    a.counter = counters + 16 * (j & 1);
    a.cK = c[K];
    a.pf = pk(k);
    const int mode = (j == 0) ? sector::MODE_INIT : (k == 0 ? sector::MODE_LAST : sector::MODE_STEP);
    if (k > 0) {
      a.ps = pk(k - 1);
      a.qs = qk(k - 1);
      a.cs = c[k - 1];
      a.rs = (j == 0) ? 0.0 : -1.0;
    }
    // the other counter is free (its sweep has completed): zero it for the next sweep
    POLFED_CUDA(cudaMemsetAsync(counters + 16 * ((j + 1) & 1), 0, sizeof(int), st));
    int rc = impl->launch(a, mode, sp->grid, sp->smem_bytes, st);
    if (rc) return rc;
  }
  return POLFED_OK;
}

}  // namespace polfed
