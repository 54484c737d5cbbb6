// Construction of the tiled format (tiled.cuh): term classification, per-class neighbour
// records in processing order, tile table, the position maps between the two layouts and the
// caller's row order, and the diagonal + cross-cut part of each layout.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "combinadic.cuh"
#include "sector.cuh"
#include "tiled.cuh"

namespace polfed {

int tiled_configure_launch(TiledPlan* plan);  // tiled_sweep.cu

namespace {

// Row of state x in the ascending order of the states with the site order reversed.
__global__ void __launch_bounds__(256) reverse_rank_kernel(int64_t n, int n_sites, int n_up,
                                                           const uint64_t* __restrict__ states,
                                                           int32_t* __restrict__ pi) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  const uint64_t y = __brevll(states[r]) >> (64 - n_sites);
  pi[r] = (int32_t)rank_state(y, n_sites, n_up);
}

// Ascending row (of one layout) -> position: one CTA per tile applies the class permutation.
__global__ void __launch_bounds__(256) position_kernel(const int32_t* __restrict__ tile_row0,
                                                       const int32_t* __restrict__ tile_rec0,
                                                       const int32_t* __restrict__ inv_sigma,
                                                       int32_t* __restrict__ pos) {
  const int row0 = tile_row0[blockIdx.x], nrows = tile_row0[blockIdx.x + 1] - row0;
  const int rec0 = tile_rec0[blockIdx.x];
  for (int i = threadIdx.x; i < nrows; i += blockDim.x) pos[row0 + i] = row0 + inv_sigma[rec0 + i];
}

// pos0/pos1: position of an ascending row of layout 0 / layout 1; pi: layout-0 row -> layout-1 row.
__global__ void __launch_bounds__(256) maps_kernel(int64_t n, const int32_t* __restrict__ pi,
                                                   const int32_t* __restrict__ pos0,
                                                   const int32_t* __restrict__ pos1,
                                                   int32_t* to_other0, int32_t* to_other1,
                                                   int32_t* to_nat0, int32_t* to_nat1,
                                                   int32_t* from_nat0, int32_t* from_nat1,
                                                   uint32_t* side0, int sw0, uint32_t* side1,
                                                   int sw1) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  const int32_t p0 = pos0[r], p1 = pos1[pi[r]];
  to_other0[p0] = p1;
  to_other1[p1] = p0;
  side0[(size_t)p0 * sw0] = (uint32_t)p1;
  side1[(size_t)p1 * sw1] = (uint32_t)p0;
  to_nat0[p0] = (int32_t)r;
  to_nat1[p1] = (int32_t)r;
  from_nat0[r] = p0;
  from_nat1[r] = p1;
}

__global__ void __launch_bounds__(256) max_offdiag_kernel(int64_t n, const int32_t* __restrict__ row_ptr,
                                                          int* out) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int v = (r < n) ? row_ptr[r + 1] - row_ptr[r] - 1 : 0;
  v = __reduce_max_sync(0xffffffffu, v);
  if ((threadIdx.x & 31) == 0) atomicMax(out, v);
}

// Distinct |value| of the off-diagonal CSR entries -> table[0..kTileMaxCrossCoef) (bit patterns,
// 0 = free slot; insertion order is arbitrary, the packed words below refer to the final slots).
__global__ void __launch_bounds__(256) cross_coef_kernel(int64_t n, const int32_t* __restrict__ row_ptr,
                                                         const int32_t* __restrict__ col,
                                                         const double* __restrict__ val,
                                                         unsigned long long* table, int* overflow) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  for (int e = row_ptr[r]; e < row_ptr[r + 1]; ++e) {
    if (col[e] == (int32_t)r || val[e] == 0.0) continue;
    const unsigned long long mag = (unsigned long long)__double_as_longlong(fabs(val[e]));
    int c = 0;
    for (; c < kTileMaxCrossCoef; ++c) {
      unsigned long long cur = table[c];
      if (cur == 0ull) cur = atomicCAS(table + c, 0ull, mag);
      if (cur == 0ull || cur == mag) break;
    }
    if (c == kTileMaxCrossCoef) *overflow = 1;
  }
}

// CSR (ascending rows of this layout, diagonal always stored) -> diagonal + packed cross-cut
// words by position (word 0 of a side record, the position in the other layout, is filled by
// maps_kernel).
__global__ void __launch_bounds__(256) dm_ell_kernel(int64_t n, int n_cross,
                                                     const int32_t* __restrict__ row_ptr,
                                                     const int32_t* __restrict__ col,
                                                     const double* __restrict__ val,
                                                     const int32_t* __restrict__ pos,
                                                     const unsigned long long* __restrict__ table,
                                                     double* __restrict__ diag, int side_words,
                                                     uint32_t* __restrict__ side) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  const int32_t p = pos[r];
  int slot = 0;
  double d = 0.0;
  for (int e = row_ptr[r]; e < row_ptr[r + 1]; ++e) {
    const int32_t c = col[e];
    if (c == (int32_t)r) {
      d += val[e];
    } else if (val[e] != 0.0) {
      const unsigned long long mag = (unsigned long long)__double_as_longlong(fabs(val[e]));
      uint32_t cls = 0;
      while (cls < (uint32_t)kTileMaxCrossCoef - 1 && table[cls] != mag) ++cls;
      side[(size_t)p * side_words + 1 + slot] = (uint32_t)pos[c] | (cls << kCrossPosBits) |
                                                (val[e] < 0.0 ? 0x80000000u : 0u);
      ++slot;
    }
  }
  diag[p] = d;
  for (; slot + 1 < side_words; ++slot) side[(size_t)p * side_words + 1 + slot] = kCrossNone;
}

inline bool off_diagonal(int kind) { return kind >= POLFED_TERM_EXCH; }

// Position of the m-bit configuration l among the configurations of equal popcount.
uint32_t class_rank(uint32_t l) {
  uint32_t r = 0;
  int j = 0;
  while (l) {
    const int p = __builtin_ctz(l);
    l &= l - 1;
    ++j;
    r += (uint32_t)host_binom(p, j);
  }
  return r;
}

template <class T>
int upload(T** d, const std::vector<T>& h) {
  POLFED_CUDA(cudaMalloc(reinterpret_cast<void**>(d), sizeof(T) * (h.size() ? h.size() : 1)));
  if (!h.empty())
    POLFED_CUDA(cudaMemcpy(*d, h.data(), sizeof(T) * h.size(), cudaMemcpyHostToDevice));
  return POLFED_OK;
}

struct Entry {
  uint32_t nbr;   // class rank of the neighbour (ascending order inside the class)
  uint32_t cls;   // amplitude class
  uint32_t sign;  // 1 = negative
};

// Records of one layout: `low` holds the tile-local hops with sites already in this layout's
// numbering (all < m).  Class k (k particles on the low m sites) owns records
// class_off[k] .. class_off[k+1].  Inside a class the rows are put in processing order (falling
// degree); inv_sigma[class_off[k] + ascending rank] = position inside the class.
int build_records(int m, const std::vector<DevTerm>& low, TiledLayout* lay,
                  std::vector<uint32_t>* rec, std::vector<int32_t>* inv_sigma,
                  const std::vector<int>& class_off) {
  lay->n_coef = 0;
  std::vector<int> cls(low.size(), -1);
  for (size_t t = 0; t < low.size(); ++t) {
    const double mag = low[t].amp < 0 ? -low[t].amp : low[t].amp;
    if (mag == 0.0) continue;
    int c = 0;
    while (c < lay->n_coef && lay->coef[c] != mag) ++c;
    if (c == lay->n_coef) {
      if (c == kTileMaxCoef)
        return fail(POLFED_EINVAL,
                    "tiled format: more than %d distinct hopping amplitudes inside a tile",
                    kTileMaxCoef);
      lay->coef[lay->n_coef++] = mag;
    }
    cls[t] = c;
  }
  const size_t n_cfg = (size_t)1 << m;
  rec->assign(n_cfg * kTileRecWords, 0u);
  inv_sigma->assign(n_cfg, 0);
  std::vector<std::vector<Entry>> ent(n_cfg);  // by class_off[k] + class_rank(l)
  for (uint32_t l = 0; l < n_cfg; ++l) {
    const int k = __builtin_popcount(l);
    std::vector<Entry>& e = ent[(size_t)class_off[k] + class_rank(l)];
    for (size_t t = 0; t < low.size(); ++t) {
      if (cls[t] < 0) continue;
      const int i = low[t].i, j = low[t].j;
      if (((l >> i) & 1u) == ((l >> j) & 1u)) continue;
      const uint32_t l2 = l ^ (1u << i) ^ (1u << j);
      uint32_t sign = low[t].amp < 0 ? 1u : 0u;
      if (low[t].kind == POLFED_TERM_HOPJW) {
        const int lo = std::min(i, j), hi = std::max(i, j);
        const uint32_t between = ((1u << hi) - 1u) & ~((2u << lo) - 1u);
        sign ^= (uint32_t)__builtin_popcount(l & between) & 1u;
      }
      e.push_back(Entry{class_rank(l2), (uint32_t)cls[t], sign});
    }
    if ((int)e.size() > kTileMaxDeg)
      return fail(POLFED_EINVAL, "tiled format: more than %d hops inside a tile for one state",
                  kTileMaxDeg);
  }
  for (int k = 0; k <= m; ++k) {
    const int n_k = class_off[k + 1] - class_off[k];
    std::vector<int> order(n_k);
    for (int r = 0; r < n_k; ++r) order[r] = r;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) {
      return ent[(size_t)class_off[k] + x].size() > ent[(size_t)class_off[k] + y].size();
    });
    int32_t* inv = inv_sigma->data() + class_off[k];
    for (int t = 0; t < n_k; ++t) inv[order[t]] = t;
    for (int t = 0; t < n_k; ++t) {
      const std::vector<Entry>& e = ent[(size_t)class_off[k] + order[t]];
      uint32_t* w = rec->data() + ((size_t)class_off[k] + t) * kTileRecWords;
      w[0] = (uint32_t)e.size();
      for (int j = 0; j < kTileMaxDeg; ++j) {
        const bool used = j < (int)e.size();
        const uint32_t pos = used ? (uint32_t)inv[e[j].nbr] : (uint32_t)n_k;  // zero row
        const uint32_t c = used ? e[j].cls : 0u, sg = used ? e[j].sign : 0u;
        uint32_t& word = w[1 + (j >> 1)];
        if ((j & 1) == 0) word |= (pos << 7) | c | (sg << 30);
        else word |= (pos << 18) | (c << 2) | (sg << 31);
      }
    }
  }
  return POLFED_OK;
}


// ---- sector sweep (sector.cuh) ---------------------------------------------------------------
// JW sign (1 = negative, the sign of amp not included) and applicability of a hop term on the
// m-bit configuration l.
inline bool hop_applies(const DevTerm& t, uint32_t l, uint32_t* l2, uint32_t* jw_sign) {
  const int i = t.i, j = t.j;
  if (((l >> i) & 1u) == ((l >> j) & 1u)) return false;
  *l2 = l ^ (1u << i) ^ (1u << j);
  uint32_t sg = 0u;
  if (t.kind == POLFED_TERM_HOPJW) {
    const int lo = std::min(i, j), hi = std::max(i, j);
    const uint32_t between = ((1u << hi) - 1u) & ~((2u << lo) - 1u);
    sg = (uint32_t)__builtin_popcount(l & between) & 1u;
  }
  *jw_sign = sg;
  return true;
}

// True when the tile-local hops of a layout are exactly one bond (i, i+1) for every i < m - 1
// with one amplitude t1 and either no or one bond (i, i+2) for every i < m - 2 with one
// amplitude t2 (all HOPJW: jw, or all EXCH).
bool sector_pattern(int m, const std::vector<DevTerm>& low, double* t1, double* t2, bool* nnn,
                    bool* jw) {
  std::vector<int> cnt1(m, 0), cnt2(m, 0);
  int n_jw = 0, n_ex = 0, n1 = 0, n2 = 0;
  *t1 = *t2 = 0.0;
  for (const DevTerm& t : low) {
    if (t.amp == 0.0) continue;
    const int lo = std::min(t.i, t.j), d = std::max(t.i, t.j) - lo;
    if (d == 1) {
      if (n1++ == 0) *t1 = t.amp;
      if (t.amp != *t1 || ++cnt1[lo] > 1) return false;
    } else if (d == 2) {
      if (n2++ == 0) *t2 = t.amp;
      if (t.amp != *t2 || ++cnt2[lo] > 1) return false;
      (t.kind == POLFED_TERM_HOPJW ? n_jw : n_ex)++;
    } else {
      return false;
    }
  }
  if (n1 != m - 1) return false;
  if (n2 != 0 && (n2 != m - 2 || (n_jw != 0 && n_ex != 0))) return false;
  *nnn = n2 != 0;
  *jw = n_jw != 0;
  return true;
}

struct SectorHost {
  std::vector<int32_t> inv_sigma;  // class_off[k] + ascending class rank -> position in class
  std::vector<uint64_t> xg;        // class_off[k] + position -> three cross-group entries
};

// Geometry shared by both layouts: sector bases, fibre pitches, work units.
void sector_geometry(int m, bool pad, SectorPlan* sp, std::vector<uint16_t>* units) {
  const int g1 = sector_g1(m), g2 = m - g1;
  sp->m = m;
  sp->g1 = g1;
  sp->g2 = g2;
  SectorTables& T = sp->tab;
  for (int j = 0; j <= kSecMaxG; ++j) {
    T.n1[j] = j <= g1 ? (short)host_binom(g1, j) : 0;
    T.n2[j] = j <= g2 ? (short)host_binom(g2, j) : 0;
    T.n1p[j] = (short)((pad && T.n1[j] > 1 && T.n1[j] % 2 == 0) ? T.n1[j] + 1 : T.n1[j]);
  }
  units->assign((size_t)2 * (m + 1) * kSecMaxUnits, 0);
  sp->max_rows_p = 1;
  for (int k = 0; k <= m; ++k) {
    int pos = 0, row = 0;
    struct U { int cost; uint16_t code; };
    std::vector<U> u1, u2;
    for (int j1 = std::max(0, k - g2); j1 <= std::min(g1, k); ++j1) {
      const int n1 = T.n1[j1], n2 = T.n2[k - j1];
      T.sbase[k][j1] = (short)pos;
      T.srow[k][j1] = (short)row;
      pos += n1 * n2;
      row += T.n1p[j1] * n2;
      for (int q = 0; q * kSecGroups < n2; ++q) u1.push_back(U{n1, (uint16_t)(j1 | (q << 3))});
      for (int q = 0; q * kSecGroups < n1; ++q) u2.push_back(U{n2, (uint16_t)(j1 | (q << 3))});
    }
    T.rows_p[k] = (short)row;
    sp->max_rows_p = std::max(sp->max_rows_p, row);
    auto by_cost = [](const U& a, const U& b) { return a.cost > b.cost; };
    std::stable_sort(u1.begin(), u1.end(), by_cost);
    std::stable_sort(u2.begin(), u2.end(), by_cost);
    T.n_units[0][k] = (short)u1.size();
    T.n_units[1][k] = (short)u2.size();
    for (size_t i = 0; i < u1.size(); ++i) (*units)[(size_t)k * kSecMaxUnits + i] = u1[i].code;
    for (size_t i = 0; i < u2.size(); ++i)
      (*units)[(size_t)(m + 1 + k) * kSecMaxUnits + i] = u2[i].code;
  }
}

// Sector order of the class rows and the cross-group entries of one layout.
void sector_tables(const SectorPlan& sp, const std::vector<DevTerm>& low,
                   const std::vector<int>& class_off, SectorHost* out) {
  const int m = sp.m, g1 = sp.g1;
  const SectorTables& T = sp.tab;
  const size_t n_cfg = (size_t)1 << m;
  out->inv_sigma.assign(n_cfg, 0);
  out->xg.assign(n_cfg, 0ull);
  auto locate = [&](uint32_t l, int* pos, int* srow) {
    const int k = __builtin_popcount(l);
    const uint32_t c1 = l & ((1u << g1) - 1u), c2 = l >> g1;
    const int j1 = __builtin_popcount(c1);
    const int i1 = (int)class_rank(c1), i2 = (int)class_rank(c2);
    *pos = T.sbase[k][j1] + i2 * T.n1[j1] + i1;
    *srow = T.srow[k][j1] + i2 * T.n1p[j1] + i1;
  };
  for (uint32_t l = 0; l < n_cfg; ++l) {
    const int k = __builtin_popcount(l);
    int pos, srow;
    locate(l, &pos, &srow);
    out->inv_sigma[(size_t)class_off[k] + class_rank(l)] = pos;
    uint64_t rec = (uint64_t)srow << 48;  // the row's own shared-memory row
    for (const DevTerm& t : low) {
      const int lo = std::min(t.i, t.j), hi = std::max(t.i, t.j);
      if (t.amp == 0.0 || !(lo < g1 && hi >= g1)) continue;
      uint32_t l2, sg;
      if (!hop_applies(t, l, &l2, &sg)) continue;
      int pos2, srow2;
      locate(l2, &pos2, &srow2);
      // slot 0: the (g1-1, g1) bond (t1); slot 1: (g1-2, g1), slot 2: (g1-1, g1+1) (t2)
      const int slot = hi - lo == 1 ? 0 : (lo == g1 - 2 ? 1 : 2);
      rec |= ((uint64_t)srow2 | kXgValid | (sg ? kXgNeg : 0u)) << (16 * slot);
    }
    out->xg[(size_t)class_off[k] + pos] = rec;
  }
}

// side (4 words) + cross-group entries + diagonal -> the 32-byte row record of sector.cuh.
__global__ void __launch_bounds__(256) sector_meta_kernel(const int32_t* __restrict__ tile_row0,
                                                          const int32_t* __restrict__ tile_rec0,
                                                          const uint4* __restrict__ side,
                                                          const double* __restrict__ diag,
                                                          const unsigned long long* __restrict__ xg,
                                                          uint4* __restrict__ meta) {
  const int row0 = tile_row0[blockIdx.x], nrows = tile_row0[blockIdx.x + 1] - row0;
  const int rec0 = tile_rec0[blockIdx.x];
  for (int i = threadIdx.x; i < nrows; i += blockDim.x) {
    const size_t p = (size_t)row0 + i;
    const uint4 sd = side[p];
    const unsigned long long x = xg[rec0 + i];
    const long long d = __double_as_longlong(diag[p]);
    meta[2 * p] = make_uint4(sd.x, (uint32_t)x, (uint32_t)(x >> 32), sd.y);
    meta[2 * p + 1] = make_uint4(sd.z, sd.w, (uint32_t)d, (uint32_t)((unsigned long long)d >> 32));
  }
}

void free_layout(TiledLayout& l) {
  cudaFree(l.d_records);
  cudaFree(l.d_diag);
  cudaFree(l.d_side);
  cudaFree(l.d_to_other);
  cudaFree(l.d_to_natural);
  cudaFree(l.d_from_natural);
  l = TiledLayout{};
}

struct DeviceTemp {  // frees what it holds at scope exit
  std::vector<void*> p;
  ~DeviceTemp() {
    for (void* q : p) cudaFree(q);
  }
  template <class T>
  cudaError_t alloc(T** out, size_t count) {
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(out), sizeof(T) * (count ? count : 1));
    if (e == cudaSuccess) p.push_back(*out);
    return e;
  }
};

}  // namespace

void destroy_tiled_plan(TiledPlan* p) {
  if (!p) return;
  for (auto& l : p->lay) free_layout(l);
  cudaFree(p->d_tile_row0);
  cudaFree(p->d_tile_rec0);
  destroy_sector_plan(p->sector);
  delete p;
}

int build_tiled_plan(const polfed_basis* basis, const std::vector<DevTerm>& terms, bool sector,
                     cudaStream_t st, TiledPlan** out) {
  *out = nullptr;
  const int L = basis->n_sites, n_up = basis->n_up;
  if (n_up < 0 || !basis->d_states)
    return fail(POLFED_EINVAL, "tiled format: needs a fixed-particle-number basis");
  if (L < 4 || L > 2 * kTileMaxSites)
    return fail(POLFED_EINVAL, "tiled format: n_sites=%d not in [4,%d]", L, 2 * kTileMaxSites);
  const int m = (L + 1) / 2;
  int rc = ensure_binomials();
  if (rc) return rc;

  // classify: inside layout 0's low sites, inside layout 1's, else diagonal / cross-cut
  std::vector<DevTerm> low[2], dm[2];
  for (const DevTerm& t : terms) {
    DevTerm r = t;  // the same term with the site order reversed
    r.i = L - 1 - t.i;
    r.j = L - 1 - t.j;
    if (!off_diagonal(t.kind)) {
      dm[0].push_back(t);
      dm[1].push_back(r);
      continue;
    }
    if (t.kind != POLFED_TERM_EXCH && t.kind != POLFED_TERM_HOPJW)
      return fail(POLFED_EINVAL, "tiled format: only EXCH and HOPJW off-diagonal terms");
    if (std::max(t.i, t.j) < m) {
      low[0].push_back(t);
    } else if (std::max(r.i, r.j) < m) {
      low[1].push_back(r);
    } else {
      dm[0].push_back(t);
      dm[1].push_back(r);
    }
  }

  TiledPlan* p = new (std::nothrow) TiledPlan;
  if (!p) return fail(POLFED_ENOMEM, "tiled format: host allocation failed");
  struct Guard {
    TiledPlan* p;
    ~Guard() { destroy_tiled_plan(p); }
  } guard{p};
  p->n_sites = L;
  p->n_up = n_up;
  p->m = m;
  p->n = basis->dim;
  const int64_t n = p->n;
  const size_t n_alloc = (size_t)(n ? n : 1);

  std::vector<int> class_off(m + 2, 0);
  for (int k = 0; k <= m; ++k) class_off[k + 1] = class_off[k] + (int)host_binom(m, k);
  std::vector<int32_t> row0, rec0, tile_class;
  long long rows = 0;
  for (uint32_t h = 0; h < (1u << (L - m)); ++h) {
    const int k = n_up - __builtin_popcount(h);
    if (k < 0 || k > m) continue;
    row0.push_back((int32_t)rows);
    rec0.push_back(class_off[k]);
    tile_class.push_back(k);
    const int nr = (int)host_binom(m, k);
    rows += nr;
    p->max_tile_rows = std::max(p->max_tile_rows, nr);
  }
  row0.push_back((int32_t)rows);
  if (rows != n) return fail(POLFED_ECUDA, "tiled format: tile table does not cover the basis");
  p->n_tiles = (int)rec0.size();
  rc = upload(&p->d_tile_row0, row0);
  if (rc) return rc;
  rc = upload(&p->d_tile_rec0, rec0);
  if (rc) return rc;

  // The sector sweep (POLFED_FORMAT_SECTOR) needs uniform NN (+ NNN) bonds inside the tiles of
  // both layouts, at most three hops across the cut and a kernel for this tile size.
  SectorHost sh[2];
  if (sector) {
    double t1[2], t2[2];
    bool nnn[2], jw[2];
    int cross_terms = 0;
    for (const DevTerm& t : dm[0]) cross_terms += off_diagonal(t.kind) && t.amp != 0.0;
    const bool pat = m >= 2 && cross_terms <= 3 &&
                     sector_pattern(m, low[0], &t1[0], &t2[0], &nnn[0], &jw[0]) &&
                     sector_pattern(m, low[1], &t1[1], &t2[1], &nnn[1], &jw[1]) &&
                     nnn[0] == nnn[1] && (!nnn[0] || jw[0] == jw[1]) &&
                     sector_m_supported(m, nnn[0], jw[0]);
    if (!pat)
      return fail(POLFED_EINVAL, "sector format: needs one amplitude on every (i,i+1) bond and none "
                                 "or one on every (i,i+2) bond inside a tile, at most 3 hopping "
                                 "terms across the cut, and ceil(n_sites/2) in the supported set");
    {
      SectorPlan* sp = new (std::nothrow) SectorPlan;
      if (!sp) return fail(POLFED_ENOMEM, "tiled format: host allocation failed");
      p->sector = sp;
      sp->nnn = nnn[0];
      sp->jw = nnn[0] && jw[0];
      std::vector<uint16_t> units;
      sector_geometry(m, /*pad=*/false, sp, &units);
      for (int l = 0; l < 2; ++l) {
        sp->lay[l].t1 = t1[l];
        sp->lay[l].t2 = t2[l];
        sector_tables(*sp, low[l], class_off, &sh[l]);
      }
      rc = upload(&sp->d_units, units);
      if (rc) return rc;
      rc = upload(&sp->d_tile_class, tile_class);
      if (rc) return rc;
    }
  }

  DeviceTemp tmp;
  int32_t* d_pi = nullptr;
  int32_t* d_pos[2] = {nullptr, nullptr};
  int* d_max = nullptr;
  POLFED_CUDA(tmp.alloc(&d_pi, n_alloc));
  POLFED_CUDA(tmp.alloc(&d_pos[0], n_alloc));
  POLFED_CUDA(tmp.alloc(&d_pos[1], n_alloc));
  POLFED_CUDA(tmp.alloc(&d_max, 1));
  unsigned long long* d_table = nullptr;
  POLFED_CUDA(tmp.alloc(&d_table, kTileMaxCrossCoef));
  if (n >= ((int64_t)1 << kCrossPosBits))
    return fail(POLFED_EINVAL, "tiled format: dimension %lld needs more than %d position bits",
                (long long)n, kCrossPosBits);
  const unsigned row_grid = (unsigned)((n + 255) / 256);

  for (int l = 0; l < 2; ++l) {
    TiledLayout& lay = p->lay[l];
    std::vector<uint32_t> rec;
    std::vector<int32_t> inv_sigma;
    if (p->sector) {
      inv_sigma = sh[l].inv_sigma;
    } else {
      rc = build_records(m, low[l], &lay, &rec, &inv_sigma, class_off);
      if (rc) return rc;
      rc = upload(&lay.d_records, rec);
      if (rc) return rc;
    }
    int32_t* d_inv = nullptr;
    POLFED_CUDA(tmp.alloc(&d_inv, inv_sigma.size()));
    POLFED_CUDA(cudaMemcpyAsync(d_inv, inv_sigma.data(), sizeof(int32_t) * inv_sigma.size(),
                                cudaMemcpyHostToDevice, st));
    if (p->n_tiles > 0) {
      position_kernel<<<(unsigned)p->n_tiles, 256, 0, st>>>(p->d_tile_row0, p->d_tile_rec0, d_inv,
                                                            d_pos[l]);
      POLFED_LAUNCH_CHECK("position_kernel");
    }
    POLFED_CUDA(cudaStreamSynchronize(st));  // inv_sigma (host) is read by the copy above

    // diagonal + cross-cut part: CSR over the ascending rows of this layout, then by position
    int32_t* d_rp = nullptr;
    int32_t* d_col = nullptr;
    double* d_val = nullptr;
    long long nnz = 0;
    rc = assemble_csr(basis, dm[l], 0, nullptr, st, &d_rp, &d_col, &d_val, &nnz);
    if (rc) return rc;
    tmp.p.push_back(d_rp);
    tmp.p.push_back(d_col);
    tmp.p.push_back(d_val);
    int n_cross = 0;
    if (n > 0) {
      POLFED_CUDA(cudaMemsetAsync(d_max, 0, sizeof(int), st));
      max_offdiag_kernel<<<row_grid, 256, 0, st>>>(n, d_rp, d_max);
      POLFED_LAUNCH_CHECK("max_offdiag_kernel");
      POLFED_CUDA(cudaMemcpyAsync(&n_cross, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
      POLFED_CUDA(cudaStreamSynchronize(st));
    }
    if (n_cross > kTileMaxCross)
      return fail(POLFED_EINVAL, "tiled format: %d hops of one state cross the cut (limit %d)",
                  n_cross, kTileMaxCross);
    lay.n_cross = n_cross;
    POLFED_CUDA(cudaMalloc(&lay.d_diag, sizeof(double) * n_alloc));
    lay.side_words = n_cross <= 3 ? 4 : 8;
    POLFED_CUDA(cudaMalloc(&lay.d_side, sizeof(uint32_t) * n_alloc * (size_t)lay.side_words));
    POLFED_CUDA(cudaMalloc(&lay.d_to_other, sizeof(int32_t) * n_alloc));
    POLFED_CUDA(cudaMalloc(&lay.d_to_natural, sizeof(int32_t) * n_alloc));
    POLFED_CUDA(cudaMalloc(&lay.d_from_natural, sizeof(int32_t) * n_alloc));
    if (n > 0) {
      POLFED_CUDA(cudaMemsetAsync(d_table, 0, sizeof(unsigned long long) * kTileMaxCrossCoef, st));
      POLFED_CUDA(cudaMemsetAsync(d_max, 0, sizeof(int), st));
      cross_coef_kernel<<<row_grid, 256, 0, st>>>(n, d_rp, d_col, d_val, d_table, d_max);
      POLFED_LAUNCH_CHECK("cross_coef_kernel");
      dm_ell_kernel<<<row_grid, 256, 0, st>>>(n, n_cross, d_rp, d_col, d_val, d_pos[l], d_table,
                                              lay.d_diag, lay.side_words, lay.d_side);
      POLFED_LAUNCH_CHECK("dm_ell_kernel");
      int overflow = 0;
      unsigned long long table[kTileMaxCrossCoef];
      POLFED_CUDA(cudaMemcpyAsync(&overflow, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
      POLFED_CUDA(cudaMemcpyAsync(table, d_table, sizeof(table), cudaMemcpyDeviceToHost, st));
      POLFED_CUDA(cudaStreamSynchronize(st));
      if (overflow)
        return fail(POLFED_EINVAL,
                    "tiled format: more than %d distinct hopping amplitudes across the cut",
                    kTileMaxCrossCoef);
      lay.n_ccoef = 0;
      for (int c = 0; c < kTileMaxCrossCoef; ++c) {
        double mag;
        memcpy(&mag, &table[c], sizeof(double));
        lay.ccoef[c] = mag;
        if (table[c]) lay.n_ccoef = c + 1;
      }
    }
  }

  if (n > 0) {
    reverse_rank_kernel<<<row_grid, 256, 0, st>>>(n, L, n_up, basis->d_states, d_pi);
    POLFED_LAUNCH_CHECK("reverse_rank_kernel");
    maps_kernel<<<row_grid, 256, 0, st>>>(n, d_pi, d_pos[0], d_pos[1], p->lay[0].d_to_other,
                                          p->lay[1].d_to_other, p->lay[0].d_to_natural,
                                          p->lay[1].d_to_natural, p->lay[0].d_from_natural,
                                          p->lay[1].d_from_natural, p->lay[0].d_side,
                                          p->lay[0].side_words, p->lay[1].d_side,
                                          p->lay[1].side_words);
    POLFED_LAUNCH_CHECK("maps_kernel");
  }
  POLFED_CUDA(cudaStreamSynchronize(st));
  if (p->sector) {
    SectorPlan* sp = p->sector;
    for (int l = 0; l < 2; ++l) {
      TiledLayout& lay = p->lay[l];
      if (lay.side_words != 4) return fail(POLFED_ECUDA, "sector sweep: wide cut");
      unsigned long long* d_xg = nullptr;
      POLFED_CUDA(tmp.alloc(&d_xg, sh[l].xg.size()));
      POLFED_CUDA(cudaMemcpyAsync(d_xg, sh[l].xg.data(), sizeof(uint64_t) * sh[l].xg.size(),
                                  cudaMemcpyHostToDevice, st));
      POLFED_CUDA(cudaMalloc(&sp->lay[l].d_meta, sizeof(uint4) * 2 * n_alloc));
      if (p->n_tiles > 0) {
        sector_meta_kernel<<<(unsigned)p->n_tiles, 256, 0, st>>>(
            p->d_tile_row0, p->d_tile_rec0, reinterpret_cast<const uint4*>(lay.d_side), lay.d_diag,
            d_xg, sp->lay[l].d_meta);
        POLFED_LAUNCH_CHECK("sector_meta_kernel");
      }
      POLFED_CUDA(cudaStreamSynchronize(st));
      // the row records carry these now
      cudaFree(lay.d_side);
      cudaFree(lay.d_diag);
      cudaFree(lay.d_to_other);
      lay.d_side = nullptr;
      lay.d_diag = nullptr;
      lay.d_to_other = nullptr;
    }
    rc = sector_configure_launch(p, sp);
  } else {
    rc = tiled_configure_launch(p);
  }
  if (rc) return rc;
  guard.p = nullptr;
  *out = p;
  return POLFED_OK;
}

}  // namespace polfed
