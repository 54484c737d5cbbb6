// Construction of the tiled format (tiled.cuh): term classification, per-class neighbour
// records, tile table, the layout permutation and the two diagonal + cross-cut CSR parts.
#include <algorithm>
#include <new>

#include "combinadic.cuh"
#include "tiled.cuh"

namespace polfed {

int tiled_configure_launch(TiledPlan* plan);  // tiled_sweep.cu

namespace {

// Row of state x in the layout with the site order reversed.
__global__ void __launch_bounds__(256) reverse_rank_kernel(int64_t n, int n_sites, int n_up,
                                                           const uint64_t* __restrict__ states,
                                                           int32_t* __restrict__ pi) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n) return;
  const uint64_t y = __brevll(states[r]) >> (64 - n_sites);
  pi[r] = (int32_t)rank_state(y, n_sites, n_up);
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

// Records of one layout: `low` holds the tile-local hops with sites already in this layout's
// numbering (all < m).  Class k (k particles on the low m sites) owns records
// class_off[k] .. class_off[k+1]; they are sorted by falling degree so that the rows a warp
// works on together have (nearly) the same number of neighbours.  Record = 16 words:
//   word 0      row index inside the tile (bits 0-10) | degree (bits 16-20)
//   words 1-12  24 entries of 16 bits: neighbour row (bits 0-10) | amplitude class (bits 11-12)
//               | sign (bit 15); unused entries point at the zero row (index = rows of the class)
int build_records(int m, const std::vector<DevTerm>& low, TiledLayout* lay,
                  std::vector<uint32_t>* rec, const std::vector<int>& class_off) {
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
  rec->assign((size_t)(1u << m) * kTileRecWords, 0u);
  std::vector<std::vector<uint16_t>> ent((size_t)1 << m);  // by class_off[k] + class_rank(l)
  for (uint32_t l = 0; l < (1u << m); ++l) {
    const int k = __builtin_popcount(l);
    std::vector<uint16_t>& e = ent[(size_t)class_off[k] + class_rank(l)];
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
      e.push_back((uint16_t)(class_rank(l2) | ((uint32_t)cls[t] << 11) | (sign << 15)));
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
    for (int t = 0; t < n_k; ++t) {
      const std::vector<uint16_t>& e = ent[(size_t)class_off[k] + order[t]];
      uint32_t* w = rec->data() + ((size_t)class_off[k] + t) * kTileRecWords;
      w[0] = (uint32_t)order[t] | ((uint32_t)e.size() << 16);
      for (int j = 0; j < kTileMaxDeg; ++j) {
        const uint32_t v = j < (int)e.size() ? e[j] : (uint32_t)n_k;  // zero row
        w[1 + (j >> 1)] |= v << (16 * (j & 1));
      }
    }
  }
  return POLFED_OK;
}

}  // namespace

void destroy_tiled_plan(TiledPlan* p) {
  if (!p) return;
  for (auto& l : p->lay) {
    cudaFree(l.d_dm_row_ptr);
    cudaFree(l.d_dm_col);
    cudaFree(l.d_dm_val);
    cudaFree(l.d_records);
  }
  cudaFree(p->d_tile_row0);
  cudaFree(p->d_tile_rec0);
  cudaFree(p->d_pi);
  cudaFree(p->d_counter);
  delete p;
}

int build_tiled_plan(const polfed_basis* basis, const std::vector<DevTerm>& terms, cudaStream_t st,
                     TiledPlan** out) {
  *out = nullptr;
  const int L = basis->n_sites, n_up = basis->n_up;
  if (n_up < 0 || !basis->d_states)
    return fail(POLFED_EINVAL, "tiled format: needs a fixed-particle-number basis");
  const int m = (L + 1) / 2;
  if (L < 4 || m > kTileMaxSites)
    return fail(POLFED_EINVAL, "tiled format: n_sites=%d not in [4,%d]", L, 2 * kTileMaxSites);
  int rc = ensure_binomials();
  if (rc) return rc;

  // classify: A = inside layout 0's low sites, B = inside layout 1's, else cross-cut
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

  std::vector<int> class_off(m + 2, 0);
  for (int k = 0; k <= m; ++k) class_off[k + 1] = class_off[k] + (int)host_binom(m, k);
  std::vector<int32_t> row0, rec0;
  long long rows = 0;
  for (uint32_t h = 0; h < (1u << (L - m)); ++h) {
    const int k = n_up - __builtin_popcount(h);
    if (k < 0 || k > m) continue;
    row0.push_back((int32_t)rows);
    rec0.push_back(class_off[k]);
    const int nr = (int)host_binom(m, k);
    rows += nr;
    p->max_tile_rows = std::max(p->max_tile_rows, nr);
  }
  row0.push_back((int32_t)rows);
  if (rows != p->n) return fail(POLFED_ECUDA, "tiled format: tile table does not cover the basis");
  p->n_tiles = (int)rec0.size();
  rc = upload(&p->d_tile_row0, row0);
  if (rc) return rc;
  rc = upload(&p->d_tile_rec0, rec0);
  if (rc) return rc;

  for (int l = 0; l < 2; ++l) {
    std::vector<uint32_t> rec;
    rc = build_records(m, low[l], &p->lay[l], &rec, class_off);
    if (rc) return rc;
    rc = upload(&p->lay[l].d_records, rec);
    if (rc) return rc;
    rc = assemble_csr(basis, dm[l], 0, nullptr, st, &p->lay[l].d_dm_row_ptr, &p->lay[l].d_dm_col,
                      &p->lay[l].d_dm_val, &p->lay[l].dm_nnz);
    if (rc) return rc;
  }

  POLFED_CUDA(cudaMalloc(&p->d_pi, sizeof(int32_t) * (size_t)(p->n ? p->n : 1)));
  if (p->n > 0) {
    reverse_rank_kernel<<<(unsigned)((p->n + 255) / 256), 256, 0, st>>>(p->n, L, n_up,
                                                                       basis->d_states, p->d_pi);
    POLFED_LAUNCH_CHECK("reverse_rank_kernel");
  }
  POLFED_CUDA(cudaMalloc(&p->d_counter, sizeof(int)));
  POLFED_CUDA(cudaMemsetAsync(p->d_counter, 0, sizeof(int), st));
  POLFED_CUDA(cudaStreamSynchronize(st));
  rc = tiled_configure_launch(p);
  if (rc) return rc;
  guard.p = nullptr;
  *out = p;
  return POLFED_OK;
}

}  // namespace polfed
