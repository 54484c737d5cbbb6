// The tiled format: the structured alternative to CSR for number-conserving chains
// (north_star: "an evaluated alternative that exploits constant off-diagonal values or generates
// rows matrix-free"; the paper's "optimized mapping").  DESIGN.md section 5b.
//
// Idea.  States are ascending integers, so all states that share their top (n_sites - m) bits
// form one contiguous run of rows -- a *tile* -- and every hop between two of the low m sites
// stays inside the tile.  Inside a tile those hops are the same small graph for every tile of
// the same low-part particle number k (a *class*): one 64-byte record per class row lists the
// in-tile neighbours (index + sign), grouped by the few distinct amplitudes.  A CTA keeps the
// tile of X in shared memory, so these gathers never leave the SM.
// The hops among the high sites are not tile-local in this labelling, but they are in the
// labelling with the site order reversed (layout 1).  The Clenshaw recurrence is therefore run
// as a pipeline of sweeps that alternate between the two layouts: the sweep in layout l
//   finishes  b_k     = P_k + p_k (O_l + DM) b_{k+1}                       (phase 2)
//   starts    P_{k-1} = c_{k-1} V + p_{k-1} O_l b_k + q_{k-1} b_k - b_{k+1} (phase 3)
// and writes both row-permuted into the other layout, where the next sweep finishes b_{k-1}
// with its own tile-local part O_{1-l}.  O_l = hops inside layout l's low m sites, DM = diagonal
// plus the few hops that cross the cut (a small CSR per layout, gathered from global memory).
// One sweep per recurrence step, five block passes of HBM traffic, no far gathers.
#pragma once

#include "common.cuh"

namespace polfed {

constexpr int kTileMaxSites = 13;     // C(13,6) rows x 128 B = 219 648 B of shared memory
constexpr int kTileRecWords = 16;     // 64-byte record per class row
constexpr int kTileMaxDeg = 24;       // in-tile neighbours per row (12 entry words)
constexpr int kTileMaxCoef = 4;       // distinct |amplitude| values per layout
constexpr int kTilePanel = 16;        // columns per panel: 128-byte rows, conflict-free in smem
constexpr int kTileThreads = 1024;

struct TiledLayout {
  int32_t* d_dm_row_ptr = nullptr;  // diagonal + cross-cut terms, CSR in this layout's row order
  int32_t* d_dm_col = nullptr;
  double* d_dm_val = nullptr;
  long long dm_nnz = 0;
  uint32_t* d_records = nullptr;    // [n_class_rows][kTileRecWords]
  double coef[kTileMaxCoef] = {0, 0, 0, 0};
  int n_coef = 0;
};

struct TiledPlan {
  int n_sites = 0, n_up = 0, m = 0;
  int64_t n = 0;
  int n_tiles = 0;
  int max_tile_rows = 0;
  int grid = 0;                     // persistent CTAs
  size_t smem_bytes = 0;
  int32_t* d_tile_row0 = nullptr;   // [n_tiles + 1]
  int32_t* d_tile_rec0 = nullptr;   // [n_tiles] first record row of the tile's class
  int32_t* d_pi = nullptr;          // [n] row in the other layout (an involution)
  int* d_counter = nullptr;         // dynamic tile scheduler
  TiledLayout lay[2];
};

}  // namespace polfed
