// The tiled format: the structured alternative to CSR for number-conserving chains
// (north_star: "an evaluated alternative that exploits constant off-diagonal values or generates
// rows matrix-free"; the paper's "optimized mapping").  DESIGN.md section 5b.
//
// Idea.  States are ascending integers, so all states that share their top (n_sites - m) bits
// form one contiguous run of rows -- a *tile* -- and every hop between two of the low m sites
// stays inside the tile.  Inside a tile those hops are the same small graph for every tile of
// the same low-part particle number k (a *class*): one 64-byte record per class row lists the
// in-tile neighbours (index, amplitude class, sign).  A CTA keeps the tile of X in shared
// memory, so these gathers never leave the SM.
// The hops among the high sites are not tile-local in this labelling, but they are in the
// labelling with the site order reversed (layout 1).  The Clenshaw recurrence is therefore run
// as a pipeline of sweeps that alternate between the two layouts: the sweep in layout l
//   finishes  b_k     = P_k + p_k (O_l + DM) b_{k+1}                       (phase 2)
//   starts    P_{k-1} = c_{k-1} V + p_{k-1} O_l b_k + q_{k-1} b_k - b_{k+1} (phase 3)
// and writes both row-permuted into the other layout, where the next sweep finishes b_{k-1}
// with its own tile-local part O_{1-l}.  O_l = hops inside layout l's low m sites, DM = diagonal
// plus the few hops that cross the cut.  One sweep per recurrence step, five block passes of HBM
// traffic, no far gathers.
//
// Row order.  Inside a tile the rows of a layout are stored in *processing order*: the rows of a
// class sorted by falling in-tile degree ("position").  A warp works on 8 consecutive positions,
// so its rows have (nearly) the same number of neighbours and every per-row stream (partial sums,
// V, diagonal, cross-cut entries, records) is one contiguous run per warp instruction.  The maps
// between positions of the two layouts and the caller's natural row order are part of the plan.
#pragma once

#include "common.cuh"

namespace polfed {

constexpr int kTileMaxSites = 13;     // C(13,6) rows x 128 B = 219 648 B of shared memory
constexpr int kTileRecWords = 16;     // 64-byte record per class row
constexpr int kTileMaxDeg = 24;       // in-tile neighbours per row (12 entry words)
constexpr int kTileMaxCoef = 4;       // distinct |amplitude| values per layout
constexpr int kTileMaxCross = 7;      // cross-cut neighbours per row
constexpr int kTileMaxCrossCoef = 15; // distinct |amplitude| values among the cross-cut hops
constexpr uint32_t kCrossNone = 0xffffffffu;
constexpr int kCrossPosBits = 26;     // cross word: bits 0-25 position, 26-29 amplitude, 31 sign
constexpr int kTilePanel = 16;        // columns per panel: 128-byte rows, conflict-free in smem
constexpr int kTileThreads = 448;       // one CTA per SM (tiles that fill the shared memory);
                                        // measured on config 5 with the register cap of the sweep
                                        // kernel, ms per sweep: 352: 4.62, 384: 4.61, 416: 4.53,
                                        // 448: 4.51, 480: 4.56, 512: 4.67
constexpr int kTileSmallThreads = 256;  // kTileSmallCtas CTAs per SM (small tiles)
constexpr int kTileSmallCtas = 3;

// Record of one class row (position order), kTileRecWords words:
//   word 0      in-tile degree
//   words 1-12  two neighbours per word:
//                 bits  7-17  position of neighbour A inside the tile     (x 128 = byte offset)
//                 bits 18-28  position of neighbour B
//                 bits  0-1   amplitude class of A      bits 2-3  amplitude class of B
//                 bit  30     sign of A                 bit  31   sign of B
//               unused entries point at the zero row (position = rows of the class)
struct TiledLayout {
  uint32_t* d_records = nullptr;      // [2^m][kTileRecWords], class blocks in position order
  double* d_diag = nullptr;           // [n] diagonal of H by position
  uint32_t* d_side = nullptr;         // [n][side_words]: position in the other layout, then the
                                      // packed cross-cut neighbours (kCrossNone = none)
  int side_words = 4;                 // 4 (n_cross <= 3) or 8
  int n_cross = 0;
  double ccoef[kTileMaxCrossCoef + 1] = {};  // |amplitude| table of the cross-cut hops
  int n_ccoef = 0;
  int32_t* d_to_other = nullptr;      // [n] position in the other layout
  int32_t* d_to_natural = nullptr;    // [n] row in the caller's order
  int32_t* d_from_natural = nullptr;  // [n] position of the caller's row
  double coef[kTileMaxCoef] = {0, 0, 0, 0};
  int n_coef = 0;
};

struct SectorPlan;  // sector.cuh

struct TiledPlan {
  int n_sites = 0, n_up = 0, m = 0;
  int64_t n = 0;
  int n_tiles = 0;
  int max_tile_rows = 0;
  int grid = 0;                     // persistent CTAs
  int threads = kTileThreads;       // threads per CTA (kTileThreads or kTileSmallThreads)
  size_t smem_bytes = 0;
  int32_t* d_tile_row0 = nullptr;   // [n_tiles + 1]
  int32_t* d_tile_rec0 = nullptr;   // [n_tiles] first record row of the tile's class
  SectorPlan* sector = nullptr;     // the sector sweep takes over (uniform NN/NNN bonds)
  TiledLayout lay[2];
};

}  // namespace polfed
