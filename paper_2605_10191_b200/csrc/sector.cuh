// The sector sweep: the tiled format (tiled.cuh) for chains whose tile-local hops are uniform
// nearest- and next-nearest-neighbour bonds (config 5: t, t' with Jordan-Wigner sign; XXZ: J/2).
// DESIGN.md section 5d.  Same alternating-layout Clenshaw pipeline (Eq. 51),
// same two phases per sweep, but the tile-local part O_l is applied from REGISTERS:
//
// The m tile sites are split into a low group G1 (g1 sites) and a high group G2 (g2 = m - g1).
// The rows of a tile with j1 particles on G1 and j2 on G2 form a *sector*, a full tensor product
// C(g1,j1) x C(g2,j2), stored row = base + i2 * n1 + i1.  Hops inside G1 keep (j1, i2): a lane
// group that holds the n1 rows (i1 = 0..n1-1, fixed i2) -- a G1-fibre -- in registers applies all
// of them without touching memory again (view 1); hops inside G2 keep (j1, i1): the same with a
// G2-fibre (view 2).  Both operators are compile-time structures (fold expressions over bonds
// and rows), so there are no neighbour records, no shuffles and no index arithmetic per entry.
// Shared memory holds the tile panel twice (64-byte rows: 8 columns): buffer A with b_{k+1}, buffer B
// with the G1 part, then b_k.  Per row and phase the shared-memory pipe sees about 5 accesses
// instead of one per stored off-diagonal; only the (at most three) bonds between G1 and G2 and
// the bonds across the tile cut remain per-row gathers.
#pragma once

#include "tiled.cuh"

namespace polfed {

constexpr int kSecPanel = 8;       // columns per panel: 64-byte rows
constexpr int kSecMaxG = 7;        // sites per group (C(7,3) = 35 rows of a fibre in registers)
constexpr int kSecThreads = 512;
constexpr int kSecMaxUnits = 48;   // work units per class and view
// Sites of the low group G1.  C(g1, j) should be odd for every j (g1 = 2^t - 1): four G1-fibres
// that a warp reads together then start at alternating 64-byte halves of the 128-byte bank row,
// so view 1 is free of bank conflicts without any padding.  m = 13 -> 7 + 6, m = 7 -> 3 + 4.
constexpr int sector_g1(int m) { return m >= 10 ? 7 : (m >= 4 ? 3 : 1); }
constexpr int kSecGroups = 4;      // lane groups (fibres) per warp: 8 lanes x 8 bytes per row

// cross-group entry (16 bits; slot 0: the (g1-1, g1) bond with amplitude t1, slots 1 and 2: the
// (g1-2, g1) and (g1-1, g1+1) bonds with amplitude t2): bits 0-10 shared-memory row of the
// partner, bit 11 valid, bit 13 negative (Jordan-Wigner sign)
constexpr uint32_t kXgValid = 0x800u, kXgNeg = 0x2000u, kXgRow = 0x7ffu;

struct SectorTables {  // passed to the kernel by value
  short sbase[kTileMaxSites + 1][kSecMaxG + 1];  // [k][j1] first in-class position of the sector
  short srow[kTileMaxSites + 1][kSecMaxG + 1];   // [k][j1] first shared-memory row of the sector
  short n1[kSecMaxG + 1], n1p[kSecMaxG + 1];     // C(g1, j1) and the fibre pitch in shared memory
  short n2[kSecMaxG + 1];                        // C(g2, j2)
  short n_units[2][kTileMaxSites + 1];           // [view][k]
  short rows_p[kTileMaxSites + 1];               // shared-memory rows of class k (with padding)
};

struct SectorLayout {
  // per position, 32 bytes: {other-layout position, xg 0|1, xg 2|own shared-memory row, cross 0}
  // {cross 1, cross 2, diag}
  uint4* d_meta = nullptr;
  double t1 = 0.0, t2 = 0.0;  // signed amplitudes of the (i,i+1) and (i,i+2) bonds
};

struct SectorPlan {
  int m = 0, g1 = 0, g2 = 0;
  bool nnn = false, jw = false;
  SectorTables tab{};
  uint16_t* d_units = nullptr;    // [2][m+1][kSecMaxUnits]: j1 | quad << 3, falling cost
  int32_t* d_tile_class = nullptr;  // [n_tiles] particles on the tile sites
  int max_rows_p = 0;             // padded rows of the largest class
  size_t smem_bytes = 0;
  int grid = 0;
  SectorLayout lay[2];
};

// sector_sweep.cu
bool sector_m_supported(int m, bool nnn, bool jw);
int sector_configure_launch(const TiledPlan* tp, SectorPlan* sp);
void destroy_sector_plan(SectorPlan* sp);

}  // namespace polfed
