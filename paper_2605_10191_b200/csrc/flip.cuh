// The flip format: the matrix-free alternative to CSR for full-space spin models whose
// off-diagonal part is a dense block on the lowest three bits plus terms that flip two bits with
// a state-independent amplitude (the quantum sun, Eq. 67; the paper's own
// matrix-free kernel for such models is Fig. 7: `newstate = state XOR mask`).
// north_star: "an evaluated alternative that ... generates rows matrix-free".  DESIGN.md 5c.
//
// Rows are the integers 0 .. 2^L - 1, so a term that flips bits i and j maps row r to r ^ mask.
// Eight consecutive rows (one configuration of bits 3 .. L-1) are a *block*; a flip term maps a
// block onto one other block (mask >> 3) and permutes the rows inside it (mask & 7).  A group of
// lanes owns a block: it holds the block of X in registers, applies the dense 8 x 8 part there
// and, per flip term, loads the eight rows of the partner block once.  No column indices, no
// values, no shuffles: per row the LSU sees 1 + n_flips row loads instead of the CSR kernel's
// 2.5 wavefronts per stored entry.
#pragma once

#include "common.cuh"

namespace polfed {

constexpr int kFlipBlockBits = 3;
constexpr int kFlipBlockRows = 1 << kFlipBlockBits;
constexpr int kFlipMaxTerms = 64;

struct FlipTerms {                 // passed to the kernel by value
  int n_flips;
  uint32_t hi[kFlipMaxTerms];      // partner block = block ^ hi
  uint32_t lo[kFlipMaxTerms];      // partner row inside it = row ^ lo
  double amp[kFlipMaxTerms];
  double dense[kFlipBlockRows * kFlipBlockRows];  // [r][c], diagonal zero (it is in `diag`)
};

struct FlipPlan {
  FlipTerms terms;
  double* d_diag = nullptr;        // [n] diagonal of H
};

}  // namespace polfed
