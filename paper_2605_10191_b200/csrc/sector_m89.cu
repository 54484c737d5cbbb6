// Sector sweep kernels (sector_kernel.cuh) for tiles of 8 sites (NN + NNN bonds with Jordan-Wigner sign), 9 sites (NN + NNN bonds with Jordan-Wigner sign).
#include "sector_kernel.cuh"

POLFED_SECTOR_DEF(8, 1, 1)
POLFED_SECTOR_DEF(9, 1, 1)
