// Sector sweep kernels (sector_kernel.cuh) for tiles of 4 sites (NN + NNN bonds with Jordan-Wigner sign), 5 sites (NN + NNN bonds with Jordan-Wigner sign), 6 sites (NN + NNN bonds with Jordan-Wigner sign), 7 sites (NN + NNN bonds with Jordan-Wigner sign).
#include "sector_kernel.cuh"

POLFED_SECTOR_DEF(4, 1, 1)
POLFED_SECTOR_DEF(5, 1, 1)
POLFED_SECTOR_DEF(6, 1, 1)
POLFED_SECTOR_DEF(7, 1, 1)
