// Sector sweep kernels (sector_kernel.cuh) for tiles of 13 sites (NN + NNN bonds with Jordan-Wigner sign).
#include "sector_kernel.cuh"

POLFED_SECTOR_DEF(13, 1, 1)
