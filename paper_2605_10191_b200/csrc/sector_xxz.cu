// Sector sweep kernels (sector_kernel.cuh) for tiles of 6 sites (NN bonds only), 7 sites (NN bonds only), 8 sites (NN bonds only), 10 sites (NN bonds only).
#include "sector_kernel.cuh"

POLFED_SECTOR_DEF(6, 0, 0)
POLFED_SECTOR_DEF(7, 0, 0)
POLFED_SECTOR_DEF(8, 0, 0)
POLFED_SECTOR_DEF(10, 0, 0)
