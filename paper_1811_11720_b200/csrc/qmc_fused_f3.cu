// Fused R1SL kernels of the sector-like family with real coefficients (interpreted integrand, see qmc_sector.cuh).
#define QMC_SECTOR_CPLX 0
#include "qmc_fused_sector.inc"
