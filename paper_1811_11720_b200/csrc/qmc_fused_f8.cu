// Fused R1SL kernels of the sector family with complex coefficients (reading C-16; see qmc_sector.cuh).
#define QMC_SECTOR_CPLX 1
#include "qmc_fused_sector.inc"
