// Fused R1SL kernels of integrand family 0 (see qmc_fused.cuh); one translation unit per family so
// that the families compile in parallel.
#define QMC_FAM 0
#include "qmc_fused_closed.inc"
