// Fused R1SL kernels of the closed-form integrand families (see qmc_fused.cuh); compiled once per
// (-DQMC_FAM=0, 1, 2 or 4, -DQMC_PART=0..3) by build.py so that the variants build in parallel.
#ifndef QMC_FAM
#error "compile with -DQMC_FAM=<family> -DQMC_PART=<part> (see paper_1811_11720_b200/build.py)"
#endif
#include "qmc_kernels.h"
#include "qmc_fused_closed.inc"
