// qmc_kernels.h -- host-callable launchers of the CUDA path (implemented in the .cu files).
#pragma once
#include <cuda_runtime.h>

#include "qmc_internal.h"

namespace qmc {


struct PointsArgs {
    unsigned long long n, k0, count;
    double inv_n;
    int dim;
    unsigned long long z[QMC_MAX_DIM];
    double shift[QMC_MAX_DIM];
    unsigned long long* out_r;
    double* out_u;
};

// records a CUDA error for qmc_last_cuda_error() and returns QMC_ERR_CUDA (qmc_host.cu)
int report_cuda_error(cudaError_t e, const char* where);

// a batch call for internal callers (qmc_host.cu): problems may be a selection of a module's batch, results go to chosen rows
size_t routed_workspace_bytes(int count, const qmc_problem* problems, const qmc_sector_module* module, const int* module_index);
int run_batch_routed(int count, const qmc_problem* problems, double* out_means, double* out_errs, double* out_shift_means,
                     void* workspace, size_t workspace_bytes, cudaStream_t st, qmc_sector_module* module, const int* module_index,
                     const int* out_row, int sm_stride);

cudaError_t launch_prepare(int count, cudaStream_t st, const DevProblem* probs, DevAux* aux, unsigned long long* prog_area);
cudaError_t launch_finalize(int count, cudaStream_t st, const FusedLaunch& a, double* means_ws, double* out_means, double* out_errs,
                            double* out_shift_means, int stride);
cudaError_t launch_finalize_means(cudaStream_t st, const double* means, int m, int nc, double* out_mean, double* out_err);
cudaError_t launch_points(cudaStream_t st, const PointsArgs& a, int sm_count);
cudaError_t launch_dfma_probe(cudaStream_t st, double* out, int blocks, int iters);

// fused kernels: closed-form families 0-2 in parts (qmc_fused_closed.inc), the sector family in qmc_fused_f3.cu
#define QMC_DECLARE_PART(FAM, PART)                                                                                         \
    cudaError_t launch_fused_part_##FAM##_##PART(int dp, bool wide, int group, int grid, cudaStream_t st, const FusedLaunch& a); \
    int occupancy_fused_part_##FAM##_##PART(int dp, bool wide, int group);
#define QMC_DECLARE_FAMILY(FAM) QMC_DECLARE_PART(FAM, 0) QMC_DECLARE_PART(FAM, 1) QMC_DECLARE_PART(FAM, 2) QMC_DECLARE_PART(FAM, 3)
QMC_DECLARE_FAMILY(0) QMC_DECLARE_FAMILY(1) QMC_DECLARE_FAMILY(2) QMC_DECLARE_FAMILY(4)
QMC_DECLARE_PART(1, 4)     // product peak, <= 8 slots, 8 shifts per group
#undef QMC_DECLARE_FAMILY
#undef QMC_DECLARE_PART
// dedicated kernels of the generic weight transforms (qmc_fused_generic.cu): family x GEN_* kind
#define QMC_DECLARE_GENERIC(FAM, KIND)                                                                              \
    cudaError_t launch_fused_generic_##FAM##_##KIND(int dp, int grid, cudaStream_t st, const FusedLaunch& a);       \
    int occupancy_fused_generic_##FAM##_##KIND(int dp);
#define QMC_DECLARE_GENERIC_FAMILY(FAM) QMC_DECLARE_GENERIC(FAM, 0)
QMC_DECLARE_GENERIC_FAMILY(0) QMC_DECLARE_GENERIC_FAMILY(1) QMC_DECLARE_GENERIC_FAMILY(2) QMC_DECLARE_GENERIC_FAMILY(4)
#undef QMC_DECLARE_GENERIC_FAMILY
#undef QMC_DECLARE_GENERIC
cudaError_t launch_fused_f3(int dp, bool wide, int grid, cudaStream_t st, const FusedLaunch& a);
int occupancy_fused_f3(int dp, bool wide);
cudaError_t launch_fused_f8(int dp, bool wide, int grid, cudaStream_t st, const FusedLaunch& a);   // complex sector family
int occupancy_fused_f8(int dp, bool wide);

}  // namespace qmc
