// qmc_spec.h -- what the launch plan (qmc_host.cu) needs to know about a module of specialised sector kernels (qmc_spec.cu).
#pragma once
#include <cuda_runtime.h>

#include "qmc_internal.h"

struct qmc_sector_module;

namespace qmc {

constexpr int kKernelFamilySpec = kKernelFamilies;     // variant key of a specialised kernel (never indexes the occupancy cache)

struct SpecProblem {              // one record per problem the module was built from
    int family, dim, n_params;
    int kernel, kase;             // the kernel that holds the problem's code and its case there; kernel < 0: not specialised
};

int spec_problem_count(const qmc_sector_module* mod);
const SpecProblem* spec_problems(const qmc_sector_module* mod);
int spec_kernel_dp(const qmc_sector_module* mod, int kernel);
int spec_kernel_threads(const qmc_sector_module* mod, int kernel);
// both load the module on the current device on first use; occupancy <= 0 and a launch error are CUDA failures whose text is
// left with report_cuda_error
int spec_occupancy(qmc_sector_module* mod, int kernel);
int spec_launch(qmc_sector_module* mod, int kernel, int grid, cudaStream_t st, const FusedLaunch& a);

}  // namespace qmc
