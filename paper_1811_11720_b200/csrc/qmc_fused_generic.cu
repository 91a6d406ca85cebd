// Dedicated kernels of the generic weight transforms (fused_generic_kernel, qmc_fused.cuh); compiled once per
// (-DQMC_FAM=0, 1, 2 or 4, -DQMC_KIND=<GEN_* kind>) by build.py.  Only kind 0, the symmetric Korobov weights, is built and
// routed (kGenKinds): Korobov (r0, r1) and Sidi compile here too but ran slower than the generic loop.
#ifndef QMC_FAM
#error "compile with -DQMC_FAM=<family> -DQMC_KIND=<GEN_* kind> (see paper_1811_11720_b200/build.py)"
#endif
#include "qmc_kernels.h"
#include "qmc_fused.cuh"

namespace qmc {

#define QMC_CAT3_(a, b, c, d) a##b##c##d
#define QMC_CAT3(a, b, c, d) QMC_CAT3_(a, b, c, d)

template <int DP> static cudaError_t launch_one(int grid, cudaStream_t st, const FusedLaunch& a) {
    fused_generic_kernel<QMC_FAM, DP, kGroup, TR_GEN0 + QMC_KIND><<<grid, kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
template <int DP> static int occ_one() {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fused_generic_kernel<QMC_FAM, DP, kGroup, TR_GEN0 + QMC_KIND>, kThreads, 0) != cudaSuccess) return -1;
    return nb;
}

#define QMC_GENERIC_TABLE(FN, ...)                \
    switch (dp) {                                 \
        case 4: return FN<4>(__VA_ARGS__);        \
        case 6: return FN<6>(__VA_ARGS__);        \
        case 8: return FN<8>(__VA_ARGS__);        \
        case 12: return FN<12>(__VA_ARGS__);      \
        case 16: return FN<16>(__VA_ARGS__);      \
    }

cudaError_t QMC_CAT3(launch_fused_generic_, QMC_FAM, _, QMC_KIND)(int dp, int grid, cudaStream_t st, const FusedLaunch& a) {
    QMC_GENERIC_TABLE(launch_one, grid, st, a)
    return cudaErrorInvalidValue;
}
int QMC_CAT3(occupancy_fused_generic_, QMC_FAM, _, QMC_KIND)(int dp) {
    QMC_GENERIC_TABLE(occ_one)
    return -1;
}

}  // namespace qmc
