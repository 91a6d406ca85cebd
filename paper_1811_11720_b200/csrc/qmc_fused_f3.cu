// Fused R1SL kernels of the sector-like family (interpreted integrand, see qmc_sector.cuh).
#include "qmc_sector.cuh"
#include "qmc_kernels.h"

namespace qmc {

template <int DP, bool WIDE> static cudaError_t launch_one(int grid, cudaStream_t st, const FusedLaunch& a) {
    fused_sector_kernel<DP, SectorGroup<DP>::value, WIDE><<<grid, kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
template <int DP, bool WIDE> static int occ_one() {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fused_sector_kernel<DP, SectorGroup<DP>::value, WIDE>, kThreads, 0) !=
        cudaSuccess)
        return -1;
    return nb;
}

#define QMC_F3_TABLE(FN, ...)                                    \
    switch (dp * 2 + (wide ? 1 : 0)) {                            \
        case 4 * 2: return FN<4, false>(__VA_ARGS__);             \
        case 4 * 2 + 1: return FN<4, true>(__VA_ARGS__);          \
        case 6 * 2: return FN<6, false>(__VA_ARGS__);             \
        case 6 * 2 + 1: return FN<6, true>(__VA_ARGS__);          \
        case 8 * 2: return FN<8, false>(__VA_ARGS__);             \
        case 8 * 2 + 1: return FN<8, true>(__VA_ARGS__);          \
        case 16 * 2: return FN<16, false>(__VA_ARGS__);           \
        case 16 * 2 + 1: return FN<16, true>(__VA_ARGS__);        \
    }

cudaError_t launch_fused_f3(int dp, bool wide, int grid, cudaStream_t st, const FusedLaunch& a) {
    QMC_F3_TABLE(launch_one, grid, st, a)
    return cudaErrorInvalidValue;
}
int occupancy_fused_f3(int dp, bool wide) {
    QMC_F3_TABLE(occ_one)
    return -1;
}
int group_fused_f3(int dp) { return dp <= 8 ? SectorGroup<8>::value : SectorGroup<16>::value; }

}  // namespace qmc
