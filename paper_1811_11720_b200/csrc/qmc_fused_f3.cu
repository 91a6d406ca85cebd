// Fused R1SL kernels of the sector-like family (interpreted integrand, see qmc_sector.cuh).
#include "qmc_sector.cuh"
#include "qmc_kernels.h"

namespace qmc {

// one CTA per SM, dynamic shared memory (the parked weights and U of 256 / 384 threads exceed the static 48 KB)
template <int DP, bool WIDE> static cudaError_t launch_one(int grid, cudaStream_t st, const FusedLaunch& a) {
    constexpr int G = SectorGroup<DP>::value, NT = SectorThreads<DP>::value;
    constexpr size_t smem = sizeof(SectorShared<DP, G, NT>);
    cudaError_t e = cudaFuncSetAttribute(fused_sector_kernel<DP, G, WIDE, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    fused_sector_kernel<DP, G, WIDE, NT><<<grid, NT, smem, st>>>(a);
    return cudaGetLastError();
}
template <int DP, bool WIDE> static int occ_one() {
    constexpr int G = SectorGroup<DP>::value, NT = SectorThreads<DP>::value;
    constexpr size_t smem = sizeof(SectorShared<DP, G, NT>);
    int nb = 0;
    if (cudaFuncSetAttribute(fused_sector_kernel<DP, G, WIDE, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fused_sector_kernel<DP, G, WIDE, NT>, NT, smem) != cudaSuccess) return -1;
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

}  // namespace qmc
