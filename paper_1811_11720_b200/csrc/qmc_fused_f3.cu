// Fused R1SL kernels of the sector-like family (interpreted integrand, see qmc_sector.cuh).
#include "qmc_sector.cuh"
#include "qmc_kernels.h"

namespace qmc {

template <int DP, int G, bool WIDE> static cudaError_t launch_one(int grid, cudaStream_t st, const FusedArgs& a,
                                                                  const unsigned long long* prog) {
    fused_sector_kernel<DP, G, WIDE><<<grid, kThreads, 0, st>>>(a.probs, a.aux, a.vq, a.partials, prog);
    return cudaGetLastError();
}
template <int DP, int G, bool WIDE> static int occ_one() {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fused_sector_kernel<DP, G, WIDE>, kThreads, 0) != cudaSuccess) return -1;
    return nb;
}

cudaError_t launch_fused_f3(int dp, bool wide, int grid, cudaStream_t st, const FusedArgs& a, const unsigned long long* prog) {
    switch (dp * 2 + (wide ? 1 : 0)) {
        case 4 * 2: return launch_one<4, kGroup, false>(grid, st, a, prog);
        case 4 * 2 + 1: return launch_one<4, kGroup, true>(grid, st, a, prog);
        case 8 * 2: return launch_one<8, kGroup, false>(grid, st, a, prog);
        case 8 * 2 + 1: return launch_one<8, kGroup, true>(grid, st, a, prog);
        case 16 * 2: return launch_one<16, 2, false>(grid, st, a, prog);
        case 16 * 2 + 1: return launch_one<16, 2, true>(grid, st, a, prog);
    }
    return cudaErrorInvalidValue;
}
int occupancy_fused_f3(int dp, bool wide) {
    switch (dp * 2 + (wide ? 1 : 0)) {
        case 4 * 2: return occ_one<4, kGroup, false>();
        case 4 * 2 + 1: return occ_one<4, kGroup, true>();
        case 8 * 2: return occ_one<8, kGroup, false>();
        case 8 * 2 + 1: return occ_one<8, kGroup, true>();
        case 16 * 2: return occ_one<16, 2, false>();
        case 16 * 2 + 1: return occ_one<16, 2, true>();
    }
    return -1;
}

}  // namespace qmc
