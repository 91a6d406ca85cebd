// qmc_spec_template.cu -- the fused sector kernel with a hole where the sector's polynomials go.
//
// The paper's integrands are compiled functors (every sector is a C++ function compiled by nvcc); the C ABI
// takes parameter blocks instead, which the default kernel (qmc_sector.cuh) interprets step by step.  This translation unit
// is the other route: it is compiled to PTX ONLY (build.py: nvcc -ptx) and embedded in the library as text; at run time
// qmc_sector_module_create (qmc_spec.cu) replaces the marker line of sector_poly_site with the straight-line code of the
// sectors of a batch -- coefficients as immediates, exponents unrolled, the Horner form of compile_polynomial -- and
// assembles the result for sm_100a (nvPTXCompiler).  Everything but the hole is the code of the interpreting kernel: tile
// queue, lattice points, transform, reductions (qmc_fused.cuh).
//
// Only the default tile loop exists here (Korobov-3, no fit map, n < 2^31: the paper's setting for loop integrals);
// the host routes every other problem to the interpreting kernel.
#include "qmc_sector.cuh"

namespace qmc {

#include "qmc_sector_site.inc"

template <int DP, int G, int NT> struct SectorEvalSpec {
    static constexpr int NC = 1;
    typedef unsigned Extra;                                  // shared address of the CTA's SectorSmem
    static __device__ __forceinline__ void eval(const typename Res<false>::T (&r)[DP], const SmemCtx<DP, G, NT>&, const unsigned& exbase,
                                                const EvalCtx& cx, double (&acc)[G][1]) {
        double x[G][DP], W[G];
        sector_coords<DP, G, false, TR_KOR3, 0>(r, cx, x, W);
        const unsigned park = exbase + SectorOff::park + 8u * threadIdx.x;
        const unsigned sel = (unsigned)(lds_u64(exbase + SectorOff::logp) >> 32);
        // num = W prod_j x_j^nu_j U^a, den = F^b, F; a sector with a log factor also parks U in rows 8 + q
        double num[G], den[G], F[G];
        sector_poly_site<DP, G>(x, W, sel, park, num, den, F);
        const int lp = (int)(unsigned)lds_u64(exbase + SectorOff::logp);
        if (lp) {                                             // (lu log U + lf log F)^p: a cold, warp-uniform branch
            const double lu = lds_f64(exbase + SectorOff::lg), lf = lds_f64(exbase + SectorOff::lg + 8u);
#pragma unroll
            for (int q = 0; q < G; ++q) sts_f64(park + 8u * NT * q, F[q]);
            sector_log_factors<NT>(park, G, lu, lf, lp);
#pragma unroll
            for (int q = 0; q < G; ++q) num[q] *= lds_f64(park + 8u * NT * q);
        }
#pragma unroll
        for (int q = 0; q < G; ++q) acc[q][0] = __fma_rn(num[q], rcp_nr(den[q]), acc[q][0]);
    }
};

template <int DP, int G, int NT> __device__ __forceinline__ void spec_kernel_body(const FusedLaunch& L) {
    const DevAux* __restrict__ aux = L.aux;
    double* __restrict__ partials = L.partials;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SectorShared<DP, G, NT>& sh = *reinterpret_cast<SectorShared<DP, G, NT>*>(smem_raw);
    SmemCtx<DP, G, NT>& sm = sh.sm;
    SectorSmem<NT>& ex = sh.ex;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(&sm), exbase = (unsigned)__cvta_generic_to_shared(&ex);
    int cur = -1, iter = 0;
    long long tile_local = 0;
    bool changed;
    while (next_tile<DP, G, true, NT>(sm, L, cur, iter, tile_local, changed)) {
        if (changed) {
            if (threadIdx.x == 32) {
                const DevAux& a = aux[cur];
                ex.lg[0] = a.sec_log[0]; ex.lg[1] = a.sec_log[1]; ex.logp = a.sec_logp; ex.sel = sm.prob.spec_case;
            }
            __syncthreads();
        }
        run_tile<SectorEvalSpec<DP, G, NT>, DP, G, false, NT>(sm, sbase, exbase, tile_local, changed, partials);
    }
}

}  // namespace qmc

// one entry point per dimension-slot count; the names are looked up in the assembled module
extern "C" __global__ void __launch_bounds__(384, 1) qmc_spec_dp4(const __grid_constant__ qmc::FusedLaunch L) { qmc::spec_kernel_body<4, 8, 384>(L); }
extern "C" __global__ void __launch_bounds__(384, 1) qmc_spec_dp6(const __grid_constant__ qmc::FusedLaunch L) { qmc::spec_kernel_body<6, 8, 384>(L); }
extern "C" __global__ void __launch_bounds__(256, 1) qmc_spec_dp8(const __grid_constant__ qmc::FusedLaunch L) { qmc::spec_kernel_body<8, 8, 256>(L); }
extern "C" __global__ void __launch_bounds__(256, 1) qmc_spec_dp16(const __grid_constant__ qmc::FusedLaunch L) { qmc::spec_kernel_body<16, 4, 256>(L); }
