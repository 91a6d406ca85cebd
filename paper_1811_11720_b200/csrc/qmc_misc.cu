// qmc_misc.cu -- the small kernels around the fused kernel: per-problem preparation, the finalize
// stage (S8), the inspection kernel (residues / coordinates) and the FP64 peak probe.
#include <cmath>

#include "qmc_sector.cuh"
#include "qmc_kernels.h"

namespace qmc {

// ---------------------------------------------------------------------------------------------
// prepare: derive the per-problem tables the fused kernel reads (one warp per problem)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) prepare_kernel(const DevProblem* __restrict__ probs, DevAux* __restrict__ aux,
                                                     unsigned long long* __restrict__ prog_area) {
    const DevProblem pb = probs[blockIdx.x];
    if (!is_sector_family(pb.family)) return;               // closed-form families derive their tables inside the fused kernel
    DevAux& a = aux[blockIdx.x];
    const int j = threadIdx.x;
    if (j < QMC_MAX_DIM) {
        const SlotConst s = derive_slot(pb, j, pb.family == QMC_FAMILY_SECTOR ? sector_threads(sector_dim_slots(pb.dim)) : kCSectorThreads);
        a.z[j] = s.z; a.step[j] = s.step; a.back[j] = s.back; a.fam_a[j] = s.fa; a.fam_b[j] = s.fb;
#pragma unroll
        for (int i = 0; i < 9; ++i) a.fit[i][j] = s.f[i];
        a.nu[j] = 0;
    }
    if (j == 0) {
        a.fam0 = derive_fam0(pb);
        a.fit_full = fit_has_poles(pb);
        a.status = 0;
        a.sec_a = a.sec_b = 0;
        a.sec_logp = 0; a.sec_log[0] = a.sec_log[1] = 0.0;
        a.sec_nops[0] = a.sec_nops[1] = a.sec_ncoef[0] = a.sec_ncoef[1] = 0;
        a.sec_c0[0] = a.sec_c0[1] = 0.0; a.sec_c0i[0] = a.sec_c0i[1] = 0.0;
    }
    {
        __syncwarp();
        prepare_sector(pb, a, prog_area);
    }
}

// ---------------------------------------------------------------------------------------------
// S8 finalize: Q_s = (sum over tiles in tile order)/n, Qbar, err (Eq. 2-3); one CTA
// per problem.  Compensated sums; per component for complex results.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void eq3_component(const double* __restrict__ means, int m, int nc, int c, double* mean_out,
                                              double* err_out) {
    CompSum t;
    for (int s = 0; s < m; ++s) t.add(means[s * nc + c]);
    const double mean = __ddiv_rn(t.value(), (double)m);
    CompSum v;
    for (int s = 0; s < m; ++s) { const double dlt = __dadd_rn(means[s * nc + c], -mean); v.add(__dmul_rn(dlt, dlt)); }
    *mean_out = mean;
    *err_out = __dsqrt_rn(__ddiv_rn(v.value(), __dmul_rn((double)m, (double)(m - 1))));
}

constexpr int kFinalizeThreads = 1024;
__global__ void __launch_bounds__(kFinalizeThreads) finalize_kernel(const __grid_constant__ FusedLaunch L, double* __restrict__ means_ws,
                                                                    double* __restrict__ out_means, double* __restrict__ out_errs,
                                                                    double* __restrict__ out_shift_means, int stride) {
    const DevProblem& pb = L.single ? L.one : L.probs[blockIdx.x];
    const double* __restrict__ partials = L.partials;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nc = pb.ncomp, m = pb.m, tiles = pb.tiles, npairs = m * nc;
    double* means = means_ws + pb.means_off;
    const bool bad = is_sector_family(pb.family) && L.aux[blockIdx.x].status != 0;
    for (int pair = warp; pair < npairs; pair += kFinalizeThreads / 32) {
        const double* src = partials + pb.partial_off + (long long)pair * tiles;
        CompSum cs;
        for (int t = lane; t < tiles; t += 32) cs.add(src[t]);
        const double v = warp_sum(cs.value());
        if (lane == 0) {
            double q = __ddiv_rn(v, (double)pb.n);
            if (bad) q = nan("");
            means[pair] = q;
            if (out_shift_means) out_shift_means[(size_t)pb.out_index * stride + pair] = q;
        }
    }
    __syncthreads();
    if (tid < 2) {
        double mean = 0.0, err = 0.0;
        if (tid < nc) eq3_component(means, m, nc, tid, &mean, &err);
        out_means[(size_t)pb.out_index * 2 + tid] = mean;
        out_errs[(size_t)pb.out_index * 2 + tid] = err;
    }
}

__global__ void __launch_bounds__(32) finalize_means_kernel(const double* __restrict__ means, int m, int nc,
                                                            double* __restrict__ out_mean, double* __restrict__ out_err) {
    if (threadIdx.x < nc) eq3_component(means, m, nc, threadIdx.x, &out_mean[threadIdx.x], &out_err[threadIdx.x]);
}

// ---------------------------------------------------------------------------------------------
// inspection: residues and coordinates through the same device functions as the fused kernel
// (first residue by mulmod, then stepping by add_mod; conversion and wrap as in S1-S2)
// ---------------------------------------------------------------------------------------------
template <bool WIDE>
__global__ void __launch_bounds__(kThreads) points_kernel(PointsArgs a) {
    typedef typename Res<WIDE>::T RT;
    const unsigned long long stride = (unsigned long long)gridDim.x * kThreads;
    unsigned long long i = (unsigned long long)blockIdx.x * kThreads + threadIdx.x;
    if (i >= a.count) return;
    const unsigned long long n = a.n;
    RT r[QMC_MAX_DIM], step[QMC_MAX_DIM];
    const unsigned long long kfirst = (a.k0 % n + i % n) % n;
    for (int j = 0; j < a.dim; ++j) {
        const unsigned long long z = a.z[j] % n;
        r[j] = (RT)mulmod_u64(kfirst, z, n);
        step[j] = (RT)mulmod_u64(stride % n, z, n);
    }
    for (; i < a.count; i += stride) {
        for (int j = 0; j < a.dim; ++j) {
            if (a.out_r) a.out_r[i * a.dim + j] = (unsigned long long)r[j];
            if (a.out_u) a.out_u[i * a.dim + j] = wrap_u(coord_t(Res<WIDE>::to_double(r[j]), a.inv_n, a.shift[j]));
            r[j] = add_mod<RT>(r[j], step[j], (RT)n);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// FP64 peak probe: 8 independent DFMA chains per thread, 2048 threads per SM.  The multiplier and the addend are
// compile-time constants, so that each DFMA reads ONE 64-bit vector-register operand pair besides its accumulator (the
// constant multiplier comes from a uniform register): with three distinct vector-register operands per DFMA (round 1's
// probe took a and b as kernel arguments, which ptxas loaded into vector registers) the register file, not the FP64
// pipe, limits the rate -- 17.07 instead of 18.38 Tinst/s on the same B200 at 1965 MHz (nominal 148 x 64 x 1.965 = 18.61).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 8) dfma_probe_kernel(double* __restrict__ out, int iters) {
    const double a = 0.999999, b = 1e-6;
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 0.1, x2 = x0 + 0.2, x3 = x0 + 0.3, x4 = x0 + 0.4, x5 = x0 + 0.5, x6 = x0 + 0.6,
           x7 = x0 + 0.7;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = __fma_rn(x0, a, b); x1 = __fma_rn(x1, a, b); x2 = __fma_rn(x2, a, b); x3 = __fma_rn(x3, a, b);
            x4 = __fma_rn(x4, a, b); x5 = __fma_rn(x5, a, b); x6 = __fma_rn(x6, a, b); x7 = __fma_rn(x7, a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// ---------------------------------------------------------------------------------------------
// host-callable launchers
// ---------------------------------------------------------------------------------------------
cudaError_t launch_prepare(int count, cudaStream_t st, const DevProblem* probs, DevAux* aux, unsigned long long* prog_area) {
    prepare_kernel<<<count, 32, 0, st>>>(probs, aux, prog_area);
    return cudaGetLastError();
}
cudaError_t launch_finalize(int count, cudaStream_t st, const FusedLaunch& a, double* means_ws, double* out_means, double* out_errs,
                            double* out_shift_means, int stride) {
    finalize_kernel<<<count, kFinalizeThreads, 0, st>>>(a, means_ws, out_means, out_errs, out_shift_means, stride);
    return cudaGetLastError();
}
cudaError_t launch_finalize_means(cudaStream_t st, const double* means, int m, int nc, double* out_mean, double* out_err) {
    finalize_means_kernel<<<1, 32, 0, st>>>(means, m, nc, out_mean, out_err);
    return cudaGetLastError();
}
cudaError_t launch_points(cudaStream_t st, const PointsArgs& a, int sm_count) {
    if (a.count == 0) return cudaSuccess;
    unsigned long long blocks = (a.count + kThreads - 1) / kThreads;
    const unsigned long long cap = (unsigned long long)sm_count * 8;
    if (blocks > cap) blocks = cap;
    if (a.n >= (1ull << 31)) points_kernel<true><<<(unsigned)blocks, kThreads, 0, st>>>(a);
    else points_kernel<false><<<(unsigned)blocks, kThreads, 0, st>>>(a);
    return cudaGetLastError();
}
cudaError_t launch_dfma_probe(cudaStream_t st, double* out, int blocks, int iters) {
    dfma_probe_kernel<<<blocks, 256, 0, st>>>(out, iters);
    return cudaGetLastError();
}

}  // namespace qmc
