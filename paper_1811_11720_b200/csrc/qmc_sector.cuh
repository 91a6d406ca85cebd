// qmc_sector.cuh -- the sector-like integrand family (BASELINE.json configs[3]; shape of the
// sector-decomposed integrands of P:L75):  f = prod_j x_j^nu_j * U(x)^a / F(x)^b with sparse
// positive-coefficient polynomials U, F.
//
// A C ABI cannot carry compiled functors (the paper compiles every sector with nvcc),
// so the parameter block is compiled ON THE DEVICE (prepare_sector) into a tiny straight-line
// program that the fused kernel interprets with warp-uniform control flow.  One program step is
// one fp64 instruction per point:
//     step = (variable j, FIRST, LAST, coefficient index)
//     FIRST & LAST : sum  = fma(coef, x_j, sum)        (degree-1 monomial)
//     FIRST        : mon  = coef * x_j
//     LAST         : sum  = fma(mon, x_j, sum)
//     otherwise    : mon *= x_j
// so a polynomial costs sum_t deg(t) fp64 instructions per point, with no separate additions.
// The decode cost of a step (load, extract, indexed branch) is shared by the G points a thread
// evaluates together.
#pragma once
#include "qmc_fused.cuh"

namespace qmc {

constexpr int kSecMaxCoef = 128;     // non-constant monomials of U and F together

struct SectorSmem {
    double coefs[kSecMaxCoef];
    unsigned short ops[kMaxSectorOps];
    double c0[2];
    int nops[2], ncoef[2];
    int a, b;
    int nu[QMC_MAX_DIM];
};

// ---- device-side compiler: params -> program (one thread; a few hundred steps at most) ---------
// program area of a problem (8-byte words at prog_area + aux_off): coefs[ncoefU + ncoefF], then
// the u16 ops of U followed by those of F.
__device__ inline void prepare_sector(const DevProblem& pb, DevAux& a, unsigned long long* prog_area) {
    if (threadIdx.x != 0) return;
    const int d = pb.dim;
    const double* p = pb.params;
    int status = 0;
    const double av = p[0], bv = p[1], nUv = p[2], nFv = p[3];
    if (!(av >= 0.0 && av <= 8.0 && bv >= 0.0 && bv <= 8.0 && nUv >= 1.0 && nUv <= kMaxSectorMono && nFv >= 1.0 &&
          nFv <= kMaxSectorMono) ||
        av != floor(av) || bv != floor(bv) || nUv != floor(nUv) || nFv != floor(nFv)) {
        a.status = QMC_ERR_PARAMS;
        return;
    }
    const int cnt[2] = {(int)nUv, (int)nFv};
    if (4 + d + (cnt[0] + cnt[1]) * (1 + d) != pb.n_params) { a.status = QMC_ERR_PARAMS; return; }
    a.sec_a = (int)av; a.sec_b = (int)bv;
    for (int j = 0; j < d; ++j) {
        const double v = p[4 + j];
        if (!(v >= 0.0 && v <= 8.0) || v != floor(v)) status = QMC_ERR_PARAMS;
        a.nu[j] = (unsigned char)(int)v;
    }
    double* coefs = reinterpret_cast<double*>(prog_area + pb.aux_off);
    const int max_coef = cnt[0] + cnt[1];
    unsigned short* ops = reinterpret_cast<unsigned short*>(prog_area + pb.aux_off + max_coef);
    const int max_ops = (pb.aux_len - max_coef) * 4;
    int nops_total = 0, ncoef_total = 0;
    const double* base = p + 4 + d;
    for (int pol = 0; pol < 2; ++pol) {
        const double* c = base;
        const double* e = base + cnt[pol];
        double c0 = 0.0;
        int nops = 0, ncoef = 0;
        for (int t = 0; t < cnt[pol]; ++t) {
            int deg = 0;
            for (int j = 0; j < d; ++j) {
                const double v = e[t * d + j];
                if (!(v >= 0.0 && v <= 8.0) || v != floor(v)) { status = QMC_ERR_PARAMS; continue; }
                deg += (int)v;
            }
            if (deg > 16 || status) { status = QMC_ERR_PARAMS; continue; }
            if (deg == 0) { c0 += c[t]; continue; }
            if (ncoef_total + ncoef >= kSecMaxCoef || nops_total + nops + deg > kMaxSectorOps ||
                nops_total + nops + deg > max_ops) { status = QMC_ERR_PARAMS; continue; }
            coefs[ncoef_total + ncoef] = c[t];
            int seen = 0;
            for (int j = 0; j < d; ++j) {
                const int ej = (int)e[t * d + j];
                for (int r = 0; r < ej; ++r) {
                    const int first = (seen == 0), last = (seen == deg - 1);
                    ops[nops_total + nops] = (unsigned short)((j * 4 + first * 2 + last) | (ncoef << 8));
                    ++nops; ++seen;
                }
            }
            ++ncoef;
        }
        a.sec_c0[pol] = c0;
        a.sec_nops[pol] = nops;
        a.sec_ncoef[pol] = ncoef;
        nops_total += nops;
        ncoef_total += ncoef;
        base += cnt[pol] * (1 + d);
    }
    a.status = status;
}

// ---- interpreter: one polynomial for G points --------------------------------------------------
#define QMC_SEC_CASE(J)                                                                                         \
    case 4 * (J) + 0:                                                                                           \
        _Pragma("unroll") for (int q = 0; q < G; ++q) mon[q] *= x[q][(J) < DP ? (J) : 0];                       \
        break;                                                                                                  \
    case 4 * (J) + 1:                                                                                           \
        _Pragma("unroll") for (int q = 0; q < G; ++q) sum[q] = __fma_rn(mon[q], x[q][(J) < DP ? (J) : 0], sum[q]); \
        break;                                                                                                  \
    case 4 * (J) + 2:                                                                                           \
        _Pragma("unroll") for (int q = 0; q < G; ++q) mon[q] = cf * x[q][(J) < DP ? (J) : 0];                   \
        break;                                                                                                  \
    case 4 * (J) + 3:                                                                                           \
        _Pragma("unroll") for (int q = 0; q < G; ++q) sum[q] = __fma_rn(cf, x[q][(J) < DP ? (J) : 0], sum[q]);  \
        break;

template <int DP, int G>
__device__ __forceinline__ void sector_poly(const double (&x)[G][DP], const unsigned short* __restrict__ ops, int nops,
                                            const double* __restrict__ coefs, double c0, double (&sum)[G]) {
    double mon[G];
#pragma unroll
    for (int q = 0; q < G; ++q) { sum[q] = c0; mon[q] = 0.0; }
#pragma unroll 1
    for (int i = 0; i < nops; ++i) {
        const unsigned op = ops[i];
        const double cf = coefs[op >> 8];
        switch (op & 0xffu) {
            QMC_SEC_CASE(0) QMC_SEC_CASE(1) QMC_SEC_CASE(2) QMC_SEC_CASE(3)
            QMC_SEC_CASE(4) QMC_SEC_CASE(5) QMC_SEC_CASE(6) QMC_SEC_CASE(7)
            QMC_SEC_CASE(8) QMC_SEC_CASE(9) QMC_SEC_CASE(10) QMC_SEC_CASE(11)
            QMC_SEC_CASE(12) QMC_SEC_CASE(13) QMC_SEC_CASE(14) QMC_SEC_CASE(15)
            default: break;
        }
    }
}
#undef QMC_SEC_CASE

template <int DP, int G, bool WIDE, int TR, bool FIT> struct SectorEval {
    static constexpr int NC = 1;
    typedef SectorSmem Extra;
    static __device__ __forceinline__ void eval(const typename Res<WIDE>::T (&r)[DP], const SmemCtx<DP, G>& sm,
                                                const SectorSmem& ex, int dim, double inv_n, double wconst, int kor_r,
                                                double (&acc)[G][1]) {
        double x[G][DP], P[G], D[G], pre[G];
#pragma unroll
        for (int q = 0; q < G; ++q) { P[q] = 1.0; D[q] = 1.0; pre[q] = 1.0; }
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            if (j < dim) {
                const double rd = Res<WIDE>::to_double(r[j]);
#pragma unroll
                for (int q = 0; q < G; ++q) x[q][j] = point_coord<DP, G, TR, FIT>(rd, inv_n, q, j, sm, kor_r, P[q], D[q]);
                const int nu = ex.nu[j];
#pragma unroll 1
                for (int e = 0; e < nu; ++e)
#pragma unroll
                    for (int q = 0; q < G; ++q) pre[q] *= x[q][j];
            } else {
#pragma unroll
                for (int q = 0; q < G; ++q) x[q][j] = 1.0;
            }
        }
        double U[G], F[G];
        sector_poly<DP, G>(x, ex.ops, ex.nops[0], ex.coefs, ex.c0[0], U);
        sector_poly<DP, G>(x, ex.ops + ex.nops[0], ex.nops[1], ex.coefs + ex.ncoef[0], ex.c0[1], F);
        double num[G], den[G];
#pragma unroll
        for (int q = 0; q < G; ++q) { num[q] = pre[q]; den[q] = 1.0; }
#pragma unroll 1
        for (int e = 0; e < ex.a; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) num[q] *= U[q];
#pragma unroll 1
        for (int e = 0; e < ex.b; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) den[q] *= F[q];
        constexpr bool USEW = (TR == TR_KOR3 || TR == TR_KORR || FIT);
#pragma unroll
        for (int q = 0; q < G; ++q) {
            const double w = USEW ? point_weight<TR, FIT>(P[q], D[q], wconst, kor_r) * num[q] : num[q];
            acc[q][0] += w / den[q];
        }
    }
};

template <int DP, int G, bool WIDE>
__global__ void __launch_bounds__(kThreads, 3) fused_sector_kernel(const DevProblem* __restrict__ probs,
                                                                   const DevAux* __restrict__ aux, VariantQueue vq,
                                                                   double* __restrict__ partials,
                                                                   const unsigned long long* __restrict__ prog_area) {
    __shared__ SmemCtx<DP, G> sm;
    __shared__ SectorSmem ex;
    int cur = -1;
    long long tile_local = 0;
    bool changed;
    while (next_tile<DP, G>(sm, probs, aux, vq, cur, tile_local, changed)) {
        if (changed) {
            const int tid = threadIdx.x;
            const DevAux& a = aux[cur];
            const DevProblem& pb = sm.prob;
            const int ncoef = a.sec_ncoef[0] + a.sec_ncoef[1], nops = a.sec_nops[0] + a.sec_nops[1];
            const int max_coef = (pb.n_params - 4 - pb.dim) / (1 + pb.dim);
            const double* coefs = reinterpret_cast<const double*>(prog_area + pb.aux_off);
            const unsigned short* ops = reinterpret_cast<const unsigned short*>(prog_area + pb.aux_off + max_coef);
            for (int i = tid; i < ncoef; i += kThreads) ex.coefs[i] = coefs[i];
            for (int i = tid; i < nops; i += kThreads) ex.ops[i] = ops[i];
            if (tid < QMC_MAX_DIM) ex.nu[tid] = a.nu[tid];
            if (tid == 32) {
                ex.c0[0] = a.sec_c0[0]; ex.c0[1] = a.sec_c0[1];
                ex.nops[0] = a.sec_nops[0]; ex.nops[1] = a.sec_nops[1];
                ex.ncoef[0] = a.sec_ncoef[0]; ex.ncoef[1] = a.sec_ncoef[1];
                ex.a = a.sec_a; ex.b = a.sec_b;
            }
            __syncthreads();
        }
        const int sel = sm.prob.tr_kind * 2 + (sm.prob.has_fit ? 1 : 0);
        switch (sel) {
#define QMC_CASE(TRK, FITB) \
    case TRK * 2 + (FITB ? 1 : 0): run_tile<SectorEval<DP, G, WIDE, TRK, FITB>, DP, G, WIDE>(sm, ex, tile_local, partials); break;
            QMC_CASE(TR_NONE, false) QMC_CASE(TR_NONE, true) QMC_CASE(TR_BAKER, false) QMC_CASE(TR_BAKER, true)
            QMC_CASE(TR_KOR3, false) QMC_CASE(TR_KOR3, true) QMC_CASE(TR_KORR, false) QMC_CASE(TR_KORR, true)
#undef QMC_CASE
            default: break;
        }
    }
}

}  // namespace qmc
