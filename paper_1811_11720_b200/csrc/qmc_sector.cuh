// qmc_sector.cuh -- the sector-like integrand family (BASELINE.json configs[3]; shape of the
// sector-decomposed integrands of P:L75):  f = prod_j x_j^nu_j * U(x)^a / F(x)^b with sparse
// positive-coefficient polynomials U, F.
//
// A C ABI cannot carry compiled functors (the paper compiles every sector with nvcc),
// so the parameter block is compiled ON THE DEVICE (prepare_sector) into a tiny straight-line
// program that the fused kernel interprets with warp-uniform control flow.  One program step is
// one fp64 instruction per point:
//     step = one byte: 4 + 4*(variable j) + 2*FIRST + LAST     (0 = no-op, 1 = end of U, 2 = end of program)
//     FIRST & LAST : sum  = fma(coef, x_j, sum)        (degree-1 monomial; coef = next coefficient)
//     FIRST        : mon  = coef * x_j
//     LAST         : sum  = fma(mon, x_j, sum)
//     otherwise    : mon *= x_j
// so a polynomial costs sum_t deg(t) fp64 instructions per point, with no separate additions.
// Steps are dispatched by one indexed branch each (PTX brx.idx, threaded code: every case fetches
// the next step and the next coefficient before its own fp64 work); the decode cost of a step is
// shared by the G points a thread evaluates together, which is why this family runs G = 8 shifts
// per lattice index where the registers allow it.  U and F are one instruction stream (the
// end-of-U step parks the sum and restarts it with F's constant).
#pragma once
#include "qmc_fused.cuh"

namespace qmc {

constexpr int kSecMaxCoef = 192;     // coefficient stream of a program: non-constant monomials of U and F + two dense linear forms
constexpr int kSecMaxWords = kMaxSectorOps / 4;

// step codes (one byte each): 0 = no-op, 1 = end of U, 2 = end of program, 3 = dense linear form (sum += sum_j c_j x_j over
// all DP slots, DP coefficients from the stream: the degree-1 monomials of a polynomial in ONE step), 4 + 4*j + 2*FIRST + LAST
enum : int { SEC_NOP = 0, SEC_ENDU = 1, SEC_END = 2, SEC_LIN = 3, SEC_BASE = 4 };

struct alignas(16) SectorSmem {
    double coefs[kSecMaxCoef];       // coefficients of the non-constant monomials, in step order
    unsigned int words[kSecMaxWords];// step bytes: U's steps, SEC_ENDU, F's steps, SEC_END (copied word-wise)
    double c0[2];                    // constant terms of U and F
    unsigned long long nu_packed;    // nu_j in 4 bits each
    int a, b;                        // powers of U and F
    double lg[2];                    // lu, lf of the log factor
    int logp, pad_;                  // its power p (0 = no log factor)
    double wpark[16 * kThreads];     // [q][thread]: the G weights of a thread, parked while the interpreter runs (registers);
                                     // with a log factor afterwards U in [0, 8), F in [8, 16) for sector_log_factors
};
struct SectorOff {                   // byte offsets of the fields above (read with ld.shared in the inner loop)
    static constexpr unsigned coefs = 0, words = kSecMaxCoef * 8, c0 = words + kSecMaxWords * 4, nu = c0 + 16, ab = nu + 8, lg = ab + 8, logp = lg + 16, wpark = logp + 8;
};

static_assert(offsetof(SectorSmem, words) == SectorOff::words && offsetof(SectorSmem, c0) == SectorOff::c0 &&
              offsetof(SectorSmem, nu_packed) == SectorOff::nu && offsetof(SectorSmem, a) == SectorOff::ab &&
              offsetof(SectorSmem, lg) == SectorOff::lg && offsetof(SectorSmem, logp) == SectorOff::logp &&
              offsetof(SectorSmem, wpark) == SectorOff::wpark, "SectorOff must mirror SectorSmem");

// ---- device-side compiler: params -> program (one thread; a few hundred steps at most) ---------
// program area of a problem (8-byte words at prog_area + aux_off): coefs[nU + nF] (upper bound),
// then the step bytes.  DevAux: sec_nops[0] = number of 32-bit step words, sec_ncoef[0] = number
// of coefficients.
__host__ __device__ inline int sector_dim_slots(int dim) { return dim <= 4 ? 4 : (dim <= 6 ? 6 : (dim <= 8 ? 8 : (dim <= 16 ? 16 : -1))); }

__device__ inline void prepare_sector(const DevProblem& pb, DevAux& a, unsigned long long* prog_area) {
    if (threadIdx.x != 0) return;
    const int d = pb.dim;
    const int dp = sector_dim_slots(d);
    const double* p = pb.params;
    int status = 0;
    // A rejected parameter block must still leave a program the interpreter can run to its end (the problem's
    // results are then replaced by NaN in the finalize stage): end-of-U, end, read-ahead padding.
    {
        const int slots = sector_coef_slots((pb.n_params - 4 - d) / (1 + d));
        unsigned char* stub = reinterpret_cast<unsigned char*>(prog_area + pb.aux_off + slots);
        stub[0] = (unsigned char)SEC_ENDU; stub[1] = (unsigned char)SEC_END;
        for (int i = 2; i < 8; ++i) stub[i] = (unsigned char)SEC_NOP;
        a.sec_nops[0] = 2; a.sec_nops[1] = 0; a.sec_ncoef[0] = 0; a.sec_ncoef[1] = 0;
        a.sec_c0[0] = a.sec_c0[1] = 1.0;
    }
    const double av = p[0], bv = p[1], nUv = p[2], nFv = p[3];
    if (!(av >= 0.0 && av <= 8.0 && bv >= 0.0 && bv <= 8.0 && nUv >= 1.0 && nUv <= kMaxSectorMono && nFv >= 1.0 &&
          nFv <= kMaxSectorMono) ||
        av != floor(av) || bv != floor(bv) || nUv != floor(nUv) || nFv != floor(nFv)) {
        a.status = QMC_ERR_PARAMS;
        return;
    }
    const int cnt[2] = {(int)nUv, (int)nFv};
    const int n_base = 4 + d + (cnt[0] + cnt[1]) * (1 + d);
    if (pb.n_params == n_base + 3) {                   // trailing [lu, lf, p]: f (lu log U + lf log F)^p, p in 1..4
        const double pw = p[n_base + 2];
        if (!(pw >= 1.0 && pw <= 4.0) || pw != floor(pw)) { a.status = QMC_ERR_PARAMS; return; }
        a.sec_log[0] = p[n_base]; a.sec_log[1] = p[n_base + 1]; a.sec_logp = (int)pw;
    } else if (pb.n_params != n_base) { a.status = QMC_ERR_PARAMS; return; }
    a.sec_a = (int)av; a.sec_b = (int)bv;
    for (int j = 0; j < d; ++j) {
        const double v = p[4 + j];
        if (!(v >= 0.0 && v <= 8.0) || v != floor(v)) status = QMC_ERR_PARAMS;
        a.nu[j] = (unsigned char)(int)v;
    }
    double* coefs = reinterpret_cast<double*>(prog_area + pb.aux_off);
    const int max_coef = sector_coef_slots((pb.n_params - 4 - d) / (1 + d));   // the same upper bound as the host plan and the kernel
    unsigned char* ops = reinterpret_cast<unsigned char*>(prog_area + pb.aux_off + max_coef);
    const int max_ops = min((pb.aux_len - max_coef) * 8, kMaxSectorOps) - 8;   // room for SEC_ENDU, SEC_END and 3+ bytes of read-ahead padding
    int nops = 0, ncoef = 0;
    const double* base = p + 4 + d;
    for (int pol = 0; pol < 2; ++pol) {
        const double* c = base;
        const double* e = base + cnt[pol];
        double c0 = 0.0;
        // the degree-1 monomials of the polynomial become one dense linear-form step when there are at least two
        int nlin = 0;
        for (int t = 0; t < cnt[pol]; ++t) {
            int deg = 0;
            for (int j = 0; j < d; ++j) deg += (int)e[t * d + j];
            nlin += (deg == 1);
        }
        const bool lin = nlin >= 2 && ncoef + dp < kSecMaxCoef - 1 && nops + 1 <= max_ops;
        if (lin) {
            for (int j = 0; j < dp; ++j) coefs[ncoef + j] = 0.0;
            for (int t = 0; t < cnt[pol]; ++t) {
                int deg = 0, var = 0;
                for (int j = 0; j < d; ++j) { const int ej = (int)e[t * d + j]; deg += ej; if (ej) var = j; }
                if (deg == 1) coefs[ncoef + var] += c[t];
            }
            ncoef += dp;
            ops[nops++] = (unsigned char)SEC_LIN;
        }
        for (int t = 0; t < cnt[pol]; ++t) {
            int deg = 0;
            for (int j = 0; j < d; ++j) {
                const double v = e[t * d + j];
                if (!(v >= 0.0 && v <= 8.0) || v != floor(v)) { status = QMC_ERR_PARAMS; continue; }
                deg += (int)v;
            }
            if (deg > 16 || status) { status = QMC_ERR_PARAMS; continue; }
            if (deg == 0) { c0 += c[t]; continue; }
            if (deg == 1 && lin) continue;
            if (ncoef >= kSecMaxCoef - 1 || nops + deg > max_ops) { status = QMC_ERR_PARAMS; continue; }
            coefs[ncoef++] = c[t];
            int seen = 0;
            for (int j = 0; j < d; ++j) {
                const int ej = (int)e[t * d + j];
                for (int r = 0; r < ej; ++r) {
                    const int first = (seen == 0), last = (seen == deg - 1);
                    ops[nops++] = (unsigned char)(SEC_BASE + j * 4 + first * 2 + last);
                    ++seen;
                }
            }
        }
        a.sec_c0[pol] = c0;
        if (!status) ops[nops++] = (unsigned char)(pol == 0 ? SEC_ENDU : SEC_END);
        base += cnt[pol] * (1 + d);
    }
    if (!status) while (nops & 3) ops[nops++] = (unsigned char)SEC_NOP;
    if (!status) {
        a.sec_nops[0] = nops / 4;
        a.sec_ncoef[0] = ncoef;
    } else {                                           // restore the stub (the loop above may have overwritten it)
        ops[0] = (unsigned char)SEC_ENDU; ops[1] = (unsigned char)SEC_END;
        for (int i = 2; i < 8; ++i) ops[i] = (unsigned char)SEC_NOP;
        a.sec_c0[0] = a.sec_c0[1] = 1.0;
    }
    a.status = status;
}

// ---- interpreter: U and F for G points (threaded code in inline PTX, see gen_sector_interp.py) ------
#include "qmc_sector_interp.inc"

// S2-S4 for the G points of one lattice index: x[q][j] and the weight W[q] (Eq. 12, Eq. 18)
template <int DP, int G, bool WIDE, int TR, int FIT>
__device__ __forceinline__ void sector_coords(const typename Res<WIDE>::T (&r)[DP], const EvalCtx& cx, double (&x)[G][DP],
                                              double (&W)[G]) {
    double P[G], D[G];
#pragma unroll
    for (int q = 0; q < G; ++q) { P[q] = 1.0; D[q] = 1.0; }
#pragma unroll
    for (int j = 0; j < DP; ++j) {
        const double rd = Res<WIDE>::to_double(r[j]);
        double fa, fb, dl[G];
        FitC fc;
        load_slot<DP, G, FIT>(cx.sbase, cx.delta, j, cx.fit_mode, fa, fb, fc, dl);
#pragma unroll
        for (int q = 0; q < G; ++q)
            x[q][j] = point_coord<TR, FIT>(rd, cx.inv_n, dl[q], fc, cx.sbase + SmemOff<DP, G>::kor, cx.kor_r, P[q], D[q]);
    }
#pragma unroll
    for (int q = 0; q < G; ++q) W[q] = point_weight<TR, FIT>(P[q], D[q], cx.wconst, cx.kor_r);
}

// (lu log U + lf log F)^p, p in 1..4 (the eps-expansion of U^(a + lu eps) / F^(b - lf eps)).
// The kernels are tuned for the plain sector integrand and only pay a never-taken warp-uniform branch for this (C-15).
// log x for the log factor.  Normal positive x (every sane U, F): x = 2^e m with m in (sqrt(1/2), sqrt(2)], log m = 2 atanh(s),
// s = (m - 1)/(m + 1), |s| <= 0.1716, by the Taylor series 2s (1 + z/3 + z^2/5 + ... + z^11/23), z = s^2 (truncation 6e-19
// relative), the quotient corrected to 1 ulp, e log 2 added as a two-term sum; measured <= 2 ulp against long double on
// 2e7 arguments in [e^-20, e^20] and relatively accurate towards x = 1.  Anything else (x <= 0, subnormal, inf, NaN) takes
// the library routine (sector_log_factors).
// Series coefficients 1/23 .. 1/3, sqrt 2 and the two halves of log 2 come from the constant bank as direct DFMA operands (as
// immediates every one of them cost two uniform moves per use).
static __constant__ double kLogC[14] = {1.0 / 23.0, 1.0 / 21.0, 1.0 / 19.0, 1.0 / 17.0, 1.0 / 15.0, 1.0 / 13.0, 1.0 / 11.0, 1.0 / 9.0,
                                        1.0 / 7.0, 1.0 / 5.0, 1.0 / 3.0, 1.4142135623730951, 0.6931471805599453, 2.3190468138462996e-17};
// The series itself is branch-free (its result is meaningless unless log_arg_is_normal_positive(x)), so that the chains of
// several logarithms share a basic block and overlap: with 3 warps per scheduler the path is bound by FP64 latency.
static __device__ __forceinline__ bool log_arg_is_normal_positive(double x) {
    const int hi = __double2hiint(x);
    return hi >= 0x00100000 && hi < 0x7ff00000;
}
static __device__ __forceinline__ double log_normal_positive(double x) {
    const int hi = __double2hiint(x);
    int e = (hi >> 20) - 1023;
    double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(x));
    const bool big = m > kLogC[11];
    m = big ? __dmul_rn(m, 0.5) : m;
    e += big;
    const double f = __dadd_rn(m, -1.0), den = __dadd_rn(m, 1.0);
    const double r = rcp_nr(den);
    double sq = __dmul_rn(f, r);
    sq = __fma_rn(__fma_rn(-sq, den, f), r, sq);
    const double z = __dmul_rn(sq, sq);
    double p = kLogC[0];
#pragma unroll
    for (int i = 1; i <= 10; ++i) p = __fma_rn(p, z, kLogC[i]);
    const double t = __dadd_rn(sq, sq);
    const double lm = __fma_rn(__dmul_rn(t, z), p, t);
    const double ed = (double)e;
    return __fma_rn(ed, kLogC[12], __fma_rn(ed, kLogC[13], lm));   // log 2 = hi + lo
}

// Once per lattice index: the caller parks U[q] at park + 8 kThreads q and F[q] at park + 8 kThreads (8 + q) (its own
// column of SectorSmem::wpark) and reads the factors back from the U slots.
static __device__ __forceinline__ void sector_log_factors(unsigned park, int g, double lu, double lf, int p) {
#pragma unroll 1
    for (int q = 0; q < g; q += 2) {                     // g is 4 or 8: two points = four independent logarithms per pass
        const unsigned at = park + 8u * kThreads * q;
        const double U0 = lds_f64(at), F0 = lds_f64(at + 64u * kThreads);
        const double U1 = lds_f64(at + 8u * kThreads), F1 = lds_f64(at + 72u * kThreads);
        double a0 = log_normal_positive(U0), b0 = log_normal_positive(F0), a1 = log_normal_positive(U1), b1 = log_normal_positive(F1);
        if (!(log_arg_is_normal_positive(U0) && log_arg_is_normal_positive(F0) && log_arg_is_normal_positive(U1) &&
              log_arg_is_normal_positive(F1))) {
            a0 = log(U0); b0 = log(F0); a1 = log(U1); b1 = log(F1);
        }
        const double L0 = __dadd_rn(__dmul_rn(lu, a0), __dmul_rn(lf, b0)), L1 = __dadd_rn(__dmul_rn(lu, a1), __dmul_rn(lf, b1));
        double r0 = L0, r1 = L1;
        for (int e = 1; e < p; ++e) { r0 = __dmul_rn(r0, L0); r1 = __dmul_rn(r1, L1); }
        sts_f64(at, r0);
        sts_f64(at + 8u * kThreads, r1);
    }
}

// Transform and fit map are selected per point by a warp-uniform switch, so that the interpreter exists once per
// tile loop.  SLOW = false: Korobov-3 without fit map, the paper's default for loop integrals, as the only
// inlined tile loop of the kernel (a smaller kernel body measurably helps the interpreter: DESIGN.md section 5); SLOW = true:
// the generic coordinate block (any transform, any fit mode at run time), reached through a real call (run_tile_call).
template <int DP, int G, bool WIDE, bool SLOW> struct SectorEval {
    static constexpr int NC = 1;
    typedef unsigned Extra;                                  // shared address of the CTA's SectorSmem
    static __device__ __forceinline__ void eval(const typename Res<WIDE>::T (&r)[DP], const SmemCtx<DP, G>&, const unsigned& exbase,
                                                const EvalCtx& cx, double (&acc)[G][1]) {
        double x[G][DP], num[G];
        if (!SLOW) {
            sector_coords<DP, G, WIDE, TR_KOR3, 0>(r, cx, x, num);
        } else {
            sector_coords<DP, G, WIDE, TR_KORR, FIT_RT>(r, cx, x, num);
        }
        // the weights are not needed until the interpreter is done: park them in shared memory ([q][thread], conflict free)
        const unsigned park = exbase + SectorOff::wpark + 8u * threadIdx.x;
#pragma unroll
        for (int q = 0; q < G; ++q) sts_f64(park + 8u * kThreads * q, num[q]);
        double c0u, c0f;
        lds_f64x2(exbase + SectorOff::c0, c0u, c0f);
        double U[G], F[G];
#pragma unroll
        for (int q = 0; q < G; ++q) { U[q] = 0.0; F[q] = c0u; }
        sector_interp<DP, G>(x, exbase + SectorOff::words, exbase + SectorOff::coefs, c0f, U, F);
#pragma unroll
        for (int q = 0; q < G; ++q) num[q] = lds_f64(park + 8u * kThreads * q);
        // num = W prod_j x_j^nu_j U^a, den = F^b   (small integer powers by repeated multiplication)
        const unsigned long long nup = lds_u64(exbase + SectorOff::nu);
        const unsigned long long ab = lds_u64(exbase + SectorOff::ab);
        const int pa = (int)(unsigned)ab, pb = (int)(ab >> 32);
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            const int nu = (int)((nup >> (4 * j)) & 15ull);
#pragma unroll 1
            for (int e = 0; e < nu; ++e)
#pragma unroll
                for (int q = 0; q < G; ++q) num[q] *= x[q][j];
        }
        // optional log factor (lu log U + lf log F)^p of an eps-expansion term: a cold, warp-uniform branch
        const int lp = (int)(unsigned)lds_u64(exbase + SectorOff::logp);
        if (lp) {
            const double lu = lds_f64(exbase + SectorOff::lg), lf = lds_f64(exbase + SectorOff::lg + 8u);
#pragma unroll
            for (int q = 0; q < G; ++q) { sts_f64(park + 8u * kThreads * q, U[q]); sts_f64(park + 8u * kThreads * (8 + q), F[q]); }
            sector_log_factors(park, G, lu, lf, lp);
#pragma unroll
            for (int q = 0; q < G; ++q) num[q] *= lds_f64(park + 8u * kThreads * q);
        }
        double den[G];
#pragma unroll
        for (int q = 0; q < G; ++q) den[q] = 1.0;
#pragma unroll 1
        for (int e = 0; e < pa; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) num[q] *= U[q];
#pragma unroll 1
        for (int e = 0; e < pb; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) den[q] *= F[q];
#pragma unroll
        for (int q = 0; q < G; ++q) acc[q][0] = __fma_rn(num[q], rcp_nr(den[q]), acc[q][0]);
    }
};

// shifts per group and resident CTAs per SM by dimension-slot count (x[G][DP] lives in registers)
template <int DP> struct SectorGroup { static constexpr int value = sector_group(DP); };
template <int DP, int G> struct SectorMinBlocks { static constexpr int value = min_blocks_sector(DP); };

template <int DP, int G, bool WIDE>
__global__ void __launch_bounds__(kThreads, SectorMinBlocks<DP, G>::value) fused_sector_kernel(const __grid_constant__ FusedLaunch L) {
    const DevAux* __restrict__ aux = L.aux;
    const unsigned long long* __restrict__ prog_area = L.prog;
    double* __restrict__ partials = L.partials;
    __shared__ SmemCtx<DP, G> sm;
    __shared__ SectorSmem ex;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(&sm), exbase = (unsigned)__cvta_generic_to_shared(&ex);
    int cur = -1, iter = 0;
    long long tile_local = 0;
    bool changed;
    while (next_tile<DP, G, true>(sm, L, cur, iter, tile_local, changed)) {
        if (changed) {
            const int tid = threadIdx.x;
            const DevAux& a = aux[cur];
            const DevProblem& pb = sm.prob;
            const int ncoef = a.sec_ncoef[0], nwords = a.sec_nops[0];
            const int max_coef = sector_coef_slots((pb.n_params - 4 - pb.dim) / (1 + pb.dim));
            const double* coefs = reinterpret_cast<const double*>(prog_area + pb.aux_off);
            const unsigned int* words = reinterpret_cast<const unsigned int*>(prog_area + pb.aux_off + max_coef);
            for (int i = tid; i <= ncoef && i < kSecMaxCoef; i += kThreads) ex.coefs[i] = i < ncoef ? coefs[i] : 0.0;
            for (int i = tid; i < nwords; i += kThreads) ex.words[i] = words[i];
            if (tid == 32) {
                ex.c0[0] = a.sec_c0[0]; ex.c0[1] = a.sec_c0[1];
                ex.a = a.sec_a; ex.b = a.sec_b;
                ex.lg[0] = a.sec_log[0]; ex.lg[1] = a.sec_log[1]; ex.logp = a.sec_logp; ex.pad_ = 0;
                unsigned long long nup = 0;
                for (int j = 0; j < 16; ++j) nup |= (unsigned long long)(a.nu[j] & 15) << (4 * j);
                ex.nu_packed = nup;
            }
            __syncthreads();
        }
        const bool fast = !sm.prob.has_fit && sm.prob.tr_kind == TR_KOR3;
        if (fast) run_tile<SectorEval<DP, G, WIDE, false>, DP, G, WIDE>(sm, sbase, exbase, tile_local, changed, partials);
        else run_tile_call<SectorEval<DP, G, WIDE, true>, DP, G, WIDE>(sm, sbase, exbase, tile_local, changed, partials);
    }
}

}  // namespace qmc
