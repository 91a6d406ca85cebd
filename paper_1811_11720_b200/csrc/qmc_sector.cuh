// qmc_sector.cuh -- the sector-like integrand family (BASELINE.json configs[3]; shape of the
// sector-decomposed integrands of P:L75):  f = prod_j x_j^nu_j * U(x)^a / F(x)^b with sparse
// positive-coefficient polynomials U, F.
//
// A C ABI cannot carry compiled functors (the paper compiles every sector with nvcc),
// so the parameter block is compiled ON THE DEVICE (prepare_sector) into a tiny straight-line
// program that the fused kernel interprets with warp-uniform control flow.  The target machine has
// two accumulators per point, S (the polynomial) and A (the current group), and five step kinds of
// one fp64 instruction per point each (gen_sector_interp.py):
//     SC j : S = fma(A, x_j, S)        SL j : S = fma(cf, x_j, S)       AL j : A = fma(cf, x_j, A)
//     ALI j: A = fma(cf, x_j, cf2)     AM j : A = A * x_j
// A polynomial is compiled into a greedy multivariate Horner form: the variable that occurs in most
// monomials is factored out, recursively, which yields groups  x^P (own + sum_k c_k x_k)  sharing
// the prefix monomial x^P:
//     ALI k_0 (cf = c_k0, cf2 = own), AL k_i ..., AM p_1 ... AM p_(D-1), SC p_D        D = deg P
// (a monomial nobody shares a prefix with is ALI, AM ..., SC: deg steps; degree 1: SL).  On the 256 seeded
// sectors of configs[3] this is 30.6 steps per point for U and F together where the monomial-by-monomial
// evaluation of round 1 took 44.4 (48.0 with its dense linear forms).
// Steps are dispatched by one indexed branch each (PTX brx.idx, threaded code); the decode cost of
// a step is shared by the G points a thread evaluates together, and the CTA is as large as the SM
// holds (one CTA per SM) so that every warp of an SM runs the same program: the cases a program
// touches must stay in the 6 KB L0 instruction cache.
#pragma once
#include "qmc_fused.cuh"
#include "qmc_sector_compile.h"

#ifndef QMC_SECTOR_PAIR_DIMS
#define QMC_SECTOR_PAIR_DIMS 1
#endif

namespace qmc {

constexpr int kSecMaxSlots = sector_slot_words(2 * kMaxSectorMono) / 2;   // coefficient slots of a program: one per monomial + end-of-polynomial + read-ahead
constexpr int kSecMaxWords = kMaxSectorOps / 4;
constexpr int kSecParkRows = 16;                       // rows of G... doubles per thread parked in shared memory: weights [0, 8), U [8, 16)


template <int NT> struct alignas(16) SectorSmem {
    double slots[kSecMaxSlots * 4];  // {cf, cf2} per coefficient-consuming step, in program order (complex family: {cf_re, cf_im, cf2_re, cf2_im})
    unsigned int words[kSecMaxWords];// step bytes: U's steps, SEC_ENDP, F's steps, SEC_END (copied word-wise)
    double c0u, c0u_im;              // constant term of U (F's travels in the slot of the end-of-polynomial step)
    unsigned long long nu_packed;    // nu_j in 4 bits each
    int a, b;                        // powers of U and F
    double lg[2];                    // lu, lf of the log factor
    int logp, sel;                   // its power p (0 = no log factor); specialised kernels: the problem's case selector
    double park[kSecParkRows * NT];  // [row][thread]: rows [0, 8) the G weights of a thread while the interpreter runs (with a log
                                     // factor afterwards F), rows [8, 16) U as the interpreter parks it (complex: (re, im) pairs)
};
struct SectorOff {                   // byte offsets of the fields above (read with ld.shared in the inner loop)
    static constexpr unsigned slots = 0, words = kSecMaxSlots * 32, c0u = words + kSecMaxWords * 4, nu = c0u + 16, ab = nu + 8, lg = ab + 8,
                              logp = lg + 16, sel = logp + 4, park = logp + 8;
};
#define QMC_SECTOR_OFF_CHECK(NT)                                                                                                      \
    static_assert(offsetof(SectorSmem<NT>, words) == SectorOff::words && offsetof(SectorSmem<NT>, c0u) == SectorOff::c0u &&           \
                  offsetof(SectorSmem<NT>, nu_packed) == SectorOff::nu && offsetof(SectorSmem<NT>, a) == SectorOff::ab &&             \
                  offsetof(SectorSmem<NT>, lg) == SectorOff::lg && offsetof(SectorSmem<NT>, logp) == SectorOff::logp &&               \
                  offsetof(SectorSmem<NT>, park) == SectorOff::park, "SectorOff must mirror SectorSmem");
QMC_SECTOR_OFF_CHECK(256) QMC_SECTOR_OFF_CHECK(384)
#undef QMC_SECTOR_OFF_CHECK

__host__ __device__ inline int sector_dim_slots(int dim) { return dim <= 4 ? 4 : (dim <= 6 ? 6 : (dim <= 8 ? 8 : (dim <= 16 ? 16 : -1))); }

__device__ inline void prepare_sector(const DevProblem& pb, DevAux& a, unsigned long long* prog_area) {
    if (threadIdx.x != 0) return;
    const int d = pb.dim;
    const bool cplx = pb.family == QMC_FAMILY_SECTOR_COMPLEX;
    const int rec = sector_mono_stride(pb.family, d), sw = cplx ? 4 : 2;                 // monomial record, doubles per slot
    const double* p = pb.params;
    const int nmono_total = (pb.n_params - 4 - d) / rec;
    double* slots = reinterpret_cast<double*>(prog_area + pb.aux_off);
    unsigned char* ops = reinterpret_cast<unsigned char*>(prog_area + pb.aux_off + sector_slot_words(nmono_total, cplx));
    // A rejected parameter block must still leave a program the interpreter can run to its end (the problem's
    // results are then replaced by NaN in the finalize stage): end-of-U, end, read-ahead padding.
    auto stub = [&]() {
        ops[0] = (unsigned char)SEC_ENDP; ops[1] = (unsigned char)SEC_END;
        for (int i = 2; i < 8; ++i) ops[i] = (unsigned char)SEC_NOP;
        for (int i = 0; i < 2 * sw; ++i) slots[i] = (i == 0) ? 1.0 : 0.0;
        a.sec_nops[0] = 2; a.sec_nops[1] = 0; a.sec_ncoef[0] = 2; a.sec_ncoef[1] = 0;
        a.sec_c0[0] = a.sec_c0[1] = 1.0; a.sec_c0i[0] = a.sec_c0i[1] = 0.0;
    };
    stub();
    const int vst = sector_block_status(p, pb.n_params, d, cplx);
    if (vst != 0) { a.status = vst; return; }
    const int cnt[2] = {(int)p[2], (int)p[3]};
    const int n_base = 4 + d + (cnt[0] + cnt[1]) * rec;
    if (pb.n_params == n_base + 3) { a.sec_log[0] = p[n_base]; a.sec_log[1] = p[n_base + 1]; a.sec_logp = (int)p[n_base + 2]; }
    a.sec_a = (int)p[0]; a.sec_b = (int)p[1];
    for (int j = 0; j < d; ++j) a.nu[j] = (unsigned char)(int)p[4 + j];
    SecEmit out;
    out.slots = slots; out.ops = ops; out.nslots = 0; out.nops = 0; out.status = 0; out.cplx = cplx;
    out.max_slots = sector_slot_words(nmono_total, cplx) / sw - 1;                       // one slot of read-ahead
    out.max_ops = min((pb.aux_len - sector_slot_words(nmono_total, cplx)) * 8, kMaxSectorOps) - 8;   // room for the two end steps and the read-ahead padding
    const double* base = p + 4 + d;                    // polynomial: Re c (cnt) [, Im c (cnt)], exponents (cnt x d)
    double c0u, c0ui, c0f, c0fi;
    compile_polynomial(base, cplx ? base + cnt[0] : nullptr, base + (cplx ? 2 : 1) * cnt[0], cnt[0], d, out, &c0u, &c0ui);
    base += cnt[0] * rec;
    // end of U: its step takes F's constant term from the slot stream -- the slot is filled after F is compiled
    const int endp_slot = out.nslots;
    out.ops[out.nops++] = (unsigned char)SEC_ENDP;          // max_ops keeps room for the end steps
    out.slot(0.0, 0.0, 0.0, 0.0);
    compile_polynomial(base, cplx ? base + cnt[1] : nullptr, base + (cplx ? 2 : 1) * cnt[1], cnt[1], d, out, &c0f, &c0fi);
    if (out.status) { stub(); a.status = out.status; return; }
    slots[sw * endp_slot] = c0f;
    if (cplx) slots[sw * endp_slot + 1] = c0fi;
    out.ops[out.nops++] = (unsigned char)SEC_END;
    out.ops[out.nops++] = (unsigned char)SEC_NOP;       // the interpreter reads two step codes ahead
    out.ops[out.nops++] = (unsigned char)SEC_NOP;
    while (out.nops & 3) out.ops[out.nops++] = (unsigned char)SEC_NOP;
    for (int i = 0; i < sw; ++i) slots[sw * out.nslots + i] = 0.0;                         // read-ahead slot
    a.sec_c0[0] = c0u; a.sec_c0[1] = c0f; a.sec_c0i[0] = c0ui; a.sec_c0i[1] = c0fi;
    a.sec_nops[0] = out.nops / 4;
    a.sec_ncoef[0] = out.nslots + 1;
    a.status = 0;
}

// ---- interpreter: U and F for G points (threaded code in inline PTX, see gen_sector_interp.py) ------
#include "qmc_sector_interp.inc"
#include "qmc_csector_interp.inc"

// S2-S4 for the G points of one lattice index: x[q][j] and the weight W[q] (Eq. 12, Eq. 18)
template <int DP, int G, bool WIDE, int TR, int FIT>
__device__ __forceinline__ void sector_coords(const typename Res<WIDE>::T (&r)[DP], const EvalCtx& cx, double (&x)[G][DP],
                                              double (&W)[G]) {
    double P[G], D[G];
#pragma unroll
    for (int q = 0; q < G; ++q) { P[q] = 1.0; D[q] = 1.0; }
    // Korobov-3 without a fit map: two dimensions per stage (see eval_point_group, PAIRED)
    constexpr bool PAIRED = QMC_SECTOR_PAIR_DIMS && TR == TR_KOR3 && FIT == 0 && DP % 2 == 0;
    if constexpr (PAIRED) {
#pragma unroll
        for (int j = 0; j < DP; j += 2) {
            double fa, fb, dl[2][G], rd[2], c[2][G], sq[2][G], g[2][G];
            FitC fc;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                rd[h] = Res<WIDE>::to_double(r[j + h]);
                load_slot<DP, G, 0>(cx.sbase, cx.delta, j + h, 0, fa, fb, fc, dl[h]);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) c[h][q] = centre_c(coord_t(rd[h], cx.inv_n, dl[h][q]));
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) sq[h][q] = c[h][q] * c[h][q];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) g[h][q] = __fma_rn(-20.0, sq[h][q], 21.0);
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) g[h][q] = __fma_rn(g[h][q], sq[h][q], -8.75);
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) g[h][q] = __fma_rn(g[h][q], sq[h][q], 2.1875);
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) x[q][j + h] = __fma_rn(c[h][q], g[h][q], 0.5);
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) P[q] = __dmul_rn(P[q], __dadd_rn(0.25, -sq[h][q]));
        }
    }
#pragma unroll
    for (int j = 0; j < (PAIRED ? 0 : DP); ++j) {
        const double rd = Res<WIDE>::to_double(r[j]);
        double fa, fb, dl[G];
        FitC fc;
        load_slot<DP, G, FIT>(cx.sbase, cx.delta, j, cx.fit_mode, fa, fb, fc, dl);
        if constexpr (TR == TR_KORR) {                        // generic tile loop: kind and fit mode decided once per dimension
            double t[G], xg[G];
#pragma unroll
            for (int q = 0; q < G; ++q) t[q] = coord_t(rd, cx.inv_n, dl[q]);
            generic_coord_group<G>(t, cx.sbase + SmemOff<DP, G>::kor, cx.kor_r, fc, xg, P, D);
#pragma unroll
            for (int q = 0; q < G; ++q) x[q][j] = xg[q];
        } else {
#pragma unroll
            for (int q = 0; q < G; ++q)
                x[q][j] = point_coord<TR, FIT>(rd, cx.inv_n, dl[q], fc, cx.sbase + SmemOff<DP, G>::kor, cx.kor_r, P[q], D[q]);
        }
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

// Once per lattice index: F[q] sits in park row q and U[q] in row 8 + q (the thread's own column of SectorSmem::park);
// the factors are written over the F rows.
template <int NT>
static __device__ __forceinline__ void sector_log_factors(unsigned park, int g, double lu, double lf, int p) {
#pragma unroll 1
    for (int q = 0; q < g; q += 2) {                     // g is 4 or 8: two points = four independent logarithms per pass
        const unsigned at = park + 8u * NT * q;
        const double F0 = lds_f64(at), U0 = lds_f64(at + 64u * NT);
        const double F1 = lds_f64(at + 8u * NT), U1 = lds_f64(at + 72u * NT);
        double a0 = log_normal_positive(U0), b0 = log_normal_positive(F0), a1 = log_normal_positive(U1), b1 = log_normal_positive(F1);
        if (!(log_arg_is_normal_positive(U0) && log_arg_is_normal_positive(F0) && log_arg_is_normal_positive(U1) &&
              log_arg_is_normal_positive(F1))) {
            a0 = log(U0); b0 = log(F0); a1 = log(U1); b1 = log(F1);
        }
        const double L0 = __dadd_rn(__dmul_rn(lu, a0), __dmul_rn(lf, b0)), L1 = __dadd_rn(__dmul_rn(lu, a1), __dmul_rn(lf, b1));
        double r0 = L0, r1 = L1;
        for (int e = 1; e < p; ++e) { r0 = __dmul_rn(r0, L0); r1 = __dmul_rn(r1, L1); }
        sts_f64(at, r0);
        sts_f64(at + 8u * NT, r1);
    }
}

// Transform and fit map are selected per point by a warp-uniform switch, so that the interpreter exists once per
// tile loop.  SLOW = false: Korobov-3 without fit map, the paper's default for loop integrals, as the only
// inlined tile loop of the kernel (a smaller kernel body measurably helps the interpreter: DESIGN.md section 5); SLOW = true:
// the generic coordinate block (any transform, any fit mode at run time), reached through a real call (run_tile_call).
template <int DP, int G, bool WIDE, bool SLOW, int NT> struct SectorEval {
    static constexpr int NC = 1;
    typedef unsigned Extra;                                  // shared address of the CTA's SectorSmem
    static __device__ __forceinline__ void eval(const typename Res<WIDE>::T (&r)[DP], const SmemCtx<DP, G, NT>&, const unsigned& exbase,
                                                const EvalCtx& cx, double (&acc)[G][1]) {
        double x[G][DP], num[G];
        if (!SLOW) {
            sector_coords<DP, G, WIDE, TR_KOR3, 0>(r, cx, x, num);
        } else {
            sector_coords<DP, G, WIDE, TR_KORR, FIT_RT>(r, cx, x, num);
        }
        // the weights are not needed until the interpreter is done: park them in shared memory ([row][thread], conflict free)
        const unsigned park = exbase + SectorOff::park + 8u * threadIdx.x;
#pragma unroll
        for (int q = 0; q < G; ++q) sts_f64(park + 8u * NT * q, num[q]);
        double F[G];
        {
            const double c0u = lds_f64(exbase + SectorOff::c0u);
#pragma unroll
            for (int q = 0; q < G; ++q) F[q] = c0u;
        }
        sector_interp<DP, G, NT>(x, exbase + SectorOff::words, exbase + SectorOff::slots, park + 64u * NT, F);   // U -> rows 8 ..
#pragma unroll
        for (int q = 0; q < G; ++q) num[q] = lds_f64(park + 8u * NT * q);
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
        double den[G];
#pragma unroll
        for (int q = 0; q < G; ++q) den[q] = 1.0;
        if (pa) {
            double U[G];
#pragma unroll
            for (int q = 0; q < G; ++q) U[q] = lds_f64(park + 8u * NT * (8 + q));
#pragma unroll 1
            for (int e = 0; e < pa; ++e)
#pragma unroll
                for (int q = 0; q < G; ++q) num[q] *= U[q];
        }
        // optional log factor (lu log U + lf log F)^p of an eps-expansion term: a cold, warp-uniform branch (after U^a: the order of the specialised kernels)
        const int lp = (int)(unsigned)lds_u64(exbase + SectorOff::logp);
        if (lp) {
            const double lu = lds_f64(exbase + SectorOff::lg), lf = lds_f64(exbase + SectorOff::lg + 8u);
#pragma unroll
            for (int q = 0; q < G; ++q) sts_f64(park + 8u * NT * q, F[q]);
            sector_log_factors<NT>(park, G, lu, lf, lp);
#pragma unroll
            for (int q = 0; q < G; ++q) num[q] *= lds_f64(park + 8u * NT * q);
        }
#pragma unroll 1
        for (int e = 0; e < pb; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) den[q] *= F[q];
#pragma unroll
        for (int q = 0; q < G; ++q) acc[q][0] = __fma_rn(num[q], rcp_nr(den[q]), acc[q][0]);
    }
};

// The complex sector family (reading C-16): U, F complex-valued polynomials of the real coordinates; f = W prod x^nu U^a / F^b
// in complex arithmetic, two accumulators per shift.  The interpreter parks U as (re, im) row pairs from row 8 on.
template <int DP, int G, bool WIDE, bool SLOW, int NT> struct CSectorEval {
    static constexpr int NC = 2;
    typedef unsigned Extra;
    static __device__ __forceinline__ void eval(const typename Res<WIDE>::T (&r)[DP], const SmemCtx<DP, G, NT>&, const unsigned& exbase,
                                                const EvalCtx& cx, double (&acc)[G][2]) {
        double x[G][DP], w[G];
        if (!SLOW) {
            sector_coords<DP, G, WIDE, TR_KOR3, 0>(r, cx, x, w);
        } else {
            sector_coords<DP, G, WIDE, TR_KORR, FIT_RT>(r, cx, x, w);
        }
        const unsigned park = exbase + SectorOff::park + 8u * threadIdx.x;
#pragma unroll
        for (int q = 0; q < G; ++q) sts_f64(park + 8u * NT * q, w[q]);
        double Fr[G], Fi[G];
        {
            double c0r, c0i;
            lds_f64x2(exbase + SectorOff::c0u, c0r, c0i);
#pragma unroll
            for (int q = 0; q < G; ++q) { Fr[q] = c0r; Fi[q] = c0i; }
        }
        csector_interp<DP, G, NT>(x, exbase + SectorOff::words, exbase + SectorOff::slots, park + 64u * NT, Fr, Fi);
#pragma unroll
        for (int q = 0; q < G; ++q) w[q] = lds_f64(park + 8u * NT * q);
        const unsigned long long nup = lds_u64(exbase + SectorOff::nu);
        const unsigned long long ab = lds_u64(exbase + SectorOff::ab);
        const int pa = (int)(unsigned)ab, pb = (int)(ab >> 32);
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            const int nu = (int)((nup >> (4 * j)) & 15ull);
#pragma unroll 1
            for (int e = 0; e < nu; ++e)
#pragma unroll
                for (int q = 0; q < G; ++q) w[q] *= x[q][j];
        }
        double nr[G], ni[G], Ur[G], Ui[G];
#pragma unroll
        for (int q = 0; q < G; ++q) {
            nr[q] = w[q]; ni[q] = 0.0;
            Ur[q] = lds_f64(park + 8u * NT * (8 + 2 * q)); Ui[q] = lds_f64(park + 8u * NT * (9 + 2 * q));
        }
#pragma unroll 1
        for (int e = 0; e < pa; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) {
                const double t = __fma_rn(nr[q], Ur[q], -(ni[q] * Ui[q]));
                ni[q] = __fma_rn(nr[q], Ui[q], ni[q] * Ur[q]);
                nr[q] = t;
            }
        // optional log factor (lu Log U + lf Log F)^p, principal branch: a cold, warp-uniform branch
        const int lp = (int)(unsigned)lds_u64(exbase + SectorOff::logp);
        if (lp) {
            const double lu = lds_f64(exbase + SectorOff::lg), lf = lds_f64(exbase + SectorOff::lg + 8u);
#pragma unroll 1
            for (int q = 0; q < G; ++q) {
                const double Lr = __fma_rn(lu, 0.5 * log(__fma_rn(Ur[q], Ur[q], Ui[q] * Ui[q])), lf * (0.5 * log(__fma_rn(Fr[q], Fr[q], Fi[q] * Fi[q]))));
                const double Li = __fma_rn(lu, atan2(Ui[q], Ur[q]), lf * atan2(Fi[q], Fr[q]));
                double pr = Lr, pi = Li;
                for (int e = 1; e < lp; ++e) { const double t = pr * Lr - pi * Li; pi = pr * Li + pi * Lr; pr = t; }
                const double t = nr[q] * pr - ni[q] * pi;
                ni[q] = nr[q] * pi + ni[q] * pr;
                nr[q] = t;
            }
        }
        double dr[G], di[G];
#pragma unroll
        for (int q = 0; q < G; ++q) { dr[q] = 1.0; di[q] = 0.0; }
#pragma unroll 1
        for (int e = 0; e < pb; ++e)
#pragma unroll
            for (int q = 0; q < G; ++q) {
                const double t = __fma_rn(dr[q], Fr[q], -(di[q] * Fi[q]));
                di[q] = __fma_rn(dr[q], Fi[q], di[q] * Fr[q]);
                dr[q] = t;
            }
        // n / d = n conj(d) / |d|^2
#pragma unroll
        for (int q = 0; q < G; ++q) {
            const double inv = rcp_nr(__fma_rn(dr[q], dr[q], di[q] * di[q]));
            acc[q][0] = __fma_rn(__fma_rn(nr[q], dr[q], ni[q] * di[q]), inv, acc[q][0]);
            acc[q][1] = __fma_rn(__fma_rn(ni[q], dr[q], -(nr[q] * di[q])), inv, acc[q][1]);
        }
    }
};

// shifts per group and threads per CTA by dimension-slot count (x[G][DP] lives in registers; one CTA per SM)
template <int DP, bool CPLX> struct SectorGroup { static constexpr int value = CPLX ? csector_group(DP) : sector_group(DP); };
template <int DP, bool CPLX> struct SectorThreads { static constexpr int value = CPLX ? kCSectorThreads : sector_threads(DP); };

template <int DP, int G, int NT> struct SectorShared {
    SmemCtx<DP, G, NT> sm;
    SectorSmem<NT> ex;
};

template <int DP, int G, bool WIDE, int NT, bool CPLX>
__global__ void __launch_bounds__(NT, 1) fused_sector_kernel(const __grid_constant__ FusedLaunch L) {
    const DevAux* __restrict__ aux = L.aux;
    const unsigned long long* __restrict__ prog_area = L.prog;
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
            const int tid = threadIdx.x;
            const DevAux& a = aux[cur];
            const DevProblem& pb = sm.prob;
            constexpr int SW = CPLX ? 4 : 2;                 // doubles per coefficient slot
            const int nslots = a.sec_ncoef[0], nwords = a.sec_nops[0];
            const int nmono_total = (pb.n_params - 4 - pb.dim) / sector_mono_stride(pb.family, pb.dim);
            const double* slots = reinterpret_cast<const double*>(prog_area + pb.aux_off);
            const unsigned int* words = reinterpret_cast<const unsigned int*>(prog_area + pb.aux_off + sector_slot_words(nmono_total, CPLX));
            for (int i = tid; i < SW * nslots && i < 4 * kSecMaxSlots; i += NT) ex.slots[i] = slots[i];
            for (int i = tid; i < nwords && i < kSecMaxWords; i += NT) ex.words[i] = words[i];
            if (tid == 32) {
                ex.c0u = a.sec_c0[0]; ex.c0u_im = a.sec_c0i[0];
                ex.a = a.sec_a; ex.b = a.sec_b;
                ex.lg[0] = a.sec_log[0]; ex.lg[1] = a.sec_log[1]; ex.logp = a.sec_logp; ex.sel = 0;
                unsigned long long nup = 0;
                for (int j = 0; j < 16; ++j) nup |= (unsigned long long)(a.nu[j] & 15) << (4 * j);
                ex.nu_packed = nup;
            }
            __syncthreads();
        }
        const bool fast = !sm.prob.has_fit && sm.prob.tr_kind == TR_KOR3;
        if constexpr (CPLX) {
            if (fast) run_tile<CSectorEval<DP, G, WIDE, false, NT>, DP, G, WIDE, NT>(sm, sbase, exbase, tile_local, changed, partials);
            else run_tile_call<CSectorEval<DP, G, WIDE, true, NT>, DP, G, WIDE, NT>(sm, sbase, exbase, tile_local, changed, partials);
        } else {
            if (fast) run_tile<SectorEval<DP, G, WIDE, false, NT>, DP, G, WIDE, NT>(sm, sbase, exbase, tile_local, changed, partials);
            else run_tile_call<SectorEval<DP, G, WIDE, true, NT>, DP, G, WIDE, NT>(sm, sbase, exbase, tile_local, changed, partials);
        }
    }
}

}  // namespace qmc
