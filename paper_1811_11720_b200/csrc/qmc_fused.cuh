// qmc_fused.cuh -- the fused persistent-grid kernel of the R1SL hot path.
//
// One launch serves a queue of tiles (problem, range of lattice indices k).  A CTA of kThreads pops
// tiles from a global counter (S9; the paper's host-side locked work queue is P:L388-L402).  For a
// tile, thread t owns the indices k0 + t + i*kThreads, i < steps.  Shifts are processed G at a
// time: for a group the thread walks its indices, steps the d residues on the integer pipe (S1),
// and evaluates G shifted points per index with all per-shift state in registers (S2-S6).  After
// the walk the G (x ncomp) per-thread sums are reduced by a fixed xor-butterfly + fixed-order
// cross-warp sum and written to the tile's fixed slot (S7).  Results therefore do not depend on
// which CTA ran a tile or in which order.
//
// Template parameters: FAMILY (integrand family), DP (dimension slots held in registers; the
// runtime dim <= DP), G (shifts per group), WIDE (64-bit residues for n >= 2^31).  Transform and
// fit map are runtime (warp-uniform) and select a fully specialised tile loop.
//
// Dimension slots j >= dim are PADDED, not branched around: z_j = 0 and Delta_j = 1/2 pin the slot
// to u = 1/2 (centred coordinate c = 0), the family constants of the slot make its factor exactly
// 1 (or its phase contribution exactly 0), the fit map of the slot is the identity, and a Korobov
// slot contributes u(1-u) = 1/4 to the weight product, which the host compensates in wconst by
// the exact factor 4^r per slot.  The per-point code is therefore one branch-free block and the
// results are bit-identical to skipping the slots.
#pragma once
#include <cstddef>

#include "qmc_device.cuh"

#ifndef QMC_PAIR_DIMS
#define QMC_PAIR_DIMS 1
#endif
#ifndef QMC_PAIR_ND
#define QMC_PAIR_ND 2
#endif

namespace qmc {

template <int FAMILY> struct FamTraits;
template <> struct FamTraits<QMC_FAMILY_GENZ_OSC> { static constexpr int NC = 1; };
template <> struct FamTraits<QMC_FAMILY_GENZ_PRODPEAK> { static constexpr int NC = 1; };
template <> struct FamTraits<QMC_FAMILY_CEXP_POLY> { static constexpr int NC = 2; };
template <> struct FamTraits<kKernelFamilyGenzMisc> { static constexpr int NC = 1; };

// Shared-memory image of the problem a CTA is working on.  The double arrays at the front are the
// operands of the inner loop; they are read with ld.shared at sbase + compile-time offsets.
template <int DP, int G, int NT = kThreads> struct alignas(16) SmemCtx {
    double delta[(DP * G > kDeltaCache) ? DP * G : kDeltaCache];   // [group][j][q] shifts (1/2 in padded slots): all groups of
                                   // the problem when they fit, else only the current group
    double fam[DP * 2];            // [j] = (fam_a, fam_b)
    double fit[DP * 10];           // [j] = (a4, a5, a6, 2 a5, 3 a6, -, a0, a2 (a0-1), a1, a3 (a1-1))  fit map of Eq. 19
    double kor[16];                // transform tables (DevProblem::kor)
    unsigned long long step[DP], back[DP], z[DP];
    double red[2][NT / 32][G * 2]; // double-buffered by group parity
    DevProblem prob;
    double fam0;
    long long tile;                // popped tile index
    int fit_full;                  // the fit map of the problem has pole terms (a2 or a3 non-zero in some dimension)
};
template <int DP, int G> struct SmemOff {
    static constexpr unsigned delta = 0;
    static constexpr unsigned fam = delta + ((DP * G > kDeltaCache) ? DP * G : kDeltaCache) * 8;
    static constexpr unsigned fit = fam + DP * 2 * 8;
    static constexpr unsigned kor = fit + DP * 10 * 8;
    static constexpr unsigned step = kor + 16 * 8;
};

// ---- per-dimension and per-point pieces of the closed-form families (S5) ----------------------
//  OSC       f = cos(2 pi u0 + sum a_j x_j)
//  PRODPEAK  f = prod 1/(c_j^-2 + (x_j - w_j)^2)  = 1 / prod(...)
//  CEXP      f = exp(i sum a_j x_j) prod (1 + b_j x_j)             BASELINE.json configs[2]
//  kernel family 4 (runtime sub-kind = public family id), s0 = the sum below, s1 = 1 once the integrand is cut to 0:
//    CORNER    f = (1 + sum c_j x_j)^-(d+1)                        P:L714-L715   fa = c_j
//    GAUSSIAN  f = exp(-sum c_j^2 (x_j - w_j)^2)                   P:L716-L717   fa = -c_j^2, fb = w_j
//    C0        f = exp(-sum c_j |x_j - w_j|)                       P:L718-L720   fa = -c_j,   fb = w_j
//    DISCONT   f = 0 if x_1 > w_1 or x_2 > w_2 else exp(sum c_j x_j)  P:L721-L722   fa = c_j, fb = w_j (j < 2), +inf beyond
template <int FAMILY> __device__ __forceinline__ void fam_init(double& s0, double& s1, double fam0) {
    if (FAMILY == QMC_FAMILY_GENZ_OSC) { s0 = fam0; s1 = 0.0; }
    else if (FAMILY == QMC_FAMILY_GENZ_PRODPEAK) { s0 = 1.0; s1 = 0.0; }
    else if (FAMILY == kKernelFamilyGenzMisc) { s0 = 0.0; s1 = 0.0; }
    else { s0 = 0.0; s1 = 1.0; }
}
template <int FAMILY> __device__ __forceinline__ void fam_dim(double& s0, double& s1, double x, double fa, double fb, int kind) {
    if (FAMILY == QMC_FAMILY_GENZ_OSC) { s0 = __fma_rn(fa, x, s0); }
    else if (FAMILY == QMC_FAMILY_GENZ_PRODPEAK) { const double t = x - fb; s0 *= __fma_rn(t, t, fa); }   // fa = c_j^-2, fb = w_j
    else if (FAMILY == kKernelFamilyGenzMisc) {
        if (kind == QMC_FAMILY_GENZ_GAUSSIAN) { const double t = x - fb; s0 = __fma_rn(fa * t, t, s0); }
        else if (kind == QMC_FAMILY_GENZ_C0) { s0 = __fma_rn(fa, fabs(x - fb), s0); }
        else { s0 = __fma_rn(fa, x, s0); if (x > fb) s1 = 1.0; }          // corner peak (fb = +inf) and discontinuous
    }
    else { s0 = __fma_rn(fa, x, s0); s1 *= __fma_rn(fb, x, 1.0); }
}
// adds W*f to acc[0..NC); kind / pw: sub-kind and exponent d + 1 of kernel family 4
template <int FAMILY> __device__ __forceinline__ void fam_finish(double s0, double s1, double W, bool use_w, double* acc, int kind, int pw) {
    if (FAMILY == kKernelFamilyGenzMisc) {
        double f;
        if (kind == QMC_FAMILY_GENZ_CORNER) f = rcp_nr(ipow_small(1.0 + s0, pw));
        else f = (s1 != 0.0) ? 0.0 : exp(s0);
        acc[0] = use_w ? __fma_rn(W, f, acc[0]) : acc[0] + f;
        return;
    }
    if (FAMILY == QMC_FAMILY_GENZ_OSC) {
        const double f = cos(s0);
        acc[0] = use_w ? __fma_rn(W, f, acc[0]) : acc[0] + f;
    } else if (FAMILY == QMC_FAMILY_GENZ_PRODPEAK) {
        const double f = rcp_nr(s0);
        acc[0] = use_w ? __fma_rn(W, f, acc[0]) : acc[0] + f;
    } else {
        double sn, cs;
        sincos(s0, &sn, &cs);
        const double a = use_w ? W * s1 : s1;
        acc[0] = __fma_rn(a, cs, acc[0]);
        acc[1] = __fma_rn(a, sn, acc[1]);
    }
}

// ---- S2-S4 for one (shift q, dimension j): coordinate, periodizing transform, fit map ----------
struct FitC {                                     // fit map of one dimension (Eq. 19)
    double f0, f1, f2, f3, f4;                    // a4, a5, a6, 2 a5, 3 a6: cubic part and its derivative
    double a0, k2, a1, k3;                        // poles: a0, a2 (a0 - 1), a1, a3 (a1 - 1)   (fit mode 2 only)
    int mode;                                     // generic tile loop (FIT_RT): fit mode of the problem, warp-uniform
};

// The generic weight transforms (Table A.2), selected per coordinate by the warp-uniform code
// gen = kind | r0 << 4 | r1 << 8; P is multiplied by omega(u) / normalisation (the constant is in wconst).
//   GEN_KOROBOV_SYM   Eq. 15, r0 = r1 = r: phi = 1/2 + c g_r(c^2), omega ~ (1/4 - c^2)^r
//   GEN_KOROBOV_ASYM  Eq. 15, r0 != r1: phi(u) = u^(r0+1) A(u) below 1/2, 1 - v^(r1+1) B(v), v = 1 - u, above
//                     (int_u^1 omega_{r0,r1} = int_0^{1-u} omega_{r1,r0}); tables zero padded to degree 6
//   GEN_SIDI          Eq. 16: omega ~ sin^r(pi u), phi = (K_r / pi) I_r(pi u) with the reduction
//                     I_n = ((n-1) I_{n-2} - sin^(n-1) cos) / n, I_0 = theta, I_1 = 1 - cos
__device__ __forceinline__ double generic_transform(double t, unsigned kor_addr, int gen, double& P) {
    const int kind = gen & 15, r0 = (gen >> 4) & 15, r1 = (gen >> 8) & 15;
    if (kind == GEN_NONE) return wrap_u(t);
    if (kind == GEN_BAKER) return 1.0 - fabs(baker_w(t));
    if (kind == GEN_KOROBOV_SYM) {
        const double c = centre_c(t);
        const double s = c * c;
        P *= ipow_small(0.25 - s, r0);
        double g = lds_f64(kor_addr + 8u * (unsigned)r0);
#pragma unroll 1
        for (int i = r0 - 1; i >= 0; --i) g = __fma_rn(g, s, lds_f64(kor_addr + 8u * (unsigned)i));
        return __fma_rn(c, g, 0.5);
    }
    const double u = wrap_u(t);
    if (kind == GEN_KOROBOV_ASYM) {
        const double um = 1.0 - u;
        const bool low = u <= 0.5;
        const double v = low ? u : um;
        const unsigned tab = kor_addr + (low ? 0u : 64u);
        double h = lds_f64(tab + 48u);
#pragma unroll 1
        for (int i = 5; i >= 0; --i) h = __fma_rn(h, v, lds_f64(tab + 8u * (unsigned)i));
        const double ph = ipow_small(v, (low ? r0 : r1) + 1) * h;
        P *= ipow_small(u, r0) * ipow_small(um, r1);
        return low ? ph : 1.0 - ph;
    }
    double s, c;
    sincospi(u, &s, &c);
    const bool even = (r0 & 1) == 0;
    double I = even ? 3.141592653589793238462643383279 * u : 1.0 - c;
    double sp = even ? s : s * s;                             // sin^(n-1) for the first reduction step
    const double s2 = s * s;
#pragma unroll 1
    for (int n = even ? 2 : 3; n <= r0; n += 2) {
        I = __ddiv_rn(__fma_rn((double)(n - 1), I, -(sp * c)), (double)n);
        sp *= s2;
    }
    P *= ipow_small(s, r0);
    return lds_f64(kor_addr) * I;
}

// Pole terms of the fit function (Eq. 19): adds a2 y (a0-1)/(a0-y) + a3 y (a1-1)/(a1-y) to p and
// a2 a0 (a0-1)/(a0-y)^2 + a3 a1 (a1-1)/(a1-y)^2 to p'; k2 = a2 (a0-1), k3 = a3 (a1-1).  a0 >= 1.001 and a1 <= -0.001
// keep the denominators away from 0 on [0,1].  Only the fit-mode-2 tile loops contain it.
__device__ __forceinline__ void fit_poles(double y, double a0, double k2, double a1, double k3, double& p, double& dp) {
    const double q0 = rcp_nr(a0 - y), q1 = rcp_nr(a1 - y);
    const double e0 = k2 * q0, e1 = k3 * q1;
    p = __fma_rn(y, e0, __fma_rn(y, e1, p));
    dp = __fma_rn(a0 * e0, q0, __fma_rn(a1 * e1, q1, dp));
}

// x^e for 0 <= e <= 7 without a loop or a branch (e is warp-uniform): squarings and selected multipliers
__device__ __forceinline__ double ipow_upto7(double x, int e) {
    const double x2 = x * x, x4 = x2 * x2;
    double r = (e & 1) ? x : 1.0;
    r *= (e & 2) ? x2 : 1.0;
    r *= (e & 4) ? x4 : 1.0;
    return r;
}

// symmetric Korobov weight, any r <= 6: g_r(s) by a fixed six-step Horner scheme on the zero-padded table k (degree r; fma(0, s, k) = k
// exactly, so the padded steps change nothing); P *= 1/4 - c^2, raised to the power r once per point (point_weight)
template <int G>
__device__ __forceinline__ void korobov_sym_points(const double (&t)[G], const double (&k)[7], double (&x)[G], double (&P)[G]) {
#pragma unroll
    for (int q = 0; q < G; ++q) {
        const double c = centre_c(t[q]);
        const double s = c * c;
        P[q] *= (0.25 - s);
        double g = k[6];
#pragma unroll
        for (int i = 5; i >= 0; --i) g = __fma_rn(g, s, k[i]);
        x[q] = __fma_rn(c, g, 0.5);
    }
}

// The three weight transforms of the generic loop for the G shifts of a group, one dimension, straight-line each (see
// generic_coord_group); r0, r1 are warp-uniform.  KIND is a GEN_* code.
template <int G, int KIND>
__device__ __forceinline__ void generic_kind_group(const double (&t)[G], unsigned kor_addr, int r0, int r1, double (&x)[G], double (&P)[G]) {
    if constexpr (KIND == GEN_KOROBOV_SYM) {
        double k[7];
#pragma unroll
        for (int i = 0; i < 7; ++i) k[i] = lds_f64(kor_addr + 8u * i);
        korobov_sym_points<G>(t, k, x, P);
    } else if constexpr (KIND == GEN_KOROBOV_ASYM) {
#pragma unroll
        for (int q = 0; q < G; ++q) {
            const double u = wrap_u(t[q]);
            const double um = 1.0 - u;
            const bool low = u <= 0.5;
            const double v = low ? u : um;
            const unsigned tab = kor_addr + (low ? 0u : 64u);
            double k[7];
#pragma unroll
            for (int i = 0; i < 7; ++i) k[i] = lds_f64(tab + 8u * i);
            double h = k[6];
#pragma unroll
            for (int i = 5; i >= 0; --i) h = __fma_rn(h, v, k[i]);
            const double ph = ipow_upto7(v, (low ? r0 : r1) + 1) * h;
            P[q] *= ipow_upto7(u, r0) * ipow_upto7(um, r1);
            x[q] = low ? ph : 1.0 - ph;
        }
    } else {                                                  // Sidi: I_n = ((n-1) I_(n-2) - sin^(n-1) cos) / n from I_0 = pi u, I_1 = 1 - cos
        const bool even = (r0 & 1) == 0;
        const double K = lds_f64(kor_addr);
#pragma unroll
        for (int q = 0; q < G; ++q) {
            const double u = wrap_u(t[q]);
            double sn, cs;
            sincospi(u, &sn, &cs);
            const double s2 = sn * sn;
            double I = even ? 3.141592653589793238462643383279 * u : 1.0 - cs;
            double sp = even ? sn : s2;                       // sin^(n-1) of the first step (n = 2 or 3)
            // at most three steps (r <= 6): n = 2, 4, 6 or 3, 5; the divisions by n are multiplications by the constants 1/n
            const double n0 = even ? 2.0 : 3.0;
#pragma unroll
            for (int st = 0; st < 3; ++st) {
                const double n = n0 + 2.0 * st;
                const double inv = (st == 0) ? (even ? 0.5 : 1.0 / 3.0) : (st == 1 ? (even ? 0.25 : 0.2) : 1.0 / 6.0);
                const double In = __fma_rn(n - 1.0, I, -(sp * cs)) * inv;
                const bool on = n <= (double)r0;
                I = on ? In : I;
                sp *= s2;
            }
            P[q] *= ipow_upto7(sn, r0);
            x[q] = K * I;
        }
    }
}

// The generic tile loop's S3-S4 for ONE dimension and the G shifts of the group: the transform kind and the fit mode are decided
// once per dimension (warp-uniform branches), the G coordinates inside each branch are straight-line code, so that their
// dependency chains overlap (a DFMA result takes ~35 cycles; decided per coordinate, as in round 1, the chains ran one after the
// other and the generic loop reached 17-19 % of the FP64 peak).  Symmetric Korobov weights carry P = prod (1/4 - c^2) and are
// raised to the power r once per point (point_weight); the others multiply their weight into P directly.
template <int G>
__device__ __forceinline__ void generic_coord_group(const double (&t)[G], unsigned kor_addr, int gen, const FitC& fc, double (&x)[G],
                                                    double (&P)[G], double (&D)[G]) {
    const int kind = gen & 15, r0 = (gen >> 4) & 15, r1 = (gen >> 8) & 15;
    if (kind == GEN_NONE) {
#pragma unroll
        for (int q = 0; q < G; ++q) x[q] = wrap_u(t[q]);
    } else if (kind == GEN_BAKER) {
#pragma unroll
        for (int q = 0; q < G; ++q) x[q] = 1.0 - fabs(baker_w(t[q]));
    } else if (kind == GEN_KOROBOV_SYM) {
        generic_kind_group<G, GEN_KOROBOV_SYM>(t, kor_addr, r0, r1, x, P);
    } else if (kind == GEN_KOROBOV_ASYM) {
        generic_kind_group<G, GEN_KOROBOV_ASYM>(t, kor_addr, r0, r1, x, P);
    } else {
        generic_kind_group<G, GEN_SIDI>(t, kor_addr, r0, r1, x, P);
    }
    if (fc.mode) {                                            // S4: fit map of Eq. 19
#pragma unroll
        for (int q = 0; q < G; ++q) {
            const double y = x[q];
            const double h = __fma_rn(y, __fma_rn(y, fc.f2, fc.f1), fc.f0);
            double dp = __fma_rn(y, __fma_rn(y, fc.f4, fc.f3), fc.f0);
            double xx = y * h;
            if (fc.mode == 2) fit_poles(y, fc.a0, fc.k2, fc.a1, fc.k3, xx, dp);
            D[q] *= dp;
            x[q] = xx;
        }
    }
}

// Returns x_j; multiplies P by u(1-u) (Korobov) and D by p'(y) (fit).
template <int TR, int FIT>
__device__ __forceinline__ double point_coord(double rd, double inv_n, double delta, const FitC& fc, unsigned kor_addr,
                                              int kor_r, double& P, double& D) {
    const double t = coord_t(rd, inv_n, delta);
    double x;
    if (TR == TR_NONE) {
        x = wrap_u(t);
    } else {
        if (TR == TR_BAKER) {
            x = 1.0 - fabs(baker_w(t));                       // Eq. 17: the tent map is even about u = 1/2, no wrap decision needed
        } else if (TR == TR_KOR3) {
            const double c = centre_c(t);
            const double s = c * c;
            P = __dmul_rn(P, __dadd_rn(0.25, -s));            // u (1-u) = 1/4 - c^2 (explicit roundings: every kernel that inlines this takes the same form)
            double g = __fma_rn(-20.0, s, 21.0);              // g_3(s) = 35/16 - 35/4 s + 21 s^2 - 20 s^3
            g = __fma_rn(g, s, -8.75);
            g = __fma_rn(g, s, 2.1875);
            x = __fma_rn(c, g, 0.5);                          // phi(u) = 1/2 + c g(c^2)
        } else {
            x = generic_transform(t, kor_addr, kor_r, P);
        }
    }
    const int mode = (FIT == FIT_RT) ? fc.mode : FIT;
    if (FIT && mode) {                                        // S4: fit map of Eq. 19
        const double y = x;
        const double h = __fma_rn(y, __fma_rn(y, fc.f2, fc.f1), fc.f0);
        double dp = __fma_rn(y, __fma_rn(y, fc.f4, fc.f3), fc.f0);   // cubic part of p'(y)
        x = y * h;                                            // cubic part of p(y)
        if (mode == 2) fit_poles(y, fc.a0, fc.k2, fc.a1, fc.k3, x, dp);
        D *= dp;
    }
    return x;
}

// Weight W = prod_j omega(u_j) p'(y_j) from the carried products (Eq. 12, Eq. 18).
template <int TR, int FIT> __device__ __forceinline__ double point_weight(double P, double D, double wconst, int kor_r) {
    double W = 1.0;
    if (TR == TR_KOR3) W = wconst * (P * P * P);
    else if (TR == TR_KORR || TR >= TR_GEN0) W = wconst * (((kor_r & 15) == GEN_KOROBOV_SYM) ? ipow_small(P, (kor_r >> 4) & 15) : P);   // symmetric Korobov: P = prod (1/4 - c^2)
    if (FIT) W = (TR == TR_KOR3 || TR == TR_KORR || TR >= TR_GEN0) ? W * D : D;
    return W;
}

// operands of dimension slot j: family constants, fit constants, the G shifts of the group
template <int DP, int G, int FIT>
__device__ __forceinline__ void load_slot(unsigned sbase, unsigned delta, int j, int fit_mode, double& fa, double& fb, FitC& fc,
                                          double (&dl)[G]) {
    typedef SmemOff<DP, G> O;
    lds_f64x2(sbase + O::fam + 16u * j, fa, fb);
    const int mode = (FIT == FIT_RT) ? fit_mode : FIT;
    fc.mode = mode;
    if (FIT && mode) {
        lds_f64x2(sbase + O::fit + 80u * j, fc.f0, fc.f1);
        lds_f64x2(sbase + O::fit + 80u * j + 16u, fc.f2, fc.f3);
        fc.f4 = lds_f64(sbase + O::fit + 80u * j + 32u);
        if (mode == 2) {
            lds_f64x2(sbase + O::fit + 80u * j + 48u, fc.a0, fc.k2);
            lds_f64x2(sbase + O::fit + 80u * j + 64u, fc.a1, fc.k3);
        }
    }
    if (G % 2 == 0) {
#pragma unroll
        for (int q = 0; q < G; q += 2) lds_f64x2(delta + 8u * (j * G + q), dl[q], dl[q + 1 < G ? q + 1 : q]);
    } else {
#pragma unroll
        for (int q = 0; q < G; ++q) dl[q] = lds_f64(delta + 8u * (j * G + q));
    }
}

// ---- one lattice index, G shifts: S2-S6 for the closed-form families --------------------------
struct EvalCtx {            // per-tile constants held in registers
    unsigned sbase;         // shared address of the CTA's SmemCtx
    unsigned delta;         // shared address of the current group's shifts
    double inv_n, wconst, fam0;
    int kor_r;              // generic weight transforms: DevProblem::gen
    int fit_mode;           // 0 none, 1 cubic, 2 cubic + pole terms (decided on the device from a2, a3)
    int sel;                // specialised tile loop: tr_kind * 2 + fit_mode, or -1 for the generic loop
    int fam_kind, fam_pow;  // kernel family 4: public family id and the corner-peak exponent d + 1
};

// resident CTAs per SM the register budget is sized for (128 / 168 / 255 registers per thread)
template <int DP, bool WIDE> struct MinBlocks { static constexpr int value = min_blocks_closed(DP, WIDE); };

template <int FAMILY, int DP, int G, bool WIDE, int TR, int FIT>
__device__ __forceinline__ void eval_point_group(const typename Res<WIDE>::T (&r)[DP], const EvalCtx& cx,
                                                 double (&acc)[G][FamTraits<FAMILY>::NC]) {
    double s0[G], s1[G], P[G], D[G];
#pragma unroll
    for (int q = 0; q < G; ++q) { fam_init<FAMILY>(s0[q], s1[q], cx.fam0); P[q] = 1.0; D[q] = 1.0; }
    if constexpr (TR >= TR_GEN0) {
        // dedicated generic kernels: the transform kind is a template parameter and there is no fit map, so the dimensions form one
        // basic block like the specialised loops' (the orders r0, r1 stay run-time values)
        static_assert(FIT == 0, "the dedicated generic kernels have no fit map");
        constexpr int KIND = TR - TR_GEN0;
        const int r0 = (cx.kor_r >> 4) & 15, r1 = (cx.kor_r >> 8) & 15;
        const unsigned kor_addr = cx.sbase + SmemOff<DP, G>::kor;
        double ksym[7];
        if constexpr (KIND == GEN_KOROBOV_SYM) {
#pragma unroll
            for (int i = 0; i < 7; ++i) ksym[i] = lds_f64(kor_addr + 8u * i);
        }
#pragma unroll
        for (int j = 0; j < DP; ++j) {
            const double rd = Res<WIDE>::to_double(r[j]);
            double fa, fb, dl[G], t[G], xg[G];
            FitC fc;
            load_slot<DP, G, 0>(cx.sbase, cx.delta, j, 0, fa, fb, fc, dl);
#pragma unroll
            for (int q = 0; q < G; ++q) t[q] = coord_t(rd, cx.inv_n, dl[q]);
            if constexpr (KIND == GEN_KOROBOV_SYM) korobov_sym_points<G>(t, ksym, xg, P);
            else generic_kind_group<G, KIND>(t, kor_addr, r0, r1, xg, P);
#pragma unroll
            for (int q = 0; q < G; ++q) fam_dim<FAMILY>(s0[q], s1[q], xg[q], fa, fb, cx.fam_kind);
        }
    }
    // Korobov-3 (no fit map / cubic fit map): two dimensions at a time, written stage by stage across the 2 G coordinates, so that
    // the assembler's scheduling window holds twice the independent chains; every coordinate sees the same operations and the
    // products over the dimensions keep their order, so the values are those of the one-dimension-at-a-time form bit for bit
    // (only in the kernels with the 168-register budget, 16 slots: measured, configs[4] 419.4 -> 413.9 ms; at 12 slots and 128 registers
    // configs[2] lost 1.5 % to the registers the second dimension holds)
    constexpr bool PAIRED = QMC_PAIR_DIMS && TR == TR_KOR3 && (FIT == 0 || FIT == 1) && DP % 2 == 0 && !WIDE && MinBlocks<DP, WIDE>::value == 3;
    if constexpr (PAIRED) {
        constexpr int ND = QMC_PAIR_ND;
#pragma unroll
        for (int j = 0; j < DP; j += ND) {
            double fa[ND], fb[ND], dl[ND][G], rd[ND], c[ND][G], sq[ND][G], g[ND][G], x[ND][G];
            FitC fc[ND];
#pragma unroll
            for (int h = 0; h < ND; ++h) {
                rd[h] = Res<WIDE>::to_double(r[j + h]);
                load_slot<DP, G, FIT>(cx.sbase, cx.delta, j + h, cx.fit_mode, fa[h], fb[h], fc[h], dl[h]);
            }
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) c[h][q] = centre_c(coord_t(rd[h], cx.inv_n, dl[h][q]));
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) sq[h][q] = c[h][q] * c[h][q];
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) g[h][q] = __fma_rn(-20.0, sq[h][q], 21.0);
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) g[h][q] = __fma_rn(g[h][q], sq[h][q], -8.75);
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) g[h][q] = __fma_rn(g[h][q], sq[h][q], 2.1875);
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) x[h][q] = __fma_rn(c[h][q], g[h][q], 0.5);
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) P[q] = __dmul_rn(P[q], __dadd_rn(0.25, -sq[h][q]));
            if constexpr (FIT == 1) {
                double dp[ND][G];
#pragma unroll
                for (int h = 0; h < ND; ++h)
#pragma unroll
                    for (int q = 0; q < G; ++q) {
                        const double y = x[h][q];
                        const double hh = __fma_rn(y, __fma_rn(y, fc[h].f2, fc[h].f1), fc[h].f0);
                        dp[h][q] = __fma_rn(y, __fma_rn(y, fc[h].f4, fc[h].f3), fc[h].f0);
                        x[h][q] = y * hh;
                    }
#pragma unroll
                for (int h = 0; h < ND; ++h)
#pragma unroll
                    for (int q = 0; q < G; ++q) D[q] *= dp[h][q];
            }
#pragma unroll
            for (int h = 0; h < ND; ++h)
#pragma unroll
                for (int q = 0; q < G; ++q) fam_dim<FAMILY>(s0[q], s1[q], x[h][q], fa[h], fb[h], cx.fam_kind);
        }
    }
#pragma unroll
    for (int j = 0; j < ((TR >= TR_GEN0 || PAIRED) ? 0 : DP); ++j) {
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
            for (int q = 0; q < G; ++q) fam_dim<FAMILY>(s0[q], s1[q], xg[q], fa, fb, cx.fam_kind);
        } else {
#pragma unroll
            for (int q = 0; q < G; ++q) {
                if (FAMILY == QMC_FAMILY_GENZ_PRODPEAK && TR == TR_BAKER && !FIT) {
                    // x - w_j = (1 - w_j) - |w| with the slot constant fb = 1 - w_j (derive_slot): the baker map folds into the factor
                    const double dd = fb - fabs(baker_w(coord_t(rd, cx.inv_n, dl[q])));
                    s0[q] *= __fma_rn(dd, dd, fa);
                } else {
                    const double x = point_coord<TR, FIT>(rd, cx.inv_n, dl[q], fc, cx.sbase + SmemOff<DP, G>::kor, cx.kor_r, P[q], D[q]);
                    fam_dim<FAMILY>(s0[q], s1[q], x, fa, fb, cx.fam_kind);
                }
            }
        }
    }
    constexpr bool USEW = (TR == TR_KOR3 || TR == TR_KORR || TR >= TR_GEN0 || FIT != 0);
#pragma unroll
    for (int q = 0; q < G; ++q)
        fam_finish<FAMILY>(s0[q], s1[q], point_weight<TR, FIT>(P[q], D[q], cx.wconst, cx.kor_r), USEW, acc[q], cx.fam_kind, cx.fam_pow);
}

struct NoExtra {};

template <int FAMILY, int DP, int G, bool WIDE, int TR, int FIT> struct ClosedEval {
    static constexpr int NC = FamTraits<FAMILY>::NC;
    typedef NoExtra Extra;
    static __device__ __forceinline__ void eval(const typename Res<WIDE>::T (&r)[DP], const SmemCtx<DP, G>&, const Extra&,
                                                const EvalCtx& cx, double (&acc)[G][NC]) {
        eval_point_group<FAMILY, DP, G, WIDE, TR, FIT>(r, cx, acc);
    }
};

// ---- one tile: residue walk (S1), G shifts per index (EV::eval = S2-S6), tile reduction (S7) ----
template <class EV, int DP, int G, bool WIDE, int NT = kThreads>
__device__ __forceinline__ void run_tile(SmemCtx<DP, G, NT>& sm, unsigned sbase, const typename EV::Extra& ex, long long tile_local,
                                         bool changed, double* __restrict__ partials) {
    typedef typename Res<WIDE>::T RT;
    constexpr int NC = EV::NC;
    constexpr int kThreads = NT, kWarps = NT / 32;           // threads of this kernel variant (shadow the closed-form default)
    // residue strides live in registers while they are few; otherwise they are re-read from shared memory
    constexpr bool STEP_IN_REGS = DP * (WIDE ? 2 : 1) <= 16;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const DevProblem& pb = sm.prob;
    const int dim = pb.dim, m = pb.m, steps = pb.steps;
    const unsigned long long n = pb.n;
    EvalCtx cx;
    cx.sbase = sbase; cx.inv_n = pb.inv_n; cx.wconst = pb.wconst; cx.fam0 = sm.fam0; cx.kor_r = pb.gen;
    cx.fit_mode = pb.has_fit ? 1 + sm.fit_full : 0;
    cx.sel = (pb.tr_kind != TR_KORR && cx.fit_mode <= 1) ? pb.tr_kind * 2 + cx.fit_mode : -1;
    cx.fam_kind = pb.family; cx.fam_pow = pb.dim + 1;
    typedef SmemCtx<DP, G, NT> Ctx;
    typedef SmemOff<DP, G> Off;
    static_assert(offsetof(Ctx, fam) == Off::fam && offsetof(Ctx, fit) == Off::fit && offsetof(Ctx, kor) == Off::kor &&
                  offsetof(Ctx, step) == Off::step, "SmemOff must mirror SmemCtx");
    const unsigned long long tile_len = (unsigned long long)pb.tile_len;
    const unsigned long long k0 = (unsigned long long)tile_local * tile_len;
    const unsigned long long kend = (k0 + tile_len < n) ? k0 + tile_len : n;
    const unsigned long long kfirst = k0 + tid;
    const int live_steps = kfirst < kend ? (int)((kend - kfirst + kThreads - 1) / kThreads) : 0;   // indices this thread owns

    RT r[DP], stp[STEP_IN_REGS ? DP : 1];
#pragma unroll
    for (int j = 0; j < DP; ++j) {
        r[j] = (RT)mulmod_u64(kfirst % n, sm.z[j], n);          // padded slots: z = 0 -> r = 0
        if (STEP_IN_REGS) stp[j] = (RT)sm.step[j];
    }

    // shifts: staged once per problem for all groups when they fit the shared-memory cache, else per group
    const int ngroups = (m + G - 1) / G;
    const bool cached = ngroups * (DP * G) <= (int)(sizeof(sm.delta) / sizeof(double));
    if (cached && changed) {
        for (int e = tid; e < ngroups * G * DP; e += kThreads) {
            const int g = e / (G * DP), rest = e - g * (G * DP), j = rest / G, s = g * G + (rest - j * G);
            sm.delta[e] = (s < m && j < dim) ? pb.shifts[(size_t)s * dim + j] : 0.5;
        }
        __syncthreads();
    }

#pragma unroll 1
    for (int g0 = 0, gi = 0; g0 < m; g0 += G, ++gi) {
        const int gcount = (m - g0 < G) ? (m - g0) : G;
        if (!cached) {
            __syncthreads();                                // previous group's readers of delta are done
            for (int e = tid; e < G * DP; e += kThreads) {
                const int j = e / G, q = e - j * G;
                sm.delta[e] = (q < gcount && j < dim) ? pb.shifts[(size_t)(g0 + q) * dim + j] : 0.5;
            }
            __syncthreads();
        }
        cx.delta = sbase + SmemOff<DP, G>::delta + (cached ? 8u * (unsigned)(gi * (G * DP)) : 0u);

        double acc[G][NC];
#pragma unroll
        for (int q = 0; q < G; ++q)
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[q][c] = 0.0;

#pragma unroll 1
        for (int i = 0; i < live_steps; ++i) {
            EV::eval(r, sm, ex, cx, acc);
#pragma unroll
            for (int j = 0; j < DP; ++j)
                r[j] = add_mod<RT>(r[j], STEP_IN_REGS ? stp[STEP_IN_REGS ? j : 0] : (RT)lds_u64(sbase + SmemOff<DP, G>::step + 8u * j), (RT)n);
        }
        // rewind to the thread's first index for the next group: back = steps * kThreads * z_j rewinds a full walk; a
        // thread one index short (ragged tile length) takes one step forward after it; anything else recomputes
        if (g0 + G < m) {
            if (live_steps + 1 >= steps) {
#pragma unroll
                for (int j = 0; j < DP; ++j) {
                    RT v = sub_mod<RT>(r[j], (RT)sm.back[j], (RT)n);
                    if (live_steps != steps) v = add_mod<RT>(v, (RT)sm.step[j], (RT)n);
                    r[j] = v;
                }
            } else {
#pragma unroll
                for (int j = 0; j < DP; ++j) r[j] = (RT)mulmod_u64(kfirst % n, sm.z[j], n);
            }
        }

        // S7: fixed-shape reduction of the group's sums, one slot per (tile, shift, component)
#pragma unroll
        for (int q = 0; q < G; ++q)
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                const double v = warp_sum(acc[q][c]);
                if (lane == 0) sm.red[gi & 1][warp][q * NC + c] = v;
            }
        __syncthreads();                                    // one barrier per group: red is double-buffered by group parity
        if (tid < G * NC) {
            const int q = tid / NC, c = tid - q * NC;
            if (q < gcount) {
                double v = sm.red[gi & 1][0][tid];
#pragma unroll
                for (int w = 1; w < kWarps; ++w) v += sm.red[gi & 1][w][tid];
                partials[pb.partial_off + ((long long)(g0 + q) * NC + c) * pb.tiles + tile_local] = v;
            }
        }
    }
}

// the same tile loop as a real (not inlined) call: used for the correctness paths so that their register needs stay theirs
template <class EV, int DP, int G, bool WIDE, int NT = kThreads>
__device__ __noinline__ void run_tile_call(SmemCtx<DP, G, NT>& sm, unsigned sbase, const typename EV::Extra& ex, long long tile_local,
                                           bool changed, double* __restrict__ partials) {
    run_tile<EV, DP, G, WIDE, NT>(sm, sbase, ex, tile_local, changed, partials);
}

// ---- S0: per-slot constants of a problem, derived from the caller's arrays ------------------------
// z mod n, the residue stride between a thread's points (threads z_j mod n), the rewind of a full walk, the family
// constants and the cubic-map constants of dimension slot j.  Slots j >= dim get the padding values (file header).
struct SlotConst {
    unsigned long long z, step, back;
    double fa, fb, f[9];
};
__device__ __forceinline__ SlotConst derive_slot(const DevProblem& pb, int j, int threads = kThreads) {
    SlotConst s;
    s.z = 0; s.step = 0; s.back = 0; s.fa = 0.0; s.fb = 0.0;
    s.f[0] = 1.0; s.f[1] = s.f[2] = s.f[3] = s.f[4] = 0.0;
    s.f[5] = 2.0; s.f[6] = 0.0; s.f[7] = -1.0; s.f[8] = 0.0;       // no pole terms (identity map in padded slots)
    const int d = pb.dim;
    const unsigned long long n = pb.n;
    if (j < d) {
        s.z = pb.z[j] % n;
        s.step = mulmod_u64((unsigned long long)threads % n, s.z, n);
        s.back = mulmod_u64(((unsigned long long)pb.steps * threads) % n, s.z, n);
        const double* p = pb.params;
        if (pb.family == QMC_FAMILY_GENZ_OSC) { s.fa = p[1 + j]; }
        else if (pb.family == QMC_FAMILY_GENZ_PRODPEAK) { const double c = p[j]; s.fa = __ddiv_rn(1.0, __dmul_rn(c, c)); s.fb = p[d + j]; }
        else if (pb.family == QMC_FAMILY_CEXP_POLY) { s.fa = p[j]; s.fb = p[d + j]; }
        else if (pb.family == QMC_FAMILY_GENZ_CORNER) { s.fa = p[j]; s.fb = __longlong_as_double(0x7ff0000000000000ll); }
        else if (pb.family == QMC_FAMILY_GENZ_GAUSSIAN) { s.fa = -__dmul_rn(p[j], p[j]); s.fb = p[d + j]; }
        else if (pb.family == QMC_FAMILY_GENZ_C0) { s.fa = -p[j]; s.fb = p[d + j]; }
        else if (pb.family == QMC_FAMILY_GENZ_DISCONT) { s.fa = p[j]; s.fb = j < 2 ? p[d + j] : __longlong_as_double(0x7ff0000000000000ll); }
        if (pb.has_fit) {
            const double* c = pb.fit + 6 * j;
            const double a4 = c[4], a5 = c[5];
            const double a6 = __dadd_rn(__dadd_rn(__dadd_rn(__dadd_rn(1.0, -c[2]), -c[3]), -a4), -a5);
            s.f[0] = a4; s.f[1] = a5; s.f[2] = a6; s.f[3] = 2.0 * a5; s.f[4] = 3.0 * a6;
            s.f[5] = c[0]; s.f[6] = __dmul_rn(c[2], __dadd_rn(c[0], -1.0)); s.f[7] = c[1]; s.f[8] = __dmul_rn(c[3], __dadd_rn(c[1], -1.0));
        }
    } else if (pb.family == QMC_FAMILY_GENZ_CORNER || pb.family == QMC_FAMILY_GENZ_DISCONT) {
        s.fb = __longlong_as_double(0x7ff0000000000000ll);      // padded slot: fa = 0 adds nothing, x > +inf never cuts
    } else if (pb.family == QMC_FAMILY_GENZ_PRODPEAK) {
        // padded slot: the coordinate is pinned to u = 1/2, i.e. x = 1 (baker) or 1/2; factor (x - fb)^2 + fa = 1
        s.fa = 1.0;
        s.fb = (pb.tr_kind == TR_BAKER) ? 1.0 : 0.5;
    }
    // product peak under the baker map without fit: the fused kernel wants 1 - w_j (eval_point_group)
    if (pb.family == QMC_FAMILY_GENZ_PRODPEAK && pb.tr_kind == TR_BAKER && !pb.has_fit) s.fb = __dadd_rn(1.0, -s.fb);
    return s;
}
__device__ __forceinline__ int fit_has_poles(const DevProblem& pb) {       // a2 or a3 non-zero in some dimension (Eq. 19)
    int any = 0;
    if (pb.has_fit)
        for (int j = 0; j < pb.dim; ++j) any |= (pb.fit[6 * j + 2] != 0.0 || pb.fit[6 * j + 3] != 0.0) ? 1 : 0;
    return any;
}
__device__ __forceinline__ double derive_fam0(const DevProblem& pb) {
    return (pb.family == QMC_FAMILY_GENZ_OSC) ? __dmul_rn(6.283185307179586476925286766559, pb.params[0]) : 0.0;
}

// ---- tile source shared by all fused kernels ---------------------------------------------------
// Next tile of this CTA; returns false when there is none.  On a problem change the CTA rebuilds its
// shared-memory image of the problem (changed = true): closed-form families derive the slot constants
// themselves (S0), the sector family reads what prepare_kernel left in DevAux.
// `cur` = problem index loaded (-1: none), `iter` = tiles this CTA has taken (single mode).
template <int DP, int G, bool SECTOR, int NT = kThreads>
__device__ __forceinline__ bool next_tile(SmemCtx<DP, G, NT>& sm, const FusedLaunch& L, int& cur, int& iter, long long& tile_local,
                                          bool& changed) {
    constexpr int kThreads = NT;
    const int tid = threadIdx.x;
    changed = false;
    __syncthreads();                                        // everyone is done with the previous tile
    int pidx = 0;
    if (L.single && L.vq.counter == nullptr) {              // at most one tile per CTA: no queue needed
        tile_local = (long long)blockIdx.x + (long long)iter * gridDim.x;
        ++iter;
        if (tile_local >= L.one.tiles) return false;
    } else if (L.single) {
        if (tid == 0) sm.tile = (long long)atomicAdd(L.vq.counter, 1ull);
        __syncthreads();
        tile_local = sm.tile;
        if (tile_local >= L.one.tiles) return false;
    } else {
        if (tid == 0) sm.tile = (long long)atomicAdd(L.vq.counter, 1ull);
        __syncthreads();
        const long long tile = sm.tile;
        if (tile >= L.vq.total_tiles) return false;
        int lo = 0, hi = L.vq.plist_len;                    // largest lo with tile_prefix[lo] <= tile
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(&L.vq.tile_prefix[mid]) <= tile) lo = mid; else hi = mid;
        }
        tile_local = tile - __ldg(&L.vq.tile_prefix[lo]);
        pidx = __ldg(&L.vq.plist[lo]);
    }
    if (pidx != cur) {
        cur = pidx;
        changed = true;
        const DevProblem& src = L.single ? L.one : L.probs[pidx];
        if (tid == 0) sm.prob = src;
        if (tid >= 64 && tid < 80) sm.kor[tid - 64] = src.kor[tid - 64];
        if (SECTOR) {
            const DevAux& a = L.aux[pidx];
            if (tid == 32) sm.fam0 = a.fam0;
            if (tid == 96) sm.fit_full = a.fit_full;
            for (int j = tid; j < DP; j += kThreads) {      // slots j >= dim hold the padding values
                sm.z[j] = a.z[j]; sm.step[j] = a.step[j]; sm.back[j] = a.back[j];
                sm.fam[2 * j] = a.fam_a[j]; sm.fam[2 * j + 1] = a.fam_b[j];
#pragma unroll
                for (int i = 0; i < 5; ++i) sm.fit[10 * j + i] = a.fit[i][j];
                sm.fit[10 * j + 5] = 0.0;
#pragma unroll
                for (int i = 5; i < 9; ++i) sm.fit[10 * j + 1 + i] = a.fit[i][j];
            }
        } else {
            if (tid == 32) sm.fam0 = derive_fam0(src);
            if (tid == 96) sm.fit_full = fit_has_poles(src);
            for (int j = tid; j < DP; j += kThreads) {
                const SlotConst s = derive_slot(src, j);
                sm.z[j] = s.z; sm.step[j] = s.step; sm.back[j] = s.back;
                sm.fam[2 * j] = s.fa; sm.fam[2 * j + 1] = s.fb;
#pragma unroll
                for (int i = 0; i < 5; ++i) sm.fit[10 * j + i] = s.f[i];
                sm.fit[10 * j + 5] = 0.0;
#pragma unroll
                for (int i = 5; i < 9; ++i) sm.fit[10 * j + 1 + i] = s.f[i];
            }
        }
        __syncthreads();
        // product peak: a padded slot must see x - fb = 0, and phi(1/2) is not 1/2 for asymmetric weights -- take it from
        // the device function of the generic loop (for none / baker / Korobov it returns exactly 1/2, 1, 1/2 as the
        // specialised loops do); the folded baker path keeps its own constant (derive_slot)
        if (!SECTOR && src.family == QMC_FAMILY_GENZ_PRODPEAK && src.dim < DP && !(src.tr_kind == TR_BAKER && !src.has_fit)) {
            if (tid >= src.dim && tid < DP) {
                double Pdummy = 1.0;
                sm.fam[2 * tid + 1] = generic_transform(0.5, (unsigned)__cvta_generic_to_shared(&sm) + SmemOff<DP, G>::kor, src.gen, Pdummy);
            }
            __syncthreads();
        }
    }
    return true;
}


template <int FAMILY, int DP, int G, bool WIDE>
__global__ void __launch_bounds__(kThreads, MinBlocks<DP, WIDE>::value) fused_kernel(const __grid_constant__ FusedLaunch L) {
    __shared__ SmemCtx<DP, G> sm;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(&sm);
    int cur = -1, iter = 0;
    long long tile_local = 0;
    bool changed;
    NoExtra ex;
    while (next_tile<DP, G, false>(sm, L, cur, iter, tile_local, changed)) {
        // six specialised tile loops (none / baker / Korobov-3 x no fit / cubic fit) are inlined; every other combination
        // (generic weight transforms, pole-term fit) runs the generic loop through a real call, so that it costs the
        // specialised loops no registers
        const int fit_mode = sm.prob.has_fit ? 1 + sm.fit_full : 0;
        const int sel = (sm.prob.tr_kind != TR_KORR && fit_mode <= 1) ? sm.prob.tr_kind * 2 + fit_mode : -1;
        switch (sel) {
#define QMC_FAST(TRK, FITM) \
    case TRK * 2 + FITM: run_tile<ClosedEval<FAMILY, DP, G, WIDE, TRK, FITM>, DP, G, WIDE>(sm, sbase, ex, tile_local, changed, L.partials); break;
            QMC_FAST(TR_NONE, 0) QMC_FAST(TR_NONE, 1) QMC_FAST(TR_BAKER, 0) QMC_FAST(TR_BAKER, 1) QMC_FAST(TR_KOR3, 0) QMC_FAST(TR_KOR3, 1)
#undef QMC_FAST
            default: run_tile_call<ClosedEval<FAMILY, DP, G, WIDE, TR_KORR, FIT_RT>, DP, G, WIDE>(sm, sbase, ex, tile_local, changed, L.partials); break;
        }
    }
}

// The generic weight transforms without a fit map as kernels of their own (TRG = TR_GEN0 + GEN_* kind): inside fused_kernel the generic
// loop is a call target that must live with the register cap of the specialised loops and decides the kind per dimension; here
// the kind is fixed at compile time and the register budget is the kernel's own.  32-bit residues only; fit maps, n >= 2^31
// and dim > 16 keep the generic loop of fused_kernel.
template <int FAMILY, int DP, int G, int TRG>
__global__ void __launch_bounds__(kThreads, min_blocks_generic(DP)) fused_generic_kernel(const __grid_constant__ FusedLaunch L) {
    __shared__ SmemCtx<DP, G> sm;
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(&sm);
    int cur = -1, iter = 0;
    long long tile_local = 0;
    bool changed;
    NoExtra ex;
    while (next_tile<DP, G, false>(sm, L, cur, iter, tile_local, changed))
        run_tile<ClosedEval<FAMILY, DP, G, false, TRG, 0>, DP, G, false>(sm, sbase, ex, tile_local, changed, L.partials);
}

}  // namespace qmc
