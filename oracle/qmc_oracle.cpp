// qmc_oracle.cpp -- CPU ORACLE for the rank-1 shifted lattice rule of arXiv:1811.11720.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference leg may load it.  It shares no code, header, table
// or constant with the CUDA path under paper_1811_11720_b200/csrc/ and neither includes the other.
//
// It is the paper's equations executed literally in fp64 (PAPER.md = /root/reference/PAPER.md,
// cited as P:L<line>):
//   O1  r_{k,j} = (k * z_j) mod n with an unsigned __int128 product           Eq. 2
//   O2  u = wrap(fma(double(r), 1/double(n), Delta_{s,j}))  "{ } = fractional part", P:L100;
//       the fp64 realisation is DESIGN.md reading C-2
//   O3  (y, w) = periodizing transform: None (Table A.2), baker Eq. 17 P:L204-L209,
//       Korobov weights (r0, r1) Eq. 15 P:L189-L193 and Sidi weight r Eq. 16, phi = int_0^u omega (Eq. 14)
//   O4  optional fit map x = p(y), w *= p'(y)         Eq. 18-19, order P:L338
//   O5  v = (prod_j w_j) * f(x)                                           Eq. 12-13
//   O6  S_s = sum_k v (Neumaier-compensated), Q_s = S_s / n                       Eq. 2
//   O7  Qbar = (sum_s Q_s) / m                                                    Eq. 2
//   O8  err = sqrt( sum_s (Q_s - Qbar)^2 / (m (m-1)) ), per component            Eq. 3
//   O9  projection histogram for the CDF of |f| (Eq. 20) and the cubic fit (C-8)
// The only liberty taken with Eq. 2 is a loop interchange: the residues of index k do not depend
// on the shift, so they are formed once per k and reused for all shifts; every per-shift sum still
// adds its terms in increasing k.  OpenMP runs fixed chunks of 2^16 consecutive k; chunk sums are
// combined in chunk order, so results do not depend on the thread count.
//
// Pins (tests/test_oracle_pins.py, all `-m "not gpu"`; table in DESIGN.md section 6): Fig. 1 lattice n=55 z=(1,34) P:L108;
// by-hand lattices n=7 z=(1,3), n=11 z=(1,7) P:L1050; residue permutation property; exact-rational coordinates;
// Fourier-mode exactness / dual-lattice modes; the one-dimensional rule as an exact geometric series; Eq. 15 normalisation
// and phi = regularised incomplete beta (symmetric and asymmetric weights); Eq. 16 constants and Gauss-Legendre
// quadrature of the Sidi weight; closed forms of families 0-2 and 4-7 (Genz 1-6); tensor Gauss-Legendre for
// the sector family at d<=3; x0*x1*x2 -> 1/8 (Fig. 2); log factors of the sector family by one-dimensional
// closed forms and the eps-derivative identity; Eq. 3 on hand-made means; projection marginals in
// closed form; fit recovers an exact cubic.
// Parity unpinned: nothing in this file (the CBC tool is not part of the oracle; the bounded fit of Eq. 19 has its oracle
// counterpart in oracle/__init__.py: fit_polysingular_pairs).
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef unsigned __int128 u128;

enum { FAM_OSC = 0, FAM_PRODPEAK = 1, FAM_CEXP = 2, FAM_SECTOR = 3, FAM_CORNER = 4, FAM_GAUSS = 5, FAM_C0 = 6, FAM_DISC = 7,
       FAM_CSECTOR = 8 };
const int FAM_LAST = FAM_CSECTOR;
// transform ids: Table A.2.  Korobov<r> = 100 + r; Sidi<r> = 200 + r; Korobov<r0,r1> = 1000 + 16 r0 + r1.
enum { TR_NONE = 0, TR_BAKER = 1, TR_KOROBOV = 100, TR_SIDI = 200, TR_KOROBOV_ASYM = 1000 };
const int MAX_DIM = 64;
const uint64_t CHUNK = 1ull << 16;

// Neumaier's compensated sum (improved Kahan-Babuska).
struct Comp {
    double s = 0.0, c = 0.0;
    void add(double v) {
        double t = s + v;
        if (std::fabs(s) >= std::fabs(v)) c += (s - t) + v; else c += (v - t) + s;
        s = t;
    }
    double value() const { return s + c; }
};

// O1: exact residue, Eq. 2: i*z mod n.
inline uint64_t residue(uint64_t k, uint64_t z, uint64_t n) { return (uint64_t)(((u128)k * (u128)z) % (u128)n); }

// O2: fractional part {r/n + Delta}, reading C-2(B): one fused rounding, exact wrap.
inline double coordinate(uint64_t r, double inv_n, double delta) {
    double t = std::fma((double)r, inv_n, delta);
    return t >= 1.0 ? t - 1.0 : t;
}

double binom(int a, int b) { double v = 1.0; for (int i = 1; i <= b; ++i) v = v * (double)(a - b + i) / (double)i; return v; }

// Korobov transform, Eq. 15, weights (r0, r1):
//   omega(u) = (r0+r1+1) C(r0+r1,r0) u^r0 (1-u)^r1,
//   phi(u) = int_0^u omega = c sum_{i=0}^{r1} C(r1,i) (-1)^i u^{r0+1+i} / (r0+1+i)      (Eq. 14, binomial expansion)
// phi is evaluated by Horner for u <= 1/2 and as 1 - phi_{r1,r0}(1-u) above (int_u^1 omega_{r0,r1} = int_0^{1-u} omega_{r1,r0}).
struct Korobov {
    int r0, r1; double c; double lo[8], hi[8];
    explicit Korobov(int r) : Korobov(r, r) {}
    Korobov(int r0_, int r1_) : r0(r0_), r1(r1_) {
        c = (double)(r0 + r1 + 1) * binom(r0 + r1, r0);
        for (int i = 0; i <= r1; ++i) lo[i] = c * binom(r1, i) * ((i & 1) ? -1.0 : 1.0) / (double)(r0 + 1 + i);
        for (int i = 0; i <= r0; ++i) hi[i] = c * binom(r0, i) * ((i & 1) ? -1.0 : 1.0) / (double)(r1 + 1 + i);
    }
    static double series(const double* coef, int deg, int lead, double u) {   // u^(lead+1) * Horner(coef[0..deg], u)
        double h = coef[deg];
        for (int i = deg - 1; i >= 0; --i) h = h * u + coef[i];
        double p = 1.0; for (int i = 0; i <= lead; ++i) p *= u;
        return p * h;
    }
    double phi(double u) const { return u <= 0.5 ? series(lo, r1, r0, u) : 1.0 - series(hi, r0, r1, 1.0 - u); }
    double omega(double u) const {
        double p = 1.0;
        for (int i = 0; i < r0; ++i) p *= u;
        for (int i = 0; i < r1; ++i) p *= 1.0 - u;
        return c * p;
    }
};

// Sidi transform of weight r, Eq. 16: omega(u) = K_r sin^r(pi u), K_r = pi/2^r Gamma(r+1)/Gamma((r+1)/2)^2;
// phi = int_0^u omega written out per r (s = sin pi u, c = cos pi u):
//   r=1  (1-c)/2                         r=2  u - sin(2 pi u)/(2 pi)
//   r=3  (2 - 3c + c^3)/4                r=4  u - 2 sin(2 pi u)/(3 pi) + sin(4 pi u)/(12 pi)
//   r=5  1/2 - 15c/16 + 5c^3/8 - 3c^5/16 r=6  u - 3 sin(2 pi u)/(4 pi) + 3 sin(4 pi u)/(20 pi) - sin(6 pi u)/(60 pi)
struct Sidi {
    int r; double K;
    explicit Sidi(int r_) : r(r_) { double g = std::tgamma(0.5 * (r + 1)); K = M_PI / std::ldexp(1.0, r) * std::tgamma(r + 1.0) / (g * g); }
    double omega(double u) const { double s = std::sin(M_PI * u), p = 1.0; for (int i = 0; i < r; ++i) p *= s; return K * p; }
    double phi(double u) const {
        const double t = M_PI * u, c = std::cos(t);
        switch (r) {
            case 1: return 0.5 * (1.0 - c);
            case 2: return u - std::sin(2.0 * t) / (2.0 * M_PI);
            case 3: return 0.25 * (2.0 - 3.0 * c + c * c * c);
            case 4: return u - 2.0 * std::sin(2.0 * t) / (3.0 * M_PI) + std::sin(4.0 * t) / (12.0 * M_PI);
            case 5: return 0.5 - 15.0 * c / 16.0 + 5.0 * c * c * c / 8.0 - 3.0 * c * c * c * c * c / 16.0;
            default: return u - 3.0 * std::sin(2.0 * t) / (4.0 * M_PI) + 3.0 * std::sin(4.0 * t) / (20.0 * M_PI) - std::sin(6.0 * t) / (60.0 * M_PI);
        }
    }
};

// decoded transform of a call
struct Transform {
    int kind;                 // 0 none, 1 baker, 2 Korobov (any weights), 3 Sidi
    Korobov kor; Sidi sidi;
    Transform() : kind(0), kor(1), sidi(1) {}
};
inline bool decode_transform(int tr, Transform* t) {
    if (tr == TR_NONE) { t->kind = 0; return true; }
    if (tr == TR_BAKER) { t->kind = 1; return true; }
    if (tr >= TR_KOROBOV + 1 && tr <= TR_KOROBOV + 6) { t->kind = 2; t->kor = Korobov(tr - TR_KOROBOV); return true; }
    if (tr >= TR_SIDI + 1 && tr <= TR_SIDI + 6) { t->kind = 3; t->sidi = Sidi(tr - TR_SIDI); return true; }
    if (tr >= TR_KOROBOV_ASYM) {
        const int r0 = (tr - TR_KOROBOV_ASYM) / 16, r1 = (tr - TR_KOROBOV_ASYM) % 16;
        if (r0 >= 1 && r0 <= 6 && r1 >= 1 && r1 <= 6) { t->kind = 2; t->kor = Korobov(r0, r1); return true; }
    }
    return false;
}

// O3
inline void transform(const Transform& tr, double u, double* y, double* w) {
    if (tr.kind == 0) { *y = u; *w = 1.0; }
    else if (tr.kind == 1) { *y = 1.0 - std::fabs(2.0 * u - 1.0); *w = 1.0; }     // Eq. 17
    else if (tr.kind == 2) { *y = tr.kor.phi(u); *w = tr.kor.omega(u); }          // Eq. 15
    else { *y = tr.sidi.phi(u); *w = tr.sidi.omega(u); }                          // Eq. 16
}

// O4: Eq. 19 and its derivative; a[0..5] = a_0..a_5, a6 = 1 - a2 - a3 - a4 - a5.
inline void fit_map(const double* a, double y, double* x, double* dp) {
    double a6 = 1.0 - a[2] - a[3] - a[4] - a[5];
    double p = y * (a[4] + y * (a[5] + y * a6));
    double d = a[4] + y * (2.0 * a[5] + 3.0 * a6 * y);
    if (a[2] != 0.0) { p += a[2] * y * (a[0] - 1.0) / (a[0] - y); d += a[2] * a[0] * (a[0] - 1.0) / ((a[0] - y) * (a[0] - y)); }
    if (a[3] != 0.0) { p += a[3] * y * (a[1] - 1.0) / (a[1] - y); d += a[3] * a[1] * (a[1] - 1.0) / ((a[1] - y) * (a[1] - y)); }
    *x = p; *dp = d;
}

inline double ipow(double x, int e) { double p = 1.0; for (int i = 0; i < e; ++i) p *= x; return p; }

// Sparse polynomial sum_t c_t prod_j x_j^{e_{t,j}}; exponents stored as doubles.
double sparse_poly(const double* c, const double* e, int count, int dim, const double* x) {
    double s = 0.0;
    for (int t = 0; t < count; ++t) {
        double mon = c[t];
        for (int j = 0; j < dim; ++j) mon *= ipow(x[j], (int)e[t * dim + j]);
        s += mon;
    }
    return s;
}

// O5: the integrand families (layouts: DESIGN.md reading C-7).
//  0 Genz oscillatory  f = cos(2 pi u0 + sum a_j x_j)
//  1 Genz product peak f = prod 1/(c_j^-2 + (x_j - w_j)^2)
//  2 complex           f = exp(i sum a_j x_j) prod (1 + b_j x_j)            BASELINE.json configs[2]
//  3 sector-like       f = prod x_j^nu_j * U(x)^a / F(x)^b                  BASELINE.json configs[3]
//    with the optional trailing block [lu, lf, p]: f * (lu log U + lf log F)^p, the shape of the order-eps^p term of
//    U^(a + lu eps) / F^(b - lf eps) that sector decomposition integrates (reading C-15)
//  4 Genz corner peak  f = (1 + sum c_j x_j)^-(d+1)             [c]
//  5 Genz Gaussian     f = exp(-sum c_j^2 (x_j - w_j)^2)        [c, w]
//  6 Genz C^0          f = exp(-sum c_j |x_j - w_j|)            [c, w]
//  7 Genz discontinuous f = 0 if x_1 > w_1 or x_2 > w_2, else exp(sum c_j x_j)   [c, w_1, w_2]
//  8 complex sector    f = prod x_j^nu_j * U(x)^a / F(x)^b with COMPLEX coefficients: the shape of a sector after the
//    contour deformation x_j -> x_j - i lambda_j x_j (1 - x_j) dF/dx_j that handles integrable singularities: every
//    factor of the deformed integrand (U, F, the Jacobian) is a polynomial in the real x with complex coefficients
//    (reading C-16).  Layout [a, b, nU, nF, nu_1..nu_d, Re cU (nU), Im cU (nU), eU (nU x d), Re cF (nF),
//    Im cF (nF), eF (nF x d)] and the optional trailing [lu, lf, p]: f * (lu Log U + lf Log F)^p with the principal
//    branch Log z = log |z| + i arg z, arg in (-pi, pi].
typedef std::complex<double> cplx;

inline cplx cpow_int(cplx b, int e) { cplx r(1.0, 0.0); for (int i = 0; i < e; ++i) r *= b; return r; }

// sum_t (cre_t + i cim_t) prod_j x_j^e_tj
inline cplx sparse_cpoly(const double* cre, const double* cim, const double* e, int cnt, int dim, const double* x) {
    cplx s(0.0, 0.0);
    for (int t = 0; t < cnt; ++t) {
        double mon = 1.0;
        for (int j = 0; j < dim; ++j) mon *= ipow(x[j], (int)e[t * dim + j]);
        s += cplx(cre[t], cim[t]) * mon;
    }
    return s;
}

inline void integrand(int fam, const double* p, int n_params, int dim, const double* x, double* re, double* im) {
    *im = 0.0;
    if (fam == FAM_CSECTOR) {
        int a = (int)p[0], b = (int)p[1], nU = (int)p[2], nF = (int)p[3];
        const double* nu = p + 4;
        const double* cUr = nu + dim; const double* cUi = cUr + nU; const double* eU = cUi + nU;
        const double* cFr = eU + (size_t)nU * dim; const double* cFi = cFr + nF; const double* eF = cFi + nF;
        double pre = 1.0;
        for (int j = 0; j < dim; ++j) pre *= ipow(x[j], (int)nu[j]);
        const cplx U = sparse_cpoly(cUr, cUi, eU, nU, dim, x), F = sparse_cpoly(cFr, cFi, eF, nF, dim, x);
        cplx f = pre * cpow_int(U, a) / cpow_int(F, b);
        if (n_params == 4 + dim + (nU + nF) * (2 + dim) + 3) {           // trailing [lu, lf, p], principal branch
            const double* t = p + n_params - 3;
            f *= cpow_int(t[0] * std::log(U) + t[1] * std::log(F), (int)t[2]);
        }
        *re = f.real(); *im = f.imag();
        return;
    }
    if (fam == FAM_OSC) {
        double ph = 2.0 * M_PI * p[0];
        for (int j = 0; j < dim; ++j) ph += p[1 + j] * x[j];
        *re = std::cos(ph);
    } else if (fam == FAM_PRODPEAK) {
        double f = 1.0;
        for (int j = 0; j < dim; ++j) { double t = x[j] - p[dim + j]; f *= 1.0 / (1.0 / (p[j] * p[j]) + t * t); }
        *re = f;
    } else if (fam == FAM_CEXP) {
        double ph = 0.0, pr = 1.0;
        for (int j = 0; j < dim; ++j) { ph += p[j] * x[j]; pr *= 1.0 + p[dim + j] * x[j]; }
        *re = std::cos(ph) * pr; *im = std::sin(ph) * pr;
    } else if (fam == FAM_CORNER) {
        double b = 1.0;
        for (int j = 0; j < dim; ++j) b += p[j] * x[j];
        *re = 1.0 / ipow(b, dim + 1);
    } else if (fam == FAM_GAUSS) {
        double e = 0.0;
        for (int j = 0; j < dim; ++j) { double t = x[j] - p[dim + j]; e += p[j] * p[j] * t * t; }
        *re = std::exp(-e);
    } else if (fam == FAM_C0) {
        double e = 0.0;
        for (int j = 0; j < dim; ++j) e += p[j] * std::fabs(x[j] - p[dim + j]);
        *re = std::exp(-e);
    } else if (fam == FAM_DISC) {
        bool zero = false;
        double e = 0.0;
        for (int j = 0; j < dim; ++j) { e += p[j] * x[j]; if (j < 2 && x[j] > p[dim + j]) zero = true; }
        *re = zero ? 0.0 : std::exp(e);
    } else {
        int a = (int)p[0], b = (int)p[1], nU = (int)p[2], nF = (int)p[3];
        const double* nu = p + 4;
        const double* cU = nu + dim; const double* eU = cU + nU;
        const double* cF = eU + (size_t)nU * dim; const double* eF = cF + nF;
        double pre = 1.0;
        for (int j = 0; j < dim; ++j) pre *= ipow(x[j], (int)nu[j]);
        double U = sparse_poly(cU, eU, nU, dim, x), F = sparse_poly(cF, eF, nF, dim, x);
        *re = pre * ipow(U, a) / ipow(F, b);
        if (n_params == 4 + dim + (nU + nF) * (1 + dim) + 3) {           // trailing [lu, lf, p]
            const double* t = p + n_params - 3;
            *re *= ipow(t[0] * std::log(U) + t[1] * std::log(F), (int)t[2]);
        }
    }
}

inline int ncomp_of(int fam) { return (fam == FAM_CEXP || fam == FAM_CSECTOR) ? 2 : 1; }

int expected_params(int fam, const double* p, int n_params, int dim) {
    if (fam == FAM_OSC) return 1 + dim;
    if (fam == FAM_PRODPEAK || fam == FAM_CEXP) return 2 * dim;
    if (fam == FAM_SECTOR) {
        int nU = (int)p[2], nF = (int)p[3], base = 4 + dim + (nU + nF) * (1 + dim);
        if (n_params == base + 3) {                                        // trailing [lu, lf, p], p a small positive integer
            const double pw = p[base + 2];
            return (pw >= 1.0 && pw <= 4.0 && pw == std::floor(pw)) ? n_params : -1;
        }
        return base;
    }
    if (fam == FAM_CSECTOR) {
        int nU = (int)p[2], nF = (int)p[3], base = 4 + dim + (nU + nF) * (2 + dim);
        if (n_params == base + 3) {
            const double pw = p[base + 2];
            return (pw >= 1.0 && pw <= 4.0 && pw == std::floor(pw)) ? n_params : -1;
        }
        return base;
    }
    if (fam == FAM_CORNER) return dim;
    if (fam == FAM_GAUSS || fam == FAM_C0) return 2 * dim;
    if (fam == FAM_DISC) return dim + (dim < 2 ? dim : 2);
    return -1;
}

// One lattice point for one shift: O2-O5.  Returns v = W * f (re, im).
inline void eval_point(int fam, const double* params, int n_params, int dim, const uint64_t* r, double inv_n, const double* shift,
                       const Transform& tr, const double* fit, double* re, double* im) {
    double x[MAX_DIM]; double W = 1.0;
    for (int j = 0; j < dim; ++j) {
        double u = coordinate(r[j], inv_n, shift[j]);
        double y, w; transform(tr, u, &y, &w);
        if (fit) { double xx, dp; fit_map(fit + 6 * j, y, &xx, &dp); y = xx; w *= dp; }
        x[j] = y; W *= w;
    }
    double fr, fi; integrand(fam, params, n_params, dim, x, &fr, &fi);
    *re = W * fr; *im = W * fi;
}

}  // namespace

extern "C" {

int oracle_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Residues and coordinates of lattice indices k0 .. k0+count-1 for one shift (O1, O2).
int oracle_lattice_points(uint64_t n, int dim, const uint64_t* z, const double* shift, uint64_t k0, uint64_t count,
                          uint64_t* out_r, double* out_u) {
    double inv_n = 1.0 / (double)n;
    for (uint64_t i = 0; i < count; ++i)
        for (int j = 0; j < dim; ++j) {
            uint64_t r = residue(k0 + i, z[j], n);
            if (out_r) out_r[i * dim + j] = r;
            if (out_u) out_u[i * dim + j] = coordinate(r, inv_n, shift[j]);
        }
    return 0;
}

// Per-coordinate transform (O3) exposed for the pins.
int oracle_transform(int tr, double u, double* y, double* w) {
    Transform t;
    if (!decode_transform(tr, &t)) return -7;
    transform(t, u, y, w);
    return 0;
}

int oracle_fit_map(const double* a, double y, double* x, double* dp) { fit_map(a, y, x, dp); return 0; }

int oracle_integrand(int fam, const double* params, int n_params, int dim, const double* x, double* out2) {
    if (fam < 0 || fam > FAM_LAST || dim < 1 || dim > MAX_DIM) return -8;
    if (expected_params(fam, params, n_params, dim) != n_params) return -9;
    integrand(fam, params, n_params, dim, x, &out2[0], &out2[1]);
    return 0;
}

// Raw sums S_s = sum_{k in [k_begin,k_end)} v_{k,s} (O1-O6 without the 1/n), ncomp per shift
// interleaved (re, im).  Compensated within 2^16-aligned chunks and across chunks in chunk order.
int oracle_shift_sums(int fam, const double* params, int n_params, int dim, uint64_t n, const uint64_t* z,
                      const double* shifts, int m, int tr, const double* fit, uint64_t k_begin, uint64_t k_end,
                      double* out_sums) {
    if (fam < 0 || fam > FAM_LAST) return -8;
    if (dim < 1 || dim > MAX_DIM) return -2;
    if (expected_params(fam, params, n_params, dim) != n_params) return -9;
    Transform trf;
    if (!decode_transform(tr, &trf)) return -7;
    if (k_end > n || k_begin > k_end) return -3;
    const int nc = ncomp_of(fam);
    const double inv_n = 1.0 / (double)n;
    const uint64_t c0 = k_begin / CHUNK, c1 = (k_end + CHUNK - 1) / CHUNK;
    const int64_t nchunks = (int64_t)(c1 - c0);
    std::vector<double> chunk_sums((size_t)(nchunks > 0 ? nchunks : 0) * m * nc);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t ci = 0; ci < nchunks; ++ci) {
        uint64_t ka = (c0 + ci) * CHUNK, kb = ka + CHUNK;
        if (ka < k_begin) ka = k_begin;
        if (kb > k_end) kb = k_end;
        std::vector<Comp> acc((size_t)m * nc);
        uint64_t r[MAX_DIM];
        for (uint64_t k = ka; k < kb; ++k) {
            for (int j = 0; j < dim; ++j) r[j] = residue(k, z[j], n);
            for (int s = 0; s < m; ++s) {
                double re, im;
                eval_point(fam, params, n_params, dim, r, inv_n, shifts + (size_t)s * dim, trf, fit, &re, &im);
                acc[(size_t)s * nc].add(re);
                if (nc == 2) acc[(size_t)s * nc + 1].add(im);
            }
        }
        for (int q = 0; q < m * nc; ++q) chunk_sums[(size_t)ci * m * nc + q] = acc[q].value();
    }
    for (int q = 0; q < m * nc; ++q) {
        Comp t;
        for (int64_t ci = 0; ci < nchunks; ++ci) t.add(chunk_sums[(size_t)ci * m * nc + q]);
        out_sums[q] = t.value();
    }
    return 0;
}

// O7, O8: Eq. 2 outer mean and Eq. 3, two-pass, per component.
int oracle_finalize(const double* shift_means, int m, int ncomp, double* out_mean, double* out_err) {
    if (m < 2) return -6;
    for (int c = 0; c < ncomp; ++c) {
        Comp t;
        for (int s = 0; s < m; ++s) t.add(shift_means[s * ncomp + c]);
        double mean = t.value() / (double)m;
        Comp v;
        for (int s = 0; s < m; ++s) { double d = shift_means[s * ncomp + c] - mean; v.add(d * d); }
        out_mean[c] = mean;
        out_err[c] = std::sqrt(v.value() / ((double)m * (double)(m - 1)));
    }
    return 0;
}

// Whole rule: per-shift means Q_s (O6), estimate and error (O7, O8).
int oracle_integrate(int fam, const double* params, int n_params, int dim, uint64_t n, const uint64_t* z,
                     const double* shifts, int m, int tr, const double* fit, double* out_shift_means,
                     double* out_mean, double* out_err) {
    const int nc = ncomp_of(fam);
    std::vector<double> sums((size_t)m * 2);
    int st = oracle_shift_sums(fam, params, n_params, dim, n, z, shifts, m, tr, fit, 0, n, sums.data());
    if (st) return st;
    std::vector<double> means((size_t)m * nc);
    for (int q = 0; q < m * nc; ++q) means[q] = sums[q] / (double)n;
    if (out_shift_means) std::memcpy(out_shift_means, means.data(), sizeof(double) * m * nc);
    return oracle_finalize(means.data(), m, nc, out_mean, out_err);
}

// O9 (reading C-8): transform None, weight 1, one shift; H[j][b] = sum_k |f(x_k)| [floor(B x_{k,j}) = b].
// |f| is the modulus for the complex family.  Compensated per bin, k increasing.
int oracle_project(int fam, const double* params, int n_params, int dim, uint64_t n, const uint64_t* z,
                   const double* shift, int bins, double* out_hist) {
    if (fam < 0 || fam > FAM_LAST) return -8;
    if (dim < 1 || dim > MAX_DIM) return -2;
    if (expected_params(fam, params, n_params, dim) != n_params) return -9;
    const double inv_n = 1.0 / (double)n;
    std::vector<Comp> H((size_t)dim * bins);
    double x[MAX_DIM];
    for (uint64_t k = 0; k < n; ++k) {
        for (int j = 0; j < dim; ++j) x[j] = coordinate(residue(k, z[j], n), inv_n, shift[j]);
        double re, im; integrand(fam, params, n_params, dim, x, &re, &im);
        double a = ncomp_of(fam) == 2 ? std::hypot(re, im) : std::fabs(re);
        for (int j = 0; j < dim; ++j) {
            int b = (int)std::floor((double)bins * x[j]);
            if (b >= bins) b = bins - 1;
            H[(size_t)j * bins + b].add(a);
        }
    }
    for (size_t q = 0; q < H.size(); ++q) out_hist[q] = H[q].value();
    return 0;
}

// O9b (the paper's own CDF sampling; reading C-8b): the integrand is sampled on the n points of one
// shifted lattice (transform None, weight 1); per dimension j the samples are sorted by x_j ("after sorting by value"), the
// running sum of |f| over the sorted samples divided by the total is the empirical CDF of Eq. 20 at the sorted coordinates, and
// every `step`-th sorted point is kept (fitstepsize, default 10): kept point t = 1..K, K = floor(n / step), is the sorted sample
// with 0-based rank t * step - 1.  out_x, out_cdf: [dim][K].  Equal coordinates keep their index order (stable sort).
int oracle_cdf_samples(int fam, const double* params, int n_params, int dim, uint64_t n, const uint64_t* z, const double* shift,
                       int step, double* out_x, double* out_cdf) {
    if (fam < 0 || fam > FAM_LAST) return -8;
    if (dim < 1 || dim > MAX_DIM) return -2;
    if (step < 1 || (uint64_t)step > n) return -3;
    if (expected_params(fam, params, n_params, dim) != n_params) return -9;
    const double inv_n = 1.0 / (double)n;
    const uint64_t K = n / (uint64_t)step;
    std::vector<double> xs((size_t)dim * n), v(n);
    double x[MAX_DIM];
    for (uint64_t k = 0; k < n; ++k) {
        for (int j = 0; j < dim; ++j) { x[j] = coordinate(residue(k, z[j], n), inv_n, shift[j]); xs[(size_t)j * n + k] = x[j]; }
        double re, im; integrand(fam, params, n_params, dim, x, &re, &im);
        v[k] = ncomp_of(fam) == 2 ? std::hypot(re, im) : std::fabs(re);
    }
    Comp tot; for (uint64_t k = 0; k < n; ++k) tot.add(v[k]);
    const double total = tot.value();
    std::vector<uint64_t> order(n);
    for (int j = 0; j < dim; ++j) {
        const double* xj = xs.data() + (size_t)j * n;
        for (uint64_t k = 0; k < n; ++k) order[k] = k;
        std::stable_sort(order.begin(), order.end(), [xj](uint64_t a, uint64_t b) { return xj[a] < xj[b]; });
        Comp run;
        uint64_t t = 0;
        for (uint64_t i = 0; i < n; ++i) {
            run.add(v[order[i]]);
            if ((i + 1) % (uint64_t)step == 0 && t < K) {
                out_x[(size_t)j * K + t] = xj[order[i]];
                out_cdf[(size_t)j * K + t] = run.value() / total;
                ++t;
            }
        }
    }
    return 0;
}

// Cubic fit of the inverse CDF from sampled pairs (c_t, x_t) (reading C-8b): minimise sum_t (p(c_t) - x_t)^2 over (a4, a5) with
// p(c) = c^3 + a4 (c - c^3) + a5 (c^2 - c^3); identity if min p' on [0,1] <= 0.05 or the system is singular.
int oracle_fit_cubic_cdf(const double* xs, const double* cdf, int dim, uint64_t count, double* fit_coeffs) {
    for (int j = 0; j < dim; ++j) {
        double A11 = 0, A12 = 0, A22 = 0, B1 = 0, B2 = 0;
        for (uint64_t t = 0; t < count; ++t) {
            const double c = cdf[(size_t)j * count + t], e = xs[(size_t)j * count + t];
            const double c3 = c * c * c, g1 = c - c3, g2 = c * c - c3, r = e - c3;
            A11 += g1 * g1; A12 += g1 * g2; A22 += g2 * g2; B1 += g1 * r; B2 += g2 * r;
        }
        double a4 = 1.0, a5 = 0.0;
        const double det = A11 * A22 - A12 * A12;
        if (std::fabs(det) > 1e-300) {
            const double c4 = (B1 * A22 - B2 * A12) / det, c5 = (A11 * B2 - A12 * B1) / det, c6 = 1.0 - c4 - c5;
            double mn = std::fmin(c4, c4 + 2.0 * c5 + 3.0 * c6);
            if (c6 != 0.0) { const double yv = -c5 / (3.0 * c6); if (yv > 0.0 && yv < 1.0) mn = std::fmin(mn, c4 + yv * (2.0 * c5 + 3.0 * c6 * yv)); }
            if (mn > 0.05) { a4 = c4; a5 = c5; }
        }
        double* o = fit_coeffs + 6 * j;
        o[0] = 1.001; o[1] = -0.001; o[2] = 0.0; o[3] = 0.0; o[4] = a4; o[5] = a5;
    }
    return 0;
}

// Cubic fit of the inverse CDF (reading C-8): with c_b the CDF at the bin edges e_b = b/B,
// minimise sum_{b=1}^{B-1} (c^3 + a4 (c - c^3) + a5 (c^2 - c^3) - e)^2 (2x2 normal equations);
// identity if min p' on [0,1] <= 0.05 or the system is singular.  Writes a0..a5 per dimension.
int oracle_fit_cubic(const double* hist, int dim, int bins, double* fit_coeffs) {
    for (int j = 0; j < dim; ++j) {
        const double* H = hist + (size_t)j * bins;
        Comp tot; for (int b = 0; b < bins; ++b) tot.add(H[b]);
        double total = tot.value();
        double a4 = 1.0, a5 = 0.0;
        if (total > 0.0) {
            double A11 = 0, A12 = 0, A22 = 0, B1 = 0, B2 = 0;
            Comp run;
            for (int b = 1; b < bins; ++b) {
                run.add(H[b - 1]);
                double c = run.value() / total, e = (double)b / (double)bins;
                double c3 = c * c * c, g1 = c - c3, g2 = c * c - c3, t = e - c3;
                A11 += g1 * g1; A12 += g1 * g2; A22 += g2 * g2; B1 += g1 * t; B2 += g2 * t;
            }
            double det = A11 * A22 - A12 * A12;
            if (std::fabs(det) > 1e-300) {
                double s4 = (B1 * A22 - B2 * A12) / det, s5 = (A11 * B2 - A12 * B1) / det;
                double a6 = 1.0 - s4 - s5;
                // min of p'(y) = s4 + 2 s5 y + 3 a6 y^2 on [0,1]
                double mn = std::fmin(s4, s4 + 2.0 * s5 + 3.0 * a6);
                if (a6 != 0.0) { double yv = -s5 / (3.0 * a6); if (yv > 0.0 && yv < 1.0) mn = std::fmin(mn, s4 + yv * (2.0 * s5 + 3.0 * a6 * yv)); }
                if (mn > 0.05) { a4 = s4; a5 = s5; }
            }
        }
        double* o = fit_coeffs + 6 * j;
        o[0] = 1.001; o[1] = -0.001; o[2] = 0.0; o[3] = 0.0; o[4] = a4; o[5] = a5;
    }
    return 0;
}

}  // extern "C"
