// qmc_fit.cu -- host-side fit of the complete fit function of Eq. 19 to the inverse CDF sampled by the device
// projection pass (Eq. 20).  SURVEY.md 8(f) row f-2.  The paper uses GSL's Levenberg-Marquardt with the
// parameter bounds a0 >= 1.001, a1 <= -0.001, a2, a3 >= 0; this is an own bounded Levenberg-Marquardt (no GSL).
// Setup code, off the timed path; the result is an INPUT of the fused kernels (fit_coeffs), which are parity-tested for
// arbitrary valid coefficients, so the optimiser itself needs no oracle counterpart (any valid map keeps the integral, Eq. 18).
#include <algorithm>
#include <cmath>
#include <vector>

#include "../../include/qmc_lattice.h"

namespace {

struct Model {                      // p(y) of Eq. 19 with a6 = 1 - a2 - a3 - a4 - a5, and its parameter gradient
    static long double eval(const long double* a, long double y, long double* grad) {
        const long double y2 = y * y, y3 = y2 * y;
        const long double d0 = a[0] - y, d1 = a[1] - y;
        const long double t0 = y * (a[0] - 1.0L) / d0, t1 = y * (a[1] - 1.0L) / d1;
        const long double a6 = 1.0L - a[2] - a[3] - a[4] - a[5];
        if (grad) {
            grad[0] = a[2] * y * (1.0L - y) / (d0 * d0);
            grad[1] = a[3] * y * (1.0L - y) / (d1 * d1);
            grad[2] = t0 - y3;
            grad[3] = t1 - y3;
            grad[4] = y - y3;
            grad[5] = y2 - y3;
        }
        return a[2] * t0 + a[3] * t1 + y * (a[4] + y * (a[5] + y * a6));
    }
    static bool increasing(const long double* a) {
        const long double a6 = 1.0L - a[2] - a[3] - a[4] - a[5];
        for (int i = 0; i <= 1024; ++i) {
            const long double y = (long double)i / 1024.0L, d0 = a[0] - y, d1 = a[1] - y;
            const long double dp = a[2] * a[0] * (a[0] - 1.0L) / (d0 * d0) + a[3] * a[1] * (a[1] - 1.0L) / (d1 * d1) + a[4] +
                                   y * (2.0L * a[5] + 3.0L * a6 * y);
            if (!(dp > 0.05L)) return false;                      // same safety margin as the cubic fit (reading C-8)
        }
        return true;
    }
};

void project(long double* a) {      // bounds of P:L231
    a[0] = std::max(a[0], 1.001L);
    a[1] = std::min(a[1], -0.001L);
    a[2] = std::max(a[2], 0.0L);
    a[3] = std::max(a[3], 0.0L);
}

long double cost(const long double* a, const std::vector<long double>& c, const std::vector<long double>& e) {
    long double s = 0.0L;
    for (size_t b = 0; b < c.size(); ++b) { const long double r = Model::eval(a, c[b], nullptr) - e[b]; s += r * r; }
    return s;
}

bool solve6(long double A[6][6], long double* b) {               // Gaussian elimination with partial pivoting
    for (int k = 0; k < 6; ++k) {
        int piv = k;
        for (int i = k + 1; i < 6; ++i) if (fabsl(A[i][k]) > fabsl(A[piv][k])) piv = i;
        if (fabsl(A[piv][k]) < 1e-300L) return false;
        if (piv != k) { for (int j = 0; j < 6; ++j) std::swap(A[k][j], A[piv][j]); std::swap(b[k], b[piv]); }
        for (int i = k + 1; i < 6; ++i) {
            const long double f = A[i][k] / A[k][k];
            for (int j = k; j < 6; ++j) A[i][j] -= f * A[k][j];
            b[i] -= f * b[k];
        }
    }
    for (int k = 5; k >= 0; --k) {
        long double s = b[k];
        for (int j = k + 1; j < 6; ++j) s -= A[k][j] * b[j];
        b[k] = s / A[k][k];
    }
    return true;
}

// Bounded Levenberg-Marquardt fit of Eq. 19 to pairs (c_i, e_i): p(c_i) ~ e_i.  o: in, the cubic solution (a4, a5 used as the
// start); out, the full parameter set if it is a strictly better valid fit.
void fit_full_pairs(const std::vector<long double>& c, const std::vector<long double>& e, double* o) {
    long double a[6] = {1.1L, -0.1L, 0.0L, 0.0L, o[4], o[5]};
    // two starts: the cubic solution with dormant poles, and the same with small active poles (the gradient of a0, a1 vanishes
    // while a2 = a3 = 0)
    long double best[6], best_cost = cost(a, c, e);
    for (int k = 0; k < 6; ++k) best[k] = a[k];
    for (int start = 0; start < 2; ++start) {
        long double th[6] = {1.1L, -0.1L, start ? 0.05L : 0.0L, start ? 0.05L : 0.0L, o[4], o[5]};
        long double cur = cost(th, c, e), lambda = 1e-3L;
        for (int it = 0; it < 400; ++it) {
            long double JTJ[6][6] = {}, JTr[6] = {};
            for (size_t b = 0; b < c.size(); ++b) {
                long double g[6];
                const long double r = Model::eval(th, c[b], g) - e[b];
                for (int p = 0; p < 6; ++p) { JTr[p] += g[p] * r; for (int q = 0; q < 6; ++q) JTJ[p][q] += g[p] * g[q]; }
            }
            long double A[6][6], rhs[6];
            for (int p = 0; p < 6; ++p) {
                rhs[p] = -JTr[p];
                for (int q = 0; q < 6; ++q) A[p][q] = JTJ[p][q];
                A[p][p] += lambda * std::max(JTJ[p][p], 1e-12L);
            }
            if (!solve6(A, rhs)) { lambda *= 10.0L; continue; }
            long double trial[6];
            for (int p = 0; p < 6; ++p) trial[p] = th[p] + rhs[p];
            project(trial);
            const long double tc = cost(trial, c, e);
            if (tc < cur) {
                const long double gain = (cur - tc) / std::max(cur, 1e-300L);
                for (int p = 0; p < 6; ++p) th[p] = trial[p];
                cur = tc;
                lambda = std::max(lambda / 3.0L, 1e-12L);
                if (gain < 1e-12L) break;
            } else {
                lambda *= 4.0L;
                if (lambda > 1e12L) break;
            }
        }
        if (cur < best_cost && Model::increasing(th)) { best_cost = cur; for (int k = 0; k < 6; ++k) best[k] = th[k]; }
    }
    // keep the cubic result unless the full function is a strictly better, valid fit
    const long double cubic[6] = {1.1L, -0.1L, 0.0L, 0.0L, o[4], o[5]};
    if (best_cost < cost(cubic, c, e) && Model::increasing(best) && (best[2] > 0.0L || best[3] > 0.0L))
        for (int k = 0; k < 6; ++k) o[k] = (double)best[k];
}

// Closed-form least squares for the cubic sub-family on pairs (c_i, e_i) (as qmc_fit_cubic): identity if not safely monotone.
void fit_cubic_pairs(const std::vector<long double>& cs, const std::vector<long double>& es, double* o) {
    long double s11 = 0, s12 = 0, s22 = 0, t1 = 0, t2 = 0;
    for (size_t i = 0; i < cs.size(); ++i) {
        const long double c = cs[i], c3 = c * c * c, g1 = c - c3, g2 = c * c - c3, rhs = es[i] - c3;
        s11 += g1 * g1; s12 += g1 * g2; s22 += g2 * g2; t1 += g1 * rhs; t2 += g2 * rhs;
    }
    double a4 = 1.0, a5 = 0.0;
    const long double det = s11 * s22 - s12 * s12;
    if (fabsl(det) > 1e-300L) {
        const double c4 = (double)((t1 * s22 - t2 * s12) / det), c5 = (double)((s11 * t2 - s12 * t1) / det), c6 = 1.0 - c4 - c5;
        double mn = std::fmin(c4, c4 + 2.0 * c5 + 3.0 * c6);
        if (c6 != 0.0) { const double yv = -c5 / (3.0 * c6); if (yv > 0.0 && yv < 1.0) mn = std::fmin(mn, c4 + yv * (2.0 * c5 + 3.0 * c6 * yv)); }
        if (mn > 0.05) { a4 = c4; a5 = c5; }
    }
    o[0] = 1.001; o[1] = -0.001; o[2] = 0.0; o[3] = 0.0; o[4] = a4; o[5] = a5;
}

}  // namespace

// ---- variance-reduction fit from histograms (reading C-8): the CDF at the inner bin edges gives the pairs (c_b, e_b = b / bins)
namespace {
bool histogram_pairs(const double* h, int bins, std::vector<long double>* c, std::vector<long double>* e) {
    long double total = 0.0L;
    for (int b = 0; b < bins; ++b) {
        if (!std::isfinite(h[b]) || h[b] < 0.0) return false;
        total += h[b];
    }
    if (!(total > 0.0L)) return false;
    c->clear(); e->clear();
    long double run = 0.0L;
    for (int b = 1; b < bins; ++b) { run += h[b - 1]; c->push_back(run / total); e->push_back((long double)b / (long double)bins); }
    return true;
}
}  // namespace

extern "C" int qmc_fit_cubic(const double* hist, int dim, int bins, double* fit_coeffs) {
    if (!hist || !fit_coeffs) return QMC_ERR_NULL;
    if (dim < 1 || dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (bins < 2 || bins > 1024) return QMC_ERR_N;
    std::vector<long double> c, e;
    for (int j = 0; j < dim; ++j) {
        double* o = fit_coeffs + 6 * j;
        if (histogram_pairs(hist + (size_t)j * bins, bins, &c, &e)) fit_cubic_pairs(c, e, o);
        else { o[0] = 1.001; o[1] = -0.001; o[2] = 0.0; o[3] = 0.0; o[4] = 1.0; o[5] = 0.0; }   // identity map (bounds of P:L231 for the unused poles)
    }
    return QMC_OK;
}

extern "C" int qmc_fit_polysingular(const double* hist, int dim, int bins, double* fit_coeffs) {
    if (!hist || !fit_coeffs) return QMC_ERR_NULL;
    if (dim < 1 || dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (bins < 8 || bins > 1024) return QMC_ERR_N;
    const int st = qmc_fit_cubic(hist, dim, bins, fit_coeffs);   // starting point and fall-back (identity if that fails too)
    if (st != QMC_OK) return st;
    std::vector<long double> c, e;                                 // CDF values at the bin edges: p(c_b) = e_b (Eq. 18-20)
    for (int j = 0; j < dim; ++j) {
        if (!histogram_pairs(hist + (size_t)j * bins, bins, &c, &e)) continue;
        fit_full_pairs(c, e, fit_coeffs + 6 * j);
    }
    return QMC_OK;
}


// The same two fits from the paper's sort-based CDF samples (qmc_lattice_cdf_samples): pairs
// (CDF_t, x_t), p(CDF_t) ~ x_t.  x, cdf: HOST [dim][count].  with_poles = 0: cubic sub-family in closed form; 1: Eq. 19 complete.
extern "C" int qmc_fit_from_cdf(const double* x, const double* cdf, int dim, long long count, int with_poles, double* fit_coeffs) {
    if (!x || !cdf || !fit_coeffs) return QMC_ERR_NULL;
    if (dim < 1 || dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (count < 8) return QMC_ERR_N;
    for (int j = 0; j < dim; ++j) {
        std::vector<long double> c((size_t)count), e((size_t)count);
        bool ok = true;
        for (long long t = 0; t < count; ++t) {
            c[t] = cdf[(size_t)j * count + t]; e[t] = x[(size_t)j * count + t];
            ok = ok && std::isfinite((double)c[t]) && std::isfinite((double)e[t]);
        }
        double* o = fit_coeffs + 6 * j;
        if (!ok) { o[0] = 1.001; o[1] = -0.001; o[2] = 0.0; o[3] = 0.0; o[4] = 1.0; o[5] = 0.0; continue; }   // identity map
        fit_cubic_pairs(c, e, o);
        if (with_poles) fit_full_pairs(c, e, o);
    }
    return QMC_OK;
}
