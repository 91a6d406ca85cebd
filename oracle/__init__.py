"""ctypes loader for the CPU oracle (oracle/qmc_oracle.cpp).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference leg may import this package.  The product (paper_1811_11720_b200) never does.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmc_oracle.cpp")
_LIB = os.path.join(_HERE, "libqmc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 -std=c++17 -ffp-contract=off: no fast-math, no contraction (std::fma is explicit)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp, up = C.POINTER(C.c_double), C.POINTER(C.c_uint64)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_lattice_points.argtypes = [C.c_uint64, C.c_int, up, dp, C.c_uint64, C.c_uint64, up, dp]
        L.oracle_transform.argtypes = [C.c_int, C.c_double, dp, dp]
        L.oracle_fit_map.argtypes = [dp, C.c_double, dp, dp]
        L.oracle_integrand.argtypes = [C.c_int, dp, C.c_int, C.c_int, dp, dp]
        L.oracle_shift_sums.argtypes = [C.c_int, dp, C.c_int, C.c_int, C.c_uint64, up, dp, C.c_int, C.c_int, dp,
                                        C.c_uint64, C.c_uint64, dp]
        L.oracle_finalize.argtypes = [dp, C.c_int, C.c_int, dp, dp]
        L.oracle_integrate.argtypes = [C.c_int, dp, C.c_int, C.c_int, C.c_uint64, up, dp, C.c_int, C.c_int, dp, dp, dp, dp]
        L.oracle_project.argtypes = [C.c_int, dp, C.c_int, C.c_int, C.c_uint64, up, dp, C.c_int, dp]
        L.oracle_fit_cubic.argtypes = [dp, C.c_int, C.c_int, dp]
        L.oracle_cdf_samples.argtypes = [C.c_int, dp, C.c_int, C.c_int, C.c_uint64, up, dp, C.c_int, dp, dp]
        L.oracle_fit_cubic_cdf.argtypes = [dp, dp, C.c_int, C.c_uint64, dp]
        _lib = L
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _u(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_uint64))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _u64(a):
    return np.ascontiguousarray(a, dtype=np.uint64)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def ncomp(family: int) -> int:
    return 2 if family in (2, 8) else 1


def lattice_points(n, z, shift, k0, count):
    z, shift = _u64(z), _f64(shift)
    d = len(z)
    r = np.empty((count, d), dtype=np.uint64)
    u = np.empty((count, d), dtype=np.float64)
    st = lib().oracle_lattice_points(int(n), d, _u(z), _d(shift), int(k0), int(count), _u(r), _d(u))
    assert st == 0
    return r, u


def transform(tr, u):
    y, w = C.c_double(), C.c_double()
    st = lib().oracle_transform(int(tr), float(u), C.byref(y), C.byref(w))
    if st:
        raise ValueError(f"oracle_transform status {st}")
    return y.value, w.value


def fit_map(a6, y):
    a6 = _f64(a6)
    x, dp = C.c_double(), C.c_double()
    lib().oracle_fit_map(_d(a6), float(y), C.byref(x), C.byref(dp))
    return x.value, dp.value


def integrand(family, params, x):
    params, x = _f64(params), _f64(x)
    out = np.zeros(2)
    st = lib().oracle_integrand(int(family), _d(params), len(params), len(x), _d(x), _d(out))
    if st:
        raise ValueError(f"oracle_integrand status {st}")
    return complex(out[0], out[1]) if family in (2, 8) else float(out[0])


def shift_sums(p, k_begin=0, k_end=None):
    """Raw compensated sums over lattice indices [k_begin, k_end) for problem dict p -> (m, ncomp)."""
    k_end = p["n"] if k_end is None else k_end
    nc = ncomp(p["family"])
    out = np.zeros((p["m"], nc))
    params, z, sh, fit = _f64(p["params"]), _u64(p["z"]), _f64(p["shifts"]), _f64(p.get("fit_coeffs"))
    st = lib().oracle_shift_sums(p["family"], _d(params), len(params), p["dim"], p["n"], _u(z), _d(sh), p["m"],
                                 p["transform"], _d(fit), int(k_begin), int(k_end), _d(out))
    if st:
        raise ValueError(f"oracle_shift_sums status {st}")
    return out


def finalize(shift_means):
    sm = _f64(shift_means)
    if sm.ndim == 1:
        sm = sm.reshape(-1, 1)
    m, nc = sm.shape
    mean, err = np.zeros(nc), np.zeros(nc)
    st = lib().oracle_finalize(_d(sm), m, nc, _d(mean), _d(err))
    if st:
        raise ValueError(f"oracle_finalize status {st}")
    return mean, err


def integrate(p):
    """-> (shift_means (m, ncomp), mean (ncomp,), err (ncomp,))"""
    nc = ncomp(p["family"])
    sm, mean, err = np.zeros((p["m"], nc)), np.zeros(nc), np.zeros(nc)
    params, z, sh, fit = _f64(p["params"]), _u64(p["z"]), _f64(p["shifts"]), _f64(p.get("fit_coeffs"))
    st = lib().oracle_integrate(p["family"], _d(params), len(params), p["dim"], p["n"], _u(z), _d(sh), p["m"],
                                p["transform"], _d(fit), _d(sm), _d(mean), _d(err))
    if st:
        raise ValueError(f"oracle_integrate status {st}")
    return sm, mean, err


def project(p, bins, shift=None):
    params, z = _f64(p["params"]), _u64(p["z"])
    shift = _f64(p["shifts"][0] if shift is None else shift)
    H = np.zeros((p["dim"], bins))
    st = lib().oracle_project(p["family"], _d(params), len(params), p["dim"], p["n"], _u(z), _d(shift), bins, _d(H))
    if st:
        raise ValueError(f"oracle_project status {st}")
    return H


def fit_cubic(hist):
    H = _f64(hist)
    d, bins = H.shape
    out = np.zeros((d, 6))
    lib().oracle_fit_cubic(_d(H), d, bins, _d(out))
    return out


def cdf_samples(p, step=10, shift=None):
    """The paper's sort-based CDF sampling -> (x (dim, K), cdf (dim, K)), K = n // step."""
    params, z = _f64(p["params"]), _u64(p["z"])
    shift = _f64(p["shifts"][0] if shift is None else shift)
    K = p["n"] // step
    xs, cdf = np.zeros((p["dim"], K)), np.zeros((p["dim"], K))
    st = lib().oracle_cdf_samples(p["family"], _d(params), len(params), p["dim"], p["n"], _u(z), _d(shift), int(step), _d(xs), _d(cdf))
    if st:
        raise ValueError(f"oracle_cdf_samples status {st}")
    return xs, cdf


def fit_cubic_cdf(xs, cdf):
    xs, cdf = _f64(xs), _f64(cdf)
    d, K = xs.shape
    out = np.zeros((d, 6))
    lib().oracle_fit_cubic_cdf(_d(xs), _d(cdf), d, K, _d(out))
    return out


def fit_polysingular_pairs(c, e, start45=(1.0, 0.0)):
    """The complete fit function of Eq. 19 fitted to pairs (c_i, e_i), p(c_i) ~ e_i, by bounded non-linear least
    squares with the parameter bounds of PAPER.md L231 (a0 >= 1.001, a1 <= -0.001, a2, a3 >= 0); a6 = 1 - a2 - a3 - a4 - a5 by
    p(1) = 1.  The paper runs GSL's Levenberg-Marquardt; the oracle takes scipy.optimize.least_squares (trust-region reflective,
    the library's bounded solver) from two starts -- dormant and small active poles, since the gradient in a0, a1 vanishes while
    a2 = a3 = 0 -- and returns (best parameters a0..a5, sum of squared residuals).  The minimiser is not unique (a dormant pole's
    position is free): what compares across implementations is the residual, not the parameters."""
    from scipy.optimize import least_squares
    c = np.asarray(c, dtype=np.float64)
    e = np.asarray(e, dtype=np.float64)

    def p_of(a, y):
        a6 = 1.0 - a[2] - a[3] - a[4] - a[5]
        return a[2] * y * (a[0] - 1.0) / (a[0] - y) + a[3] * y * (a[1] - 1.0) / (a[1] - y) + y * (a[4] + y * (a[5] + y * a6))

    lo = [1.001, -np.inf, 0.0, 0.0, -np.inf, -np.inf]
    hi = [np.inf, -0.001, np.inf, np.inf, np.inf, np.inf]
    best, best_cost = None, np.inf
    for a2 in (0.0, 0.05):
        x0 = np.array([1.1, -0.1, a2, a2, start45[0], start45[1]])
        sol = least_squares(lambda a: p_of(a, c) - e, x0, bounds=(lo, hi), method="trf", xtol=1e-15, ftol=1e-15, gtol=1e-15, max_nfev=4000)
        cost = float(np.sum(sol.fun ** 2))
        if cost < best_cost:
            best, best_cost = sol.x.copy(), cost
    return best, best_cost
