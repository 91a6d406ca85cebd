"""Seeded synthetic inputs shared by the tests, bench.py and the oracle checks.

This module holds NO arithmetic of the method (no lattice points, transforms, integrands or
reductions): it only draws parameters and shifts and loads committed generating vectors.  Both the
CUDA path and the CPU oracle receive exactly these arrays.

Recipe: std::mt19937_64-compatible generator (the paper's default engine,
PAPER.md L854, L881-L885; the sequence is fixed by the C++ standard), u = (x >> 11) * 2^-53 in
[0,1); draw order = family parameters in layout order, then the shifts row-major by shift
(shifts[s*dim + j], Eq. 2: Delta_k in [0,1)^d).  Seed of config c is 1811117200 + c;
sector p of config 3 uses 1811117300 + p.
"""
from __future__ import annotations

import json
import os

import numpy as np

FAMILY_GENZ_OSC, FAMILY_GENZ_PRODPEAK, FAMILY_CEXP_POLY, FAMILY_SECTOR = 0, 1, 2, 3
FAMILY_GENZ_CORNER, FAMILY_GENZ_GAUSSIAN, FAMILY_GENZ_C0, FAMILY_GENZ_DISCONT = 4, 5, 6, 7
# integrand difficulties ||c||_1 of the paper's Genz protocol, families 1..6
GENZ_DIFFICULTY = {FAMILY_GENZ_OSC: 6.0, FAMILY_GENZ_PRODPEAK: 18.0, FAMILY_GENZ_CORNER: 2.2, FAMILY_GENZ_GAUSSIAN: 15.2,
                   FAMILY_GENZ_C0: 16.1, FAMILY_GENZ_DISCONT: 16.4}
TRANSFORM_NONE, TRANSFORM_BAKER, TRANSFORM_KOROBOV = 0, 1, 100      # Korobov weight r = 100 + r
TRANSFORM_SIDI = 200                                                # Sidi weight r = 200 + r
TRANSFORM_KOROBOV_ASYM = 1000                                       # Korobov weights (r0, r1) = 1000 + 16 r0 + r1

_DATA = os.path.join(os.path.dirname(os.path.abspath(__file__)), "data", "genvecs.json")


class MT19937_64:
    """The 64-bit Mersenne Twister of the C++ standard library (std::mt19937_64)."""
    _N, _M = 312, 156
    _A = 0xB5026F5AA96619E9
    _MASK = (1 << 64) - 1

    def __init__(self, seed: int = 5489):
        mt = [0] * self._N
        mt[0] = seed & self._MASK
        for i in range(1, self._N):
            mt[i] = (6364136223846793005 * (mt[i - 1] ^ (mt[i - 1] >> 62)) + i) & self._MASK
        self.mt, self.idx = mt, self._N

    def _twist(self):
        mt, N, M = self.mt, self._N, self._M
        for i in range(N):
            x = (mt[i] & 0xFFFFFFFF80000000) | (mt[(i + 1) % N] & 0x7FFFFFFF)
            xa = x >> 1
            if x & 1:
                xa ^= self._A
            mt[i] = mt[(i + M) % N] ^ xa
        self.idx = 0

    def next_u64(self) -> int:
        if self.idx >= self._N:
            self._twist()
        x = self.mt[self.idx]
        self.idx += 1
        x ^= (x >> 29) & 0x5555555555555555
        x ^= (x << 17) & 0x71D67FFFEDA60000
        x ^= (x << 37) & 0xFFF7EEE000000000
        x ^= x >> 43
        return x & self._MASK

    def uniform(self) -> float:
        """53-bit uniform in [0,1)."""
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)

    def uniform_range(self, lo: float, hi: float) -> float:
        return lo + (hi - lo) * self.uniform()


def genvec(n: int, d: int):
    """Committed CBC generating vector for (n, d) (paper_1811_11720_b200/cbc.py wrote it)."""
    with open(_DATA) as f:
        table = json.load(f)
    key = f"{n}:{d}"
    if key not in table:
        raise KeyError(f"no committed generating vector for n={n}, d={d}")
    return np.array(table[key]["z"], dtype=np.uint64)


def ladder(d: int, n_max: int, n_min: int = 1021):
    """The committed lattice ladder for dimension d: largest primes below 2^10, 2^12, ... plus the configs' own sizes, with
    their CBC vectors (ascending n, n_min <= n <= n_max) -> (ladder_n (L,), ladder_z (L, d)).  Stand-in for the paper's
    generating-vector tables (PAPER.md, Table A.1), which are not available."""
    with open(_DATA) as f:
        table = json.load(f)
    ns = sorted(v["n"] for v in table.values() if v["d"] == d and n_min <= v["n"] <= n_max)
    return (np.array(ns, dtype=np.uint64), np.array([table[f"{n}:{d}"]["z"] for n in ns], dtype=np.uint64).reshape(len(ns), d))


def korobov_form_vector(n: int, d: int, a: int):
    """z = (1, a, a^2, ...) mod n: any valid z exercises the same code path (used by tests)."""
    z, cur = [], 1
    for _ in range(d):
        z.append(cur)
        cur = cur * a % n
    return np.array(z, dtype=np.uint64)


def draw_shifts(rng: MT19937_64, m: int, d: int):
    return np.array([rng.uniform() for _ in range(m * d)], dtype=np.float64).reshape(m, d)


def genz_osc(rng, d, a_hi=1.0):
    u0 = rng.uniform()
    a = [rng.uniform_range(0.0, a_hi) for _ in range(d)]
    return np.array([u0] + a, dtype=np.float64)


def genz_prodpeak(rng, d):
    c = [rng.uniform_range(1.0, 5.0) for _ in range(d)]
    w = [rng.uniform() for _ in range(d)]
    return np.array(c + w, dtype=np.float64)


def genz_protocol(rng, family, d):
    """Parameters of one Genz test integral as in the paper's protocol: w_i ~ U[0,1), c_i > 0 random and
    rescaled to the family's difficulty ||c||_1; packed in the family's layout (include/qmc_lattice.h)."""
    c = np.array([rng.uniform() + 1e-3 for _ in range(d)])
    c *= GENZ_DIFFICULTY[family] / c.sum()
    w = np.array([rng.uniform() for _ in range(d)])
    if family == FAMILY_GENZ_OSC:
        return np.concatenate([[w[0]], c])
    if family == FAMILY_GENZ_CORNER:
        return c.copy()
    if family == FAMILY_GENZ_DISCONT:
        return np.concatenate([c, w[:min(d, 2)]])
    return np.concatenate([c, w])


def cexp_poly(rng, d):
    a = [rng.uniform_range(-3.0, 3.0) for _ in range(d)]
    b = [rng.uniform() for _ in range(d)]
    return np.array(a + b, dtype=np.float64)


def sector(rng, d, deg_u=2, deg_f=3, n_lo=6, n_span=15):
    """Sector-like integrand parameters, layout
    [a, b, nU, nF, nu_1..nu_d, cU_1..cU_nU, eU_{1,1}..eU_{nU,d}, cF_1..cF_nF, eF_{1,1}..eF_{nF,d}].
    Every polynomial has the constant monomial first with a coefficient in [0.5, 2)."""
    nU = n_lo + rng.next_u64() % n_span
    nF = n_lo + rng.next_u64() % n_span
    a = 1 + rng.next_u64() % 2
    b = 2 + rng.next_u64() % 2
    nu = [rng.next_u64() % 2 for _ in range(d)]

    def poly(count, deg):
        # cap the monomial count by the number of distinct monomials of degree <= deg in d variables
        from math import comb
        count = min(count, comb(d + deg, deg))
        coeffs, exps, seen = [rng.uniform_range(0.5, 2.0)], [tuple([0] * d)], {tuple([0] * d)}
        while len(exps) < count:
            t = 1 + rng.next_u64() % deg
            e = [0] * d
            for _ in range(t):
                e[rng.next_u64() % d] += 1
            e = tuple(e)
            if e in seen:
                continue
            seen.add(e)
            exps.append(e)
            coeffs.append(rng.uniform_range(0.1, 2.0))
        return coeffs, exps

    cU, eU = poly(nU, deg_u)
    cF, eF = poly(nF, deg_f)
    out = [float(a), float(b), float(len(cU)), float(len(cF))] + [float(v) for v in nu]
    out += cU + [float(v) for e in eU for v in e]
    out += cF + [float(v) for e in eF for v in e]
    return np.array(out, dtype=np.float64)


def sector_log(rng, d, **kw):
    """Sector-like integrand with the trailing block [lu, lf, p]: f * (lu log U + lf log F)^p, the shape of the
    order-eps^p term of U^(a + lu eps) / F^(b - lf eps).  lu in [0.5, 2), lf in [-3, -1), p in 1..3."""
    prm = sector(rng, d, **kw)
    lu = rng.uniform_range(0.5, 2.0)
    lf = rng.uniform_range(-3.0, -1.0)
    pw = 1 + rng.next_u64() % 3
    return np.concatenate([prm, np.array([lu, lf, float(pw)])])


FAMILY_SECTOR_COMPLEX = 8


def sector_complex(rng, d, lam=0.5, log_block=False, **kw):
    """Complex sector integrand (family 8): the shape of a sector after contour deformation -- polynomials in the real x with
    complex coefficients (reading C-16).  The real sector recipe gives exponents and real parts; then, in layout
    order, Im cU_t = Re cU_t * U[-lam, lam) and Im cF_t = -Re cF_t * U[0.1 lam, lam): Im F < 0 on the whole cube (the
    Feynman prescription F - i delta after deformation), so F has no zero.  Layout
    [a, b, nU, nF, nu_j, Re cU, Im cU, eU, Re cF, Im cF, eF] (+ [lu, lf, p])."""
    prm = sector(rng, d, **kw)
    nU, nF = int(prm[2]), int(prm[3])
    off = 4 + d
    cU, eU = prm[off:off + nU], prm[off + nU:off + nU + nU * d]
    off += nU * (1 + d)
    cF, eF = prm[off:off + nF], prm[off + nF:off + nF + nF * d]
    iU = np.array([c * rng.uniform_range(-lam, lam) for c in cU])
    iF = np.array([-c * rng.uniform_range(0.1 * lam, lam) for c in cF])
    out = np.concatenate([prm[:4 + d], cU, iU, eU, cF, iF, eF])
    if log_block:
        out = np.concatenate([out, [rng.uniform_range(0.5, 2.0), rng.uniform_range(-3.0, -1.0), float(1 + rng.next_u64() % 3)]])
    return out


def problem(family, params, n, z, shifts, transform, fit_coeffs=None, name=""):
    shifts = np.ascontiguousarray(shifts, dtype=np.float64)
    return {"name": name, "family": int(family), "params": np.ascontiguousarray(params, dtype=np.float64),
            "dim": int(shifts.shape[1]), "n": int(n), "z": np.ascontiguousarray(z, dtype=np.uint64),
            "shifts": shifts, "m": int(shifts.shape[0]), "transform": int(transform),
            "fit_coeffs": None if fit_coeffs is None else np.ascontiguousarray(fit_coeffs, dtype=np.float64)}


CONFIG_SEED = 1811117200
SECTOR_SEED = 1811117300
CONFIG_SHAPES = {  # (d, n, m) of BASELINE.json configs[0..4]
    0: (4, 65537, 10), 1: (8, 1048573, 32), 2: (12, 16777213, 32), 3: (6, 4194301, 16),
    4: (16, 1073741789, 20)}
CONFIG4_NFIT = 1048573       # lattice of the projection pass of config 4
PROJECTION_BINS = 256


def config(c: int, n_override=None, count_override=None):
    """The list of problems of BASELINE.json configs[c] (one problem, or 256 for c = 3).
    n_override substitutes a smaller lattice (with a Korobov-form vector unless a committed CBC
    vector exists) so that parity tests can run the same parameters at oracle-friendly sizes."""
    d, n, m = CONFIG_SHAPES[c]
    if n_override is not None:
        n = int(n_override)

    def vec():
        try:
            return genvec(n, d)
        except KeyError:
            return korobov_form_vector(n, d, 1 + (n // 3))

    if c == 3:
        count = 256 if count_override is None else count_override
        z = vec()
        out = []
        for p in range(count):
            rng = MT19937_64(SECTOR_SEED + p)
            prm = sector(rng, d)
            sh = draw_shifts(rng, m, d)
            out.append(problem(FAMILY_SECTOR, prm, n, z, sh, TRANSFORM_KOROBOV + 3, name=f"cfg3.sector{p}"))
        return out
    rng = MT19937_64(CONFIG_SEED + c)
    if c == 0:
        prm, fam, tr = genz_osc(rng, d), FAMILY_GENZ_OSC, TRANSFORM_KOROBOV + 3
    elif c == 1:
        prm, fam, tr = genz_prodpeak(rng, d), FAMILY_GENZ_PRODPEAK, TRANSFORM_BAKER
    elif c == 2:
        prm, fam, tr = cexp_poly(rng, d), FAMILY_CEXP_POLY, TRANSFORM_KOROBOV + 3
    elif c == 4:
        prm, fam, tr = genz_osc(rng, d, a_hi=0.5), FAMILY_GENZ_OSC, TRANSFORM_KOROBOV + 3
    else:
        raise ValueError(c)
    sh = draw_shifts(rng, m, d)
    return [problem(fam, prm, n, vec(), sh, tr, name=f"cfg{c}")]


def cubic_fit_coeffs(d, a4=0.6, a5=0.3):
    """fit_coeffs[j*6 + i] = a_i of PAPER.md Eq. 19 for dimension j; the cubic sub-family has
    a2 = a3 = 0 (a0, a1 then unused; set to the bounds of PAPER.md L231)."""
    row = [1.001, -0.001, 0.0, 0.0, a4, a5]
    return np.array(row * d, dtype=np.float64).reshape(d, 6)
