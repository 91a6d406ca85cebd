"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU needed).

Every check compares oracle/ with something that is NOT the oracle: values written out by hand from
the paper's tiny lattices, exact rational arithmetic, library special functions (scipy betainc,
quad, leggauss), closed-form integrals, brute-force tensor quadrature.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.integrate
import scipy.special

import oracle
from paper_1811_11720_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")
K3 = synth.TRANSFORM_KOROBOV + 3


# ------------------------------------------------------------------ residues (O1, Eq. 2)
def test_residues_paper_lattices():
    for line in open(os.path.join(GOLD, "lattice_small.txt")):
        if line.startswith("#") or not line.strip():
            continue
        head, vals = line.split(":")
        n, z2 = (int(v) for v in head.split())
        want = np.array([int(v) for v in vals.split()], dtype=np.uint64)
        r, _ = oracle.lattice_points(n, [1, z2], [0.0, 0.0], 0, n)
        assert np.array_equal(r[:, 0], np.arange(n, dtype=np.uint64))
        assert np.array_equal(r[:, 1], want)


@pytest.mark.parametrize("n", [7, 11, 55, 1021, 65537])
def test_residues_are_permutations(n):
    z = [c for c in range(1, n) if math.gcd(c, n) == 1][:: max(1, n // 7)][:6]
    r, _ = oracle.lattice_points(n, z, [0.0] * len(z), 0, n)
    for j in range(len(z)):
        assert np.array_equal(np.sort(r[:, j]), np.arange(n, dtype=np.uint64))


def test_residues_large_n_bigint():
    n = 15173222401                      # the paper's largest lattice, P:L1032 (needs > 64-bit products)
    z = [1, 6543210987, 15173222400, 9999999967]
    rng = np.random.default_rng(1)
    for k0 in [0, 1, n - 5, int(rng.integers(1 << 32, n - 10))]:
        r, _ = oracle.lattice_points(n, z, [0.0] * 4, k0, 5)
        for i in range(5):
            for j in range(4):
                assert int(r[i, j]) == ((k0 + i) * z[j]) % n


# -------------------------------------------------------- coordinates (O2, "{ }" P:L100, reading C-2)
@pytest.mark.parametrize("n", [55, 65537, 1073741789, 15173222401])
def test_coordinates_exact_rational(n):
    rng = np.random.default_rng(n % 1000)
    z = [1, n // 3 + 1 if math.gcd(n // 3 + 1, n) == 1 else n // 3 + 2, n - 1]
    shift = rng.random(3)
    shift[2] = 1.0 - 2.0 ** -53          # largest double below 1
    cnt = min(200, n)
    k0 = int(rng.integers(0, n - cnt + 1))
    r, u = oracle.lattice_points(n, z, shift, k0, cnt)
    assert np.all(u >= 0.0) and np.all(u < 1.0)
    for i in range(cnt):
        for j in range(3):
            exact = Fraction(int(r[i, j]), n) + Fraction(float(shift[j]))
            exact -= int(exact)           # fractional part
            err = abs(Fraction(float(u[i, j])) - exact)
            err = min(err, 1 - err)       # a value that rounds up to 1.0 wraps to 0.0
            assert err <= Fraction(1, 2 ** 52)


def test_coordinates_d1_mean_closed_form():
    # z = 1: mean over k of {k/n + D} = (n-1)/(2n) + frac(n D)/n
    n, D = 1021, 0.3437
    _, u = oracle.lattice_points(n, [1], [D], 0, n)
    want = (n - 1) / (2 * n) + ((n * D) % 1.0) / n
    assert abs(math.fsum(u[:, 0]) / n - want) < 1e-14


# ---------------------------------------------------------------------------- transforms (O3)
@pytest.mark.parametrize("r", [1, 2, 3, 4, 5, 6])
def test_korobov_normalisation_and_phi(r):
    # Eq. 15: (2r+1) C(2r,r) = 1 / B(r+1, r+1);  Eq. 14: phi = regularised incomplete beta
    c = 1.0 / scipy.special.beta(r + 1, r + 1)
    assert abs(c - (2 * r + 1) * math.comb(2 * r, r)) < 1e-9 * c
    for u in [0.0, 1e-9, 0.003, 0.1, 0.31, 0.5, 0.5000001, 0.77, 0.999, 1.0 - 2.0 ** -53]:
        y, w = oracle.transform(synth.TRANSFORM_KOROBOV + r, u)
        want_y = scipy.special.betainc(r + 1, r + 1, u)
        assert abs(y - want_y) <= 4e-15 * max(want_y, 1e-300) + 1e-300 or abs(y - want_y) < 1e-16
        assert abs(w - c * u ** r * (1 - u) ** r) <= 1e-14 * c
        y2, _ = oracle.transform(synth.TRANSFORM_KOROBOV + r, 1.0 - u)
        assert abs(y + y2 - 1.0) < 1e-15
    assert oracle.transform(synth.TRANSFORM_KOROBOV + r, 0.0) == (0.0, 0.0)
    # phi as the integral of omega (Eq. 14) by Gauss-Legendre, exact for these polynomials
    xs, ws = np.polynomial.legendre.leggauss(12)
    for u in [0.2, 0.6, 0.95]:
        t = 0.5 * u * (xs + 1.0)
        quad = 0.5 * u * np.sum(ws * np.array([oracle.transform(synth.TRANSFORM_KOROBOV + r, v)[1] for v in t]))
        assert abs(quad - oracle.transform(synth.TRANSFORM_KOROBOV + r, u)[0]) < 1e-14


@pytest.mark.parametrize("r0,r1", [(1, 2), (2, 1), (3, 1), (1, 4), (5, 3), (2, 6), (6, 6), (4, 4)])
def test_korobov_asymmetric_is_the_incomplete_beta(r0, r1):
    # Eq. 15: omega = u^r0 (1-u)^r1 / B(r0+1, r1+1); Eq. 14: phi = I_u(r0+1, r1+1); Korobov<5,3> is the paper's example
    tr = synth.TRANSFORM_KOROBOV_ASYM + 16 * r0 + r1
    c = 1.0 / scipy.special.beta(r0 + 1, r1 + 1)
    assert abs(c - (r0 + r1 + 1) * math.comb(r0 + r1, r0)) < 1e-9 * c
    for u in [0.0, 1e-7, 0.02, 0.3, 0.5, 0.50001, 0.8, 0.9999, 1.0 - 2.0 ** -53]:
        y, w = oracle.transform(tr, u)
        want = scipy.special.betainc(r0 + 1, r1 + 1, u)
        assert abs(y - want) <= 8e-15 * want + 1e-300 or abs(y - want) < 2e-16
        assert abs(w - c * u ** r0 * (1 - u) ** r1) <= 1e-14 * c
        ym, _ = oracle.transform(synth.TRANSFORM_KOROBOV_ASYM + 16 * r1 + r0, 1.0 - u)   # mirror symmetry
        assert abs(y + ym - 1.0) < 1e-15
    if r0 == r1:                                            # the symmetric id is the same transform
        for u in [0.1, 0.5, 0.9]:
            assert oracle.transform(tr, u) == oracle.transform(synth.TRANSFORM_KOROBOV + r0, u)
    for bad in (synth.TRANSFORM_KOROBOV_ASYM + 16 * 0 + 3, synth.TRANSFORM_KOROBOV_ASYM + 16 * 7 + 1, synth.TRANSFORM_KOROBOV_ASYM + 16 * 2 + 9):
        with pytest.raises(ValueError):
            oracle.transform(bad, 0.5)


@pytest.mark.parametrize("r", [1, 2, 3, 4, 5, 6])
def test_sidi_normalisation_and_phi(r):
    # Eq. 16: omega = K_r sin^r(pi u), K_r = pi/2^r Gamma(r+1)/Gamma((r+1)/2)^2 = 1 / int_0^1 sin^r(pi t) dt
    tr = synth.TRANSFORM_SIDI + r
    K = math.pi / 2 ** r * math.gamma(r + 1) / math.gamma((r + 1) / 2) ** 2
    assert abs(K - {1: math.pi / 2, 2: 2.0, 3: 3 * math.pi / 4, 4: 8 / 3, 5: 15 * math.pi / 16, 6: 16 / 5}[r]) < 1e-14 * K
    norm, _ = scipy.integrate.quad(lambda t: math.sin(math.pi * t) ** r, 0.0, 1.0, epsabs=1e-13, epsrel=1e-13)
    assert abs(K * norm - 1.0) < 1e-13
    assert oracle.transform(tr, 0.0)[0] == 0.0 and abs(oracle.transform(tr, 0.0)[1]) < 1e-15
    assert abs(oracle.transform(tr, 1.0 - 2.0 ** -53)[0] - 1.0) < 1e-15
    assert abs(oracle.transform(tr, 0.5)[0] - 0.5) < 1e-15 and abs(oracle.transform(tr, 0.5)[1] - K) < 1e-14 * K
    xs, ws = np.polynomial.legendre.leggauss(40)
    for u in [0.003, 0.2, 0.45, 0.6, 0.95, 0.999]:
        y, w = oracle.transform(tr, u)
        assert abs(w - K * math.sin(math.pi * u) ** r) <= 1e-14 * K
        t = 0.5 * u * (xs + 1.0)                             # phi = int_0^u omega (Eq. 14) by Gauss-Legendre
        quad = 0.5 * u * np.sum(ws * K * np.sin(np.pi * t) ** r)
        assert abs(quad - y) < 1e-14
        y2, _ = oracle.transform(tr, 1.0 - u)
        assert abs(y + y2 - 1.0) < 2e-15
    with pytest.raises(ValueError):
        oracle.transform(synth.TRANSFORM_SIDI + 7, 0.5)


@pytest.mark.parametrize("tr,rel", [(synth.TRANSFORM_SIDI + 2, 3e-6), (synth.TRANSFORM_SIDI + 3, 3e-7),
                                    (synth.TRANSFORM_KOROBOV_ASYM + 16 * 3 + 2, 1e-5), (synth.TRANSFORM_KOROBOV_ASYM + 16 * 1 + 4, 1e-3)])
def test_new_transforms_leave_the_integral_invariant(tr, rel):
    """Eq. 12: the transformed rule still integrates f; closed form of Genz oscillatory"""
    rng = synth.MT19937_64(2024)
    prm = synth.genz_osc(rng, 4)
    p = synth.problem(0, prm, 8191, synth.genvec(65537, 4) % 8191, synth.draw_shifts(rng, 8, 4), tr)
    _check_vs_exact(p, closed_osc(prm), rel=rel)


def test_baker_and_none():
    # Eq. 17: 2u below 1/2, 2-2u above; weight 1
    for u, y in [(0.0, 0.0), (0.25, 0.5), (0.5, 1.0), (0.75, 0.5), (0.9, 0.2)]:
        got = oracle.transform(synth.TRANSFORM_BAKER, u)
        assert abs(got[0] - y) < 1e-15 and got[1] == 1.0
        assert oracle.transform(synth.TRANSFORM_NONE, u) == (u, 1.0)
    with pytest.raises(ValueError):
        oracle.transform(synth.TRANSFORM_KOROBOV + 7, 0.5)


# ------------------------------------------------------------------------------- fit map (O4)
def test_fit_map_endpoints_and_derivative():
    for a in [[1.001, -0.001, 0.0, 0.0, 0.6, 0.3], [1.5, -0.4, 0.2, 0.1, 0.3, 0.25], [2.0, -1.0, 0.05, 0.3, 1.0, -0.2]]:
        assert oracle.fit_map(a, 0.0)[0] == 0.0            # p(0) = 0
        assert abs(oracle.fit_map(a, 1.0)[0] - 1.0) < 1e-15  # p(1) = 1
        for y in [0.1, 0.37, 0.8]:
            h = 1e-6
            fd = (oracle.fit_map(a, y + h)[0] - oracle.fit_map(a, y - h)[0]) / (2 * h)
            assert abs(fd - oracle.fit_map(a, y)[1]) < 1e-8
    # Eq. 19 written out for one point
    a0, a1, a2, a3, a4, a5 = 1.5, -0.4, 0.2, 0.1, 0.3, 0.25
    y = 0.3
    want = a2 * y * (a0 - 1) / (a0 - y) + a3 * y * (a1 - 1) / (a1 - y) + a4 * y + a5 * y ** 2 + (1 - a2 - a3 - a4 - a5) * y ** 3
    assert abs(oracle.fit_map([a0, a1, a2, a3, a4, a5], y)[0] - want) < 1e-15


# --------------------------------------------------------- lattice rule on Fourier modes (O1-O6)
def _mode_problem(n, z, h, shifts):
    d = len(z)
    prm = np.array([2 * math.pi * v for v in h] + [0.0] * d)      # f = exp(2 pi i h.x)
    return synth.problem(synth.FAMILY_CEXP_POLY, prm, n, z, shifts, synth.TRANSFORM_NONE)


def test_rule_exact_on_fourier_modes():
    n, z = 1021, [1, 374, 147]
    rng = synth.MT19937_64(7)
    sh = synth.draw_shifts(rng, 3, 3)
    # h.z != 0 (mod n): the rule returns 0; h.z == 0: it returns exp(2 pi i h.Delta)
    for h in [(1, 0, 0), (0, 2, -1), (3, -2, 5), (-7, 1, 1)]:
        assert sum(a * b for a, b in zip(h, z)) % n != 0
        sm, _, _ = oracle.integrate(_mode_problem(n, z, h, sh))
        assert np.max(np.abs(sm)) < 1e-12
    for h in [(-374, 1, 0), (-147, 0, 1), (n, 0, 0), (0, 0, 0)]:
        assert sum(a * b for a, b in zip(h, z)) % n == 0
        sm, _, _ = oracle.integrate(_mode_problem(n, z, h, sh))
        for s in range(3):
            ph = 2 * math.pi * math.fsum(a * b for a, b in zip(h, sh[s]))
            tol = 2 * math.pi * sum(abs(v) for v in h) * 2.0 ** -51 + 1e-13
            assert abs(sm[s, 0] - math.cos(ph)) < tol and abs(sm[s, 1] - math.sin(ph)) < tol


@pytest.mark.parametrize("n,z", [(65537, 25016), (1048573, 32373), (55, 34)])
def test_one_dimensional_rule_is_a_geometric_series(n, z):
    """d = 1, transform None: k z mod n runs through 0..n-1 (z coprime to n), so Eq. 2 is the equispaced sum
    (1/n) sum_j cos(phi + a (j + theta)/n), theta = frac(n Delta) = sin(a/2) / (n sin(a/(2n))) cos(phi + a (theta - 1/2)/n + a/2):
    an exact value of the whole rule (residues, coordinates, integrand, compensated sum) to rounding"""
    prm = np.array([0.3125, 1.75])
    sh = np.array([[0.6180339887498949], [0.1415926535897932], [0.0]])
    p = synth.problem(0, prm, n, np.array([z], dtype=np.uint64), sh, synth.TRANSFORM_NONE)
    sm, mean, err = oracle.integrate(p)
    phi, a = 2 * np.pi * prm[0], prm[1]
    for s_, delta in enumerate(sh[:, 0]):
        theta = float((Fraction(delta) * n) % 1)
        want = np.sin(a / 2) / (n * np.sin(a / (2 * n))) * np.cos(phi + a * (theta - 0.5) / n + a / 2)
        assert abs(sm[s_, 0] - want) <= 2e-15 * abs(want)


def test_sum_against_fsum_python():
    # the whole chain in slow exact-ish python: Fractions for the point, math.fsum for the sum
    n, z = 251, [1, 97, 33]
    prm = np.array([0.3, 0.9, 0.4, 0.7])
    sh = synth.draw_shifts(synth.MT19937_64(3), 2, 3)
    p = synth.problem(synth.FAMILY_GENZ_OSC, prm, n, z, sh, synth.TRANSFORM_NONE)
    sums = oracle.shift_sums(p)
    for s in range(2):
        terms = []
        for k in range(n):
            x = [float((Fraction(k * z[j] % n, n) + Fraction(float(sh[s, j]))) % 1) for j in range(3)]
            terms.append(math.cos(2 * math.pi * prm[0] + math.fsum(prm[1 + j] * x[j] for j in range(3))))
        assert abs(sums[s, 0] - math.fsum(terms)) < 1e-12
    # sub-ranges add up to the whole
    part = oracle.shift_sums(p, 0, 100) + oracle.shift_sums(p, 100, n)
    assert np.allclose(part, sums, rtol=0, atol=1e-13)


# --------------------------------------------------------------- closed forms of the families (O5)
def closed_osc(prm):
    u0, a = prm[0], prm[1:]
    return math.cos(2 * math.pi * u0 + 0.5 * a.sum()) * np.prod(np.sin(a / 2) / (a / 2))


def closed_prodpeak(prm):
    d = len(prm) // 2
    c, w = prm[:d], prm[d:]
    return np.prod(c * (np.arctan(c * (1 - w)) + np.arctan(c * w)))


def closed_cexp(prm):
    d = len(prm) // 2
    out = 1.0 + 0j
    for a, b in zip(prm[:d], prm[d:]):
        ia = 1j * a
        e = np.exp(ia)
        out *= (e - 1) / ia + b * (e / ia - (e - 1) / ia ** 2)
    return out


def test_closed_cexp_matches_quad():
    a, b = 1.7, 0.6
    re = scipy.integrate.quad(lambda x: math.cos(a * x) * (1 + b * x), 0, 1)[0]
    im = scipy.integrate.quad(lambda x: math.sin(a * x) * (1 + b * x), 0, 1)[0]
    assert abs(closed_cexp(np.array([a, b])) - complex(re, im)) < 1e-13


def _check_vs_exact(p, exact, nsig=6.0, rel=None, floor=1e-14):
    # floor = relative accuracy of `exact` itself (1e-14 for closed forms, larger for quadrature)
    sm, mean, err = oracle.integrate(p)
    val = complex(mean[0], mean[1]) if len(mean) == 2 else mean[0]
    e = float(np.max(err))
    assert abs(val - exact) <= nsig * e + floor * abs(exact), (val, exact, e)
    if rel is not None:
        assert abs(val - exact) <= rel * abs(exact), (val, exact)
    return val, e


@pytest.mark.parametrize("tr,rel", [(synth.TRANSFORM_NONE, 3e-3), (synth.TRANSFORM_BAKER, 1e-5), (K3, 1e-7),
                                    (synth.TRANSFORM_KOROBOV + 1, 1e-4), (synth.TRANSFORM_KOROBOV + 2, 1e-6),
                                    (synth.TRANSFORM_KOROBOV + 5, 1e-6)])
def test_family0_closed_form_all_transforms(tr, rel):
    # invariance of the integral under every periodizing transform, Eq. 12
    n, d = 65537, 4
    rng = synth.MT19937_64(11)
    prm = synth.genz_osc(rng, d)
    p = synth.problem(synth.FAMILY_GENZ_OSC, prm, n, synth.genvec(n, d), synth.draw_shifts(rng, 12, d), tr)
    _check_vs_exact(p, closed_osc(prm), rel=rel)


def test_family1_closed_form():
    n, d = 65537, 4
    rng = synth.MT19937_64(12)
    prm = synth.genz_prodpeak(rng, d)
    for tr, rel in [(synth.TRANSFORM_BAKER, 1e-4), (K3, 1e-5)]:
        p = synth.problem(synth.FAMILY_GENZ_PRODPEAK, prm, n, synth.genvec(n, d), synth.draw_shifts(rng, 12, d), tr)
        _check_vs_exact(p, closed_prodpeak(prm), rel=rel)


def test_family2_closed_form():
    n, d = 65537, 4
    rng = synth.MT19937_64(13)
    prm = synth.cexp_poly(rng, d)
    p = synth.problem(synth.FAMILY_CEXP_POLY, prm, n, synth.genvec(n, d), synth.draw_shifts(rng, 12, d), K3)
    _check_vs_exact(p, closed_cexp(prm), rel=1e-6)


def closed_genz(fam, prm, d):
    """analytic integrals of Genz families 3-6 over the unit cube"""
    c = prm[:d]
    if fam == synth.FAMILY_GENZ_CORNER:                     # inclusion-exclusion over the corners
        tot = 0.0
        for mask in range(1 << d):
            sel = [j for j in range(d) if mask >> j & 1]
            tot += (-1.0) ** len(sel) / (1.0 + sum(c[j] for j in sel))
        return tot / (math.factorial(d) * np.prod(c))
    if fam == synth.FAMILY_GENZ_GAUSSIAN:
        w = prm[d:]
        return float(np.prod(np.sqrt(np.pi) / (2 * c) * (scipy.special.erf(c * (1 - w)) + scipy.special.erf(c * w))))
    if fam == synth.FAMILY_GENZ_C0:
        w = prm[d:]
        return float(np.prod((2.0 - np.exp(-c * w) - np.exp(-c * (1 - w))) / c))
    b = np.ones(d)
    b[:min(d, 2)] = prm[d:]
    return float(np.prod(np.expm1(c * b) / c))


@pytest.mark.parametrize("fam", [4, 5, 6, 7])
def test_genz_families_3_to_6_pointwise_and_closed_form(fam):
    rng = synth.MT19937_64(600 + fam)
    d = 4
    prm = synth.genz_protocol(rng, fam, d)
    # pointwise against the definitions
    for _ in range(20):
        x = np.array([rng.uniform() for _ in range(d)])
        c = prm[:d]
        if fam == 4:
            want = (1.0 + c @ x) ** -(d + 1)
        elif fam == 5:
            want = math.exp(-np.sum(c ** 2 * (x - prm[d:]) ** 2))
        elif fam == 6:
            want = math.exp(-np.sum(c * np.abs(x - prm[d:])))
        else:
            want = 0.0 if (x[0] > prm[d] or x[1] > prm[d + 1]) else math.exp(c @ x)
        assert abs(oracle.integrand(fam, prm, x) - want) <= 1e-14 * max(abs(want), 1e-300)
    # the rule integrates them: closed form inside the error bar (baker copes with the kinks of families 5, 6)
    n = 65521
    tr = synth.TRANSFORM_KOROBOV + 3 if fam in (4, 5) else synth.TRANSFORM_BAKER
    p = synth.problem(fam, prm, n, synth.genvec(n, 4), synth.draw_shifts(rng, 8, d), tr)
    _check_vs_exact(p, closed_genz(fam, prm, d), nsig=6.0, rel={4: 1e-8, 5: 1e-6, 6: 1e-4, 7: 2e-2}[fam])
    with pytest.raises(ValueError):
        oracle.integrand(fam, prm[:-1], np.zeros(d))


def test_corner_peak_closed_form_against_nested_quadrature():
    # the inclusion-exclusion formula itself, checked by tensor Gauss-Legendre at d = 3
    c = np.array([0.9, 0.4, 0.7])
    xs, ws = np.polynomial.legendre.leggauss(24)
    xs, ws = 0.5 * (xs + 1), 0.5 * ws
    X = np.stack(np.meshgrid(xs, xs, xs, indexing="ij"), -1)
    quad = np.sum(np.einsum("i,j,k->ijk", ws, ws, ws) * (1.0 + X @ c) ** -4.0)
    assert abs(quad - closed_genz(4, c, 3)) < 1e-13


def test_fit_map_leaves_integral_invariant():
    # Eq. 18 with arbitrary valid coefficients, composed as x = p(phi(u))
    n, d = 65537, 4
    rng = synth.MT19937_64(14)
    prm = synth.genz_osc(rng, d)
    sh = synth.draw_shifts(rng, 12, d)
    fit = synth.cubic_fit_coeffs(d, 0.6, 0.3)
    fit[1] = [1.4, -0.3, 0.15, 0.1, 0.5, 0.2]            # full Eq. 19 in one dimension
    p = synth.problem(synth.FAMILY_GENZ_OSC, prm, n, synth.genvec(n, d), sh, K3, fit_coeffs=fit)
    _check_vs_exact(p, closed_osc(prm), rel=1e-6)


def test_minimal_example_one_eighth():
    # Fig. 2: f = x0 x1 x2, Korobov-3 -> 1/8; here as a degenerate sector integrand
    d, n = 3, 8191
    prm = np.array([1, 2, 1, 1, 1, 1, 1, 1.0, 0, 0, 0, 1.0, 0, 0, 0], dtype=np.float64)   # U = F = 1, nu = (1,1,1)
    rng = synth.MT19937_64(15)
    p = synth.problem(synth.FAMILY_SECTOR, prm, n, synth.korobov_form_vector(n, d, 1487), synth.draw_shifts(rng, 32, d), K3)
    _check_vs_exact(p, 0.125, rel=1e-6)


def _sector_numpy(prm, d, X):
    """Independent vectorised evaluation of prod x^nu U^a / F^b on points X (N, d)."""
    a, b, nU, nF = (int(v) for v in prm[:4])
    nu = prm[4:4 + d]
    o = 4 + d
    cU, eU = prm[o:o + nU], prm[o + nU:o + nU + nU * d].reshape(nU, d)
    o += nU * (1 + d)
    cF, eF = prm[o:o + nF], prm[o + nF:o + nF + nF * d].reshape(nF, d)
    U = sum(cU[t] * np.prod(X ** eU[t], axis=1) for t in range(nU))
    F = sum(cF[t] * np.prod(X ** eF[t], axis=1) for t in range(nF))
    return np.prod(X ** nu, axis=1) * U ** a / F ** b


@pytest.mark.parametrize("d,seed", [(2, 21), (3, 22), (3, 23)])
def test_family3_tensor_gauss_legendre(d, seed):
    rng = synth.MT19937_64(seed)
    prm = synth.sector(rng, d)
    xs, ws = np.polynomial.legendre.leggauss(24)
    xs, ws = 0.5 * (xs + 1), 0.5 * ws
    grids = np.meshgrid(*([xs] * d), indexing="ij")
    X = np.stack([g.ravel() for g in grids], axis=1)
    Wt = np.prod(np.stack([g.ravel() for g in np.meshgrid(*([ws] * d), indexing="ij")], axis=1), axis=1)
    exact = float(np.sum(Wt * _sector_numpy(prm, d, X)))
    n = 65537
    p = synth.problem(synth.FAMILY_SECTOR, prm, n, synth.genvec(n, 4)[:d], synth.draw_shifts(rng, 12, d), K3)
    _check_vs_exact(p, exact, rel=1e-7, floor=1e-11)      # 24-node Gauss-Legendre is good to ~1e-12
    # pointwise: oracle integrand vs the numpy restatement
    pts = np.array([[rng.uniform() for _ in range(d)] for _ in range(5)])
    for x, want in zip(pts, _sector_numpy(prm, d, pts)):
        assert abs(oracle.integrand(synth.FAMILY_SECTOR, prm, x) - want) <= 1e-14 * abs(want)


# --- log factors of the sector family (trailing [lu, lf, p], reading C-15) ---
def _one_dim_log_problem(prm, n=65537, seed=31):
    rng = synth.MT19937_64(seed)
    return synth.problem(synth.FAMILY_SECTOR, np.array(prm, dtype=np.float64), n, np.array([1], dtype=np.uint64),
                         synth.draw_shifts(rng, 8, 1), K3)


def test_sector_log_closed_forms_one_dimension():
    L2 = math.log(2.0)
    # U = 1 + x, F = 1, a = b = 0:  int log(1+x) = 2 ln 2 - 1;  int log^2(1+x) = 2 ln^2 2 - 4 ln 2 + 2
    base = [0, 0, 2, 1, 0, 1.0, 1.0, 0, 1, 1.0, 0]
    _check_vs_exact(_one_dim_log_problem(base + [1.0, 0.0, 1]), 2 * L2 - 1, rel=1e-9)
    _check_vs_exact(_one_dim_log_problem(base + [1.0, 0.0, 2]), 2 * L2 * L2 - 4 * L2 + 2, rel=1e-9)
    # coefficient lu scales the term; lf multiplies log F = log 1 = 0 here
    _check_vs_exact(_one_dim_log_problem(base + [-2.5, 7.0, 1]), -2.5 * (2 * L2 - 1), rel=1e-9)
    # U = 1, F = 1 + x, b = 1: int log(1+x)/(1+x) = ln^2 2 / 2 (lf picks F, lu picks U = 1)
    base = [0, 1, 1, 2, 0, 1.0, 0, 1.0, 1.0, 0, 1]
    _check_vs_exact(_one_dim_log_problem(base + [9.0, 1.0, 1]), 0.5 * L2 * L2, rel=1e-9)
    # U = 1 + x, a = 1, F = 2 (constant): int (1+x)/2 * (log(1+x) - log 2) = [ (1+x)^2 (2 log(1+x) - 1) / 8 ]_0^1 - 3 ln 2 / 4
    base = [1, 1, 2, 1, 0, 1.0, 1.0, 0, 1, 2.0, 0]
    exact = (4 * (2 * L2 - 1) / 8 + 1 / 8) - 0.75 * L2
    _check_vs_exact(_one_dim_log_problem(base + [1.0, -1.0, 1]), exact, rel=1e-9)


@pytest.mark.parametrize("d,seed", [(2, 41), (3, 42), (6, 43)])
def test_sector_log_is_the_epsilon_derivative(d, seed):
    """f L^p is the p-th eps-derivative at 0 of prod x^nu U^(a + lu eps) F^(-b + lf eps): checked pointwise against real
    powers (numpy, central differences in extended steps), which involve no logarithm of the oracle's."""
    rng = synth.MT19937_64(seed)
    prm = synth.sector_log(rng, d)
    lu, lf, pw = prm[-3], prm[-2], int(prm[-1])
    base = prm[:-3]
    a, b, nU, nF = (int(v) for v in base[:4])
    o = 4 + d
    cU, eU = base[o:o + nU], base[o + nU:o + nU + nU * d].reshape(nU, d)
    o += nU * (1 + d)
    cF, eF = base[o:o + nF], base[o + nF:o + nF + nF * d].reshape(nF, d)
    X = np.array([[rng.uniform() for _ in range(d)] for _ in range(6)])
    U = np.array([sum(cU[t] * np.prod(x ** eU[t]) for t in range(nU)) for x in X]).astype(np.longdouble)
    F = np.array([sum(cF[t] * np.prod(x ** eF[t]) for t in range(nF)) for x in X]).astype(np.longdouble)
    pre = np.prod(X ** base[4:4 + d], axis=1).astype(np.longdouble)

    def g(eps):
        eps = np.longdouble(eps)
        return pre * U ** (a + np.longdouble(lu) * eps) * F ** (-b + np.longdouble(lf) * eps)

    h = 2e-3 if pw > 1 else 1e-4
    # central differences, O(h^2) error removed by one Richardson step
    def deriv(h):
        if pw == 1:
            return (g(h) - g(-h)) / (2 * h)
        if pw == 2:
            return (g(h) - 2 * g(0) + g(-h)) / (h * h)
        return (g(2 * h) - 2 * g(h) + 2 * g(-h) - g(-2 * h)) / (2 * h ** 3)
    want = (4 * deriv(h / 2) - deriv(h)) / 3
    # the difference quotient is accurate relative to the size of its terms, not to a result that nearly cancels
    scale = np.asarray(g(0) * (abs(lu) * np.abs(np.log(U)) + abs(lf) * np.abs(np.log(F))) ** pw, dtype=np.float64)
    for x, w, sc in zip(X, want, scale):
        got = oracle.integrand(synth.FAMILY_SECTOR, prm, x)
        assert abs(got - float(w)) <= 2e-6 * sc, (got, float(w), sc)
    # and p is only accepted as an integer in 1..4
    bad = prm.copy(); bad[-1] = 0.0
    with pytest.raises(ValueError):
        oracle.integrand(synth.FAMILY_SECTOR, bad, X[0])


def test_integrand_param_count_checked():
    with pytest.raises(ValueError):
        oracle.integrand(synth.FAMILY_GENZ_OSC, [0.1, 0.2], [0.5, 0.5])


# ------------------------------------------------------------------------- Eq. 3 (O7, O8)
@pytest.mark.parametrize("m", [2, 10, 33])
def test_error_estimate_hand_made(m):
    mean, err = oracle.finalize(np.arange(1, m + 1, dtype=np.float64))
    assert abs(mean[0] - (m + 1) / 2) < 1e-15 * m
    assert abs(err[0] - math.sqrt((m + 1) / 12.0)) < 1e-15 * m
    # complex: components separately
    q = np.stack([np.arange(1, m + 1.0), 5.0 - 2.0 * np.arange(1, m + 1.0)], axis=1)
    mean, err = oracle.finalize(q)
    assert abs(mean[1] - (5.0 - (m + 1))) < 1e-13 and abs(err[1] - 2 * math.sqrt((m + 1) / 12.0)) < 1e-14 * m
    with pytest.raises(ValueError):
        oracle.finalize(np.array([1.0]))


# ------------------------------------------------------------- projection and cubic fit (O9)
def test_projection_marginals_product_peak():
    n, d, B = 65537, 3, 16
    rng = synth.MT19937_64(31)
    prm = synth.genz_prodpeak(rng, d)
    p = synth.problem(synth.FAMILY_GENZ_PRODPEAK, prm, n, synth.genvec(n, 4)[:d], synth.draw_shifts(rng, 1, d), synth.TRANSFORM_NONE)
    H = oracle.project(p, B)
    tot = oracle.shift_sums(p)[0, 0]                   # f > 0: sum |f| = sum f
    c, w = prm[:d], prm[d:]
    for j in range(d):
        assert abs(H[j].sum() - tot) < 1e-12 * tot
        edges = np.arange(B + 1) / B
        cdf = np.arctan(c[j] * (edges - w[j]))
        want = np.diff(cdf) / (cdf[-1] - cdf[0])
        assert np.max(np.abs(H[j] / tot - want)) < 2e-3


def test_fit_recovers_exact_cubic():
    B, a4, a5 = 256, 0.55, 0.35
    a6 = 1 - a4 - a5
    edges = np.arange(B + 1) / B
    cdf = np.array([0.0] + [min(r.real for r in np.roots([a6, a5, a4, -e]) if abs(r.imag) < 1e-12 and -1e-12 <= r.real <= 1 + 1e-12)
                            for e in edges[1:]])
    H = np.stack([np.diff(cdf), np.full(B, 1.0 / B)])
    out = oracle.fit_cubic(H)
    assert abs(out[0, 4] - a4) < 1e-9 and abs(out[0, 5] - a5) < 1e-9
    assert abs(out[1, 4] - 1.0) < 1e-12 and abs(out[1, 5]) < 1e-12      # flat marginal -> identity
    assert np.all(out[:, 2:4] == 0.0)
    # a non-monotone least-squares solution falls back to the identity
    H2 = np.zeros((1, B)); H2[0, 0] = 1.0
    out2 = oracle.fit_cubic(H2)
    assert out2[0, 4] == 1.0 and out2[0, 5] == 0.0


# ------------------------------------------------------------------------------------------------
# stored full-size records (tests/golden/fullsize_oracle.json) must be what the committed oracle computes
# ------------------------------------------------------------------------------------------------
def test_fullsize_goldens_are_what_the_live_oracle_computes():
    """Recomputes one stored record (sector 17 of configs[3] at full size, a few seconds of oracle time) with the live
    oracle and requires BIT identity, so that a golden file that lags an oracle change cannot go unnoticed (a stored mean
    is a whole-lattice sum: a cheaper partial check does not exist)."""
    import json
    path = os.path.join(GOLD, "fullsize_oracle.json")
    with open(path) as f:
        g = json.load(f)
    assert sorted(int(k) for k in g["3"]["sectors"]) == list(range(256))
    for key in ("2", "3", "4"):
        assert len(g["provenance"][key]["oracle_sha256"]) == 64          # which oracle source wrote the record
    rec = g["3"]["sectors"]["17"]
    p = synth.config(3)[17]
    assert rec["n"] == p["n"] and rec["m"] == p["m"] and rec["dim"] == p["dim"] and rec["name"] == p["name"]
    sm, mean, err = oracle.integrate(p)
    assert [float(v).hex() for v in np.asarray(sm).ravel()] == rec["shift_means"]
    assert [float(v).hex() for v in np.asarray(mean).ravel()] == rec["mean"]
    assert [float(v).hex() for v in np.asarray(err).ravel()] == rec["err"]


# ------------------------------------------------------------------------------------------------
# family 8: sector polynomials with COMPLEX coefficients (contour-deformed shape; reading C-16)
# ------------------------------------------------------------------------------------------------
def csector(a, b, nu, U, F, log_block=None):
    """U, F: lists of (complex coefficient, exponent tuple) -> parameter block of family 8"""
    d = len(nu)
    out = [float(a), float(b), float(len(U)), float(len(F))] + [float(v) for v in nu]
    for poly in (U, F):
        out += [complex(c).real for c, _ in poly] + [complex(c).imag for c, _ in poly]
        for _, e in poly:
            assert len(e) == d
            out += [float(v) for v in e]
    if log_block is not None:
        out += [float(v) for v in log_block]
    return np.array(out)


def gl_integral(prm, d, order=40):
    """tensor Gauss-Legendre of the oracle's integrand over the unit cube (d <= 2)"""
    xs, ws = np.polynomial.legendre.leggauss(order)
    xs, ws = 0.5 * (xs + 1.0), 0.5 * ws
    tot = 0.0 + 0.0j
    if d == 1:
        for x, w in zip(xs, ws):
            tot += w * oracle.integrand(8, prm, [x])
    else:
        for x0, w0 in zip(xs, ws):
            for x1, w1 in zip(xs, ws):
                tot += w0 * w1 * oracle.integrand(8, prm, [x0, x1])
    return tot


def test_complex_sector_one_dimensional_closed_forms():
    """int_0^1 1/(1+ix) = pi/4 - i ln2/2;  int 1/(1+ix)^2 = (1-i)/2;  int x/(1+ix)^2 = (1-ln2)/2 - i (pi/4 - 1/2);
    int (1+ix)^2 = 2/3 + i  -- which coefficient is the imaginary part, the powers a and b, the prefactor x^nu, the division"""
    one = [(1.0, (0,))]
    lin = [(1.0, (0,)), (1j, (1,))]
    ln2 = math.log(2.0)
    cases = [(csector(0, 1, [0], one, lin), math.pi / 4 - 0.5j * ln2),
             (csector(0, 2, [0], one, lin), 0.5 - 0.5j),
             (csector(0, 2, [1], one, lin), 0.5 * (1.0 - ln2) - 1j * (math.pi / 4 - 0.5)),
             (csector(2, 0, [0], lin, one), 2.0 / 3.0 + 1j),
             (csector(1, 1, [0], [(2.0 - 1j, (0,))], [(0.5j, (0,))]), (2.0 - 1j) / 0.5j)]     # constants: complex division alone
    for prm, exact in cases:
        got = gl_integral(prm, 1)
        assert abs(got - exact) <= 1e-13 * abs(exact), (got, exact)


def test_complex_sector_two_dimensional_product():
    """F = (1 + i x0)(1 + i x1) = 1 + i x0 + i x1 - x0 x1 (a negative real and two imaginary coefficients):
    int int 1/F = (pi/4 - i ln2/2)^2;  with a = 1, U = 1 + i x0: int int U/F = pi/4 - i ln2/2"""
    F = [(1.0, (0, 0)), (1j, (1, 0)), (1j, (0, 1)), (-1.0, (1, 1))]
    v = math.pi / 4 - 0.5j * math.log(2.0)
    assert abs(gl_integral(csector(0, 1, [0, 0], [(1.0, (0, 0))], F), 2) - v * v) <= 1e-13
    assert abs(gl_integral(csector(1, 1, [0, 0], [(1.0, (0, 0)), (1j, (1, 0))], F), 2) - v) <= 1e-13


@pytest.mark.parametrize("lam", [0.0, 0.3, 1.0, 2.5])
def test_complex_sector_cauchy_invariance_under_contour_deformation(lam):
    """The deformation z = x - i lam x (1 - x) dF/dx of int_0^1 dx / (c + x)^2 and of int int dx0 dx1 / (c + x0 + x1)^2 (x0
    deformed): every factor becomes a polynomial in the real x with complex coefficients (reading C-16), and by Cauchy's
    theorem the integral keeps its value 1/c - 1/(1+c), ln((c+1)^2 / (c (c+2))) for every lam."""
    c = 0.7
    U1 = [(1.0 - 1j * lam, (0,)), (2j * lam, (1,))]                          # Jacobian 1 - i lam (1 - 2x)
    F1 = [(c, (0,)), (1.0 - 1j * lam, (1,)), (1j * lam, (2,))]               # c + z
    got = gl_integral(csector(1, 2, [0], U1, F1), 1, order=60)
    assert abs(got - (1.0 / c - 1.0 / (1.0 + c))) <= 1e-12
    U2 = [(1.0 - 1j * lam, (0, 0)), (2j * lam, (1, 0))]
    F2 = [(c, (0, 0)), (1.0 - 1j * lam, (1, 0)), (1j * lam, (2, 0)), (1.0, (0, 1))]
    got2 = gl_integral(csector(1, 2, [0, 0], U2, F2), 2, order=60)
    assert abs(got2 - math.log((c + 1.0) ** 2 / (c * (c + 2.0)))) <= 1e-12


def test_complex_sector_log_factor_takes_the_principal_branch():
    """int_0^1 Log(1 + i x) dx and int_0^1 Log(-1 - i x) dx from the antiderivative (z Log z - z)/z' with arg in (-pi, pi]
    (the second path lies in the third quadrant: arg -> -pi, not +pi); a squared logarithm against scipy quadrature"""
    import cmath
    one = [(1.0, (0,))]
    G = lambda z: z * cmath.log(z) - z
    prm = csector(0, 0, [0], [(1.0, (0,)), (1j, (1,))], one, log_block=[1.0, 0.0, 1])
    assert abs(gl_integral(prm, 1, order=60) - (G(1 + 1j) - G(1 + 0j)) / 1j) <= 1e-13
    prm = csector(0, 0, [0], one, [(-1.0, (0,)), (-1j, (1,))], log_block=[0.0, 1.0, 1])
    exact = (G(-1 - 1j) - (-1.0) * complex(0.0, -math.pi) - 1.0) / (-1j)       # G(-1 - i0+) = (-1)(-i pi) + 1
    got = gl_integral(prm, 1, order=200)
    assert abs(got - exact) <= 1e-9 * abs(exact), (got, exact)                 # the integrand has a log kink at the end point
    assert got.imag < -2.0                                                     # arg near -pi: the other branch would give > +2
    prm = csector(1, 1, [0], [(1.0, (0,)), (0.5j, (1,))], [(2.0, (0,)), (-1j, (1,))], log_block=[0.7, -1.3, 2])
    f = lambda x: (1 + 0.5j * x) / (2 - 1j * x) * (0.7 * cmath.log(1 + 0.5j * x) - 1.3 * cmath.log(2 - 1j * x)) ** 2
    re = scipy.integrate.quad(lambda x: f(x).real, 0, 1, epsabs=1e-14, epsrel=1e-14)[0]
    im = scipy.integrate.quad(lambda x: f(x).imag, 0, 1, epsabs=1e-14, epsrel=1e-14)[0]
    assert abs(gl_integral(prm, 1) - complex(re, im)) <= 1e-13


def test_complex_sector_with_real_coefficients_is_the_real_sector():
    """imaginary parts zero: the value is that of family 3 for the same polynomials (and the imaginary part vanishes)"""
    rng = synth.MT19937_64(8801)
    for d in (2, 4, 6):
        prm3 = synth.sector(rng, d)
        nU, nF = int(prm3[2]), int(prm3[3])
        off = 4 + d
        cU, eU = prm3[off:off + nU], prm3[off + nU:off + nU + nU * d]
        off += nU * (1 + d)
        cF, eF = prm3[off:off + nF], prm3[off + nF:off + nF + nF * d]
        prm8 = np.concatenate([prm3[:4 + d], cU, np.zeros(nU), eU, cF, np.zeros(nF), eF])
        for _ in range(20):
            x = np.array([rng.uniform() for _ in range(d)])
            v3, v8 = oracle.integrand(3, prm3, x), oracle.integrand(8, prm8, x)
            assert abs(v8.real - v3) <= 2e-15 * abs(v3) and v8.imag == 0.0      # complex division rounds differently by ulps


def test_complex_sector_whole_rule():
    """Eq. 2-3 with family 8: the lam-deformed one-dimensional integral through the lattice rule (Korobov 3, baker, none)
    lands on 1/c - 1/(1+c) inside its error bars; both components get an error estimate"""
    c, lam = 0.7, 0.8
    prm = csector(1, 2, [0], [(1.0 - 1j * lam, (0,)), (2j * lam, (1,))], [(c, (0,)), (1.0 - 1j * lam, (1,)), (1j * lam, (2,))])
    rng = synth.MT19937_64(8802)
    exact = 1.0 / c - 1.0 / (1.0 + c)
    for tr in (K3, synth.TRANSFORM_BAKER):
        p = synth.problem(8, prm, 65537, [1], synth.draw_shifts(rng, 16, 1), tr)
        sm, mean, err = oracle.integrate(p)
        assert sm.shape == (16, 2) and err.shape == (2,)
        assert abs(mean[0] - exact) <= 6 * err[0] + 1e-12 and abs(mean[1]) <= 6 * err[1] + 1e-12
        assert abs(mean[0] - exact) < 1e-7


# ------------------------------------------------------------------------------------------------
# O9b: the paper's sort-based CDF sampling (reading C-8b)
# ------------------------------------------------------------------------------------------------
def test_cdf_samples_constant_integrand():
    """f = 1 (product of (1 + 0 x)): the empirical CDF at the t-th kept point is exactly t * step / n and the kept
    coordinates are the (t * step)-th smallest of the lattice's coordinates, whatever the dimension"""
    n, step, d = 1021, 10, 3
    rng = synth.MT19937_64(77001)
    p = synth.problem(2, np.zeros(2 * d), n, synth.korobov_form_vector(n, d, 341), synth.draw_shifts(rng, 1, d), synth.TRANSFORM_NONE)
    xs, cdf = oracle.cdf_samples(p, step)
    K = n // step
    assert xs.shape == (d, K)
    _, u = oracle.lattice_points(n, p["z"], p["shifts"][0], 0, n)
    for j in range(d):
        srt = np.sort(u[:, j])
        assert np.array_equal(xs[j], srt[step - 1::step][:K])
        np.testing.assert_allclose(cdf[j], (np.arange(1, K + 1) * step) / n, rtol=1e-15)


def test_cdf_samples_follow_the_marginal_cdf_in_closed_form():
    """product peak: the marginal CDF of dimension j is (atan(c (x - w)) + atan(c w)) / (atan(c (1 - w)) + atan(c w)); the
    sampled CDF must follow it to O(1/n) + the lattice's integration error; coordinates ascending, CDF non-decreasing, ends near 1"""
    n, step, d = 65537, 10, 4
    rng = synth.MT19937_64(77002)
    prm = synth.genz_prodpeak(rng, d)
    p = synth.problem(1, prm, n, synth.genvec(n, 4), synth.draw_shifts(rng, 1, d), synth.TRANSFORM_NONE)
    xs, cdf = oracle.cdf_samples(p, step)
    c, w = prm[:d], prm[d:]
    for j in range(d):
        assert np.all(np.diff(xs[j]) > 0) and np.all(np.diff(cdf[j]) >= 0)
        exact = (np.arctan(c[j] * (xs[j] - w[j])) + np.arctan(c[j] * w[j])) / (np.arctan(c[j] * (1 - w[j])) + np.arctan(c[j] * w[j]))
        assert np.max(np.abs(cdf[j] - exact)) < 2e-3
        assert 1.0 - cdf[j][-1] < 2.0 * step / n * 30


def test_cdf_samples_one_dimension_by_hand():
    """n = 11, z = 1, shift 0.05, f = 1 + 2 x (complex exp * poly family with a = 0, b = 2: |f| = 1 + 2x), step = 3: the three
    kept points and their cumulative sums written out with exact rationals"""
    n, step = 11, 3
    p = synth.problem(2, np.array([0.0, 2.0]), n, [1], np.array([[0.05]]), synth.TRANSFORM_NONE)
    xs, cdf = oracle.cdf_samples(p, step)
    x_all = sorted(Fraction(k, n) + Fraction(1, 20) for k in range(n))           # no wrap: 10/11 + 0.05 < 1
    f_all = [1 + 2 * x for x in x_all]
    tot = sum(f_all)
    for t in range(1, n // step + 1):
        i = t * step - 1
        assert abs(xs[0, t - 1] - float(x_all[i])) <= 2e-16
        assert abs(cdf[0, t - 1] - float(sum(f_all[:i + 1]) / tot)) <= 1e-15


def test_cubic_fit_from_cdf_samples_recovers_an_exact_cubic():
    """pairs (c, x) with x = p(c) for a cubic p of the family: the least squares returns its (a4, a5)"""
    a4, a5 = 0.55, 0.35
    c = np.linspace(0.001, 0.999, 500)
    x = c * (a4 + c * (a5 + c * (1 - a4 - a5)))
    out = oracle.fit_cubic_cdf(np.stack([x, x]), np.stack([c, c]))
    assert np.allclose(out[:, 4], a4, atol=1e-12) and np.allclose(out[:, 5], a5, atol=1e-12)
    assert np.all(out[:, 2] == 0) and np.all(out[:, 3] == 0)
