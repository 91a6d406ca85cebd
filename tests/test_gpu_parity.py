"""GPU parity: the CUDA path, called through the C ABI (paper_1811_11720_b200.binding), against the CPU
oracle element by element on the same seeded inputs.  Bars (BASELINE.json north_star):
  residues / coordinates  bit-exact
  per-shift means         |Q_s^gpu - Q_s^oracle| <= 1e-13 |Q_s^oracle|  (complex: modulus)
  error estimate          stage test 1e-12 relative; end to end with the propagated tolerance (C-6)
Run on the B200 box: python -m pytest tests -m gpu
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_1811_11720_b200 import binding, synth

pytestmark = pytest.mark.gpu

K = synth.TRANSFORM_KOROBOV
NONE, BAKER = synth.TRANSFORM_NONE, synth.TRANSFORM_BAKER
REL_MEANS = 1e-13
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fullsize_oracle.json")


# ------------------------------------------------------------------------------------------------
# helpers
# ------------------------------------------------------------------------------------------------
def run_gpu(problems, **plan_options):
    batch = binding.DeviceBatch(problems, **plan_options)
    batch.integrate()
    return batch.results()


def assert_means(sm_gpu, sm_or, what=""):
    """1e-13 relative per shift; for complex results relative to the modulus (a component may vanish)."""
    sm_gpu, sm_or = np.asarray(sm_gpu), np.asarray(sm_or)
    assert sm_gpu.shape == sm_or.shape, what
    scale = np.abs(sm_or) if sm_or.shape[1] == 1 else np.repeat(np.hypot(sm_or[:, :1], sm_or[:, 1:]), 2, axis=1)
    delta = np.abs(sm_gpu - sm_or)
    worst = float(np.max(delta / np.maximum(scale, 1e-300)))
    assert np.all(delta <= REL_MEANS * scale), f"{what}: worst relative deviation {worst:.3e}"
    return worst


def assert_err(err_gpu, err_or, sm_or, what=""):
    """Reading C-6 (ii): |err_gpu - err_or| <= 1e-12 err_or + 1e-13 max|Q_s| / sqrt(m-1)."""
    m, nc = sm_or.shape
    for c in range(nc):
        qmax = np.max(np.abs(sm_or[:, c])) if nc == 1 else np.max(np.hypot(sm_or[:, 0], sm_or[:, 1]))
        tol = 1e-12 * err_or[c] + 1e-13 * qmax / np.sqrt(m - 1)
        assert abs(err_gpu[c] - err_or[c]) <= tol, f"{what}: err {err_gpu[c]!r} vs {err_or[c]!r} (tol {tol:.3e})"


def check_against_oracle(problems, **plan_options):
    sms, means, errs = run_gpu(problems, **plan_options)
    for i, p in enumerate(problems):
        nc = oracle.ncomp(p["family"])
        sm_or, mean_or, err_or = oracle.integrate(p)
        assert_means(sms[i], sm_or, p["name"])
        # the outer mean inherits the tolerance of the per-shift means
        scale = np.max(np.abs(sm_or)) if nc == 1 else np.max(np.hypot(sm_or[:, 0], sm_or[:, 1]))
        assert np.all(np.abs(means[i, :nc] - mean_or) <= REL_MEANS * scale), p["name"]
        assert_err(errs[i, :nc], err_or, sm_or, p["name"])
        # stage test, reading C-6 (i): Eq. 3 on the GPU's own per-shift means, oracle formula vs device finalize
        mean_st, err_st = oracle.finalize(sms[i])
        np.testing.assert_allclose(errs[i, :nc], err_st, rtol=1e-12, atol=0, err_msg=p["name"])
        np.testing.assert_allclose(means[i, :nc], mean_st, rtol=1e-15, atol=1e-300, err_msg=p["name"])
        if nc == 1:
            assert means[i, 1] == 0.0 and errs[i, 1] == 0.0
    return sms, means, errs


def make(fam, d, n, m, tr, seed, fit=False, z=None, a_hi=1.0):
    rng = synth.MT19937_64(seed)
    if fam == 0:
        prm = synth.genz_osc(rng, d, a_hi)
    elif fam == 1:
        prm = synth.genz_prodpeak(rng, d)
    elif fam == 2:
        prm = synth.cexp_poly(rng, d)
    elif fam == 8:
        prm = synth.sector_complex(rng, d)                   # complex sector polynomials (reading C-16)
    elif fam >= 4:
        prm = synth.genz_protocol(rng, fam, d)               # Genz families 3-6 at the paper's difficulties
    else:
        prm = synth.sector(rng, d)
    sh = synth.draw_shifts(rng, m, d)
    if z is None:
        z = synth.korobov_form_vector(n, d, 1 + n // 3)
    fc = None
    if fit == "full":
        # Eq. 19 with pole terms inside the bounds of PAPER.md L231; every third dimension stays a pure cubic
        fc = np.array([[1.001 + 0.5 * rng.uniform(), -0.001 - 0.5 * rng.uniform(), 0.25 * rng.uniform() * (j % 3 != 2),
                        0.25 * rng.uniform() * (j % 3 != 2), 0.45 + 0.3 * rng.uniform(), 0.2 * rng.uniform() - 0.05] for j in range(d)])
    elif fit:
        fc = np.array([[1.001, -0.001, 0.0, 0.0, 0.45 + 0.5 * rng.uniform(), 0.5 * rng.uniform() - 0.1] for _ in range(d)])
    return synth.problem(fam, prm, n, z, sh, tr, fc, name=f"f{fam}.d{d}.n{n}.m{m}.tr{tr}.fit{fit if isinstance(fit, str) else int(fit)}")


# ------------------------------------------------------------------------------------------------
# S1-S2: residues and coordinates, bit-exact (Eq. 2; reading C-2)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,d", [(7, 2), (11, 2), (55, 2), (1021, 5), (65537, 4), (1048573, 8), (16777213, 12),
                                 (1073741789, 16), (2147483659, 3), (4294967311, 4), (15173222401, 6),
                                 ((1 << 53) - 111, 3)])
def test_points_bit_exact(n, d):
    if n == 55:
        z = np.array([1, 34], dtype=np.uint64)              # Fig. 1
    elif n == 7:
        z = np.array([1, 3], dtype=np.uint64)
    elif n == 11:
        z = np.array([1, 7], dtype=np.uint64)
    else:
        z = synth.korobov_form_vector(n, d, 1 + n // 3)
    rng = synth.MT19937_64(99 + d)
    shift = np.array([rng.uniform() for _ in range(d)])
    shift[0] = 0.0                                           # the unshifted lattice in one dimension
    windows = [(0, min(n, 5000))]
    if n > 5000:
        windows += [(n - 3001, 3001), (n // 2 - 7, 4097)]
    if n > 140000:
        windows += [(rng.next_u64() % (n - 70000), 66000)]
    for k0, cnt in windows:
        r_or, u_or = oracle.lattice_points(n, z, shift, k0, cnt)
        r_g, u_g = binding.qmc_lattice_points(n, z, shift, k0, cnt)
        assert np.array_equal(r_g, r_or), (n, k0)
        assert u_g.tobytes() == u_or.tobytes(), (n, k0)      # memcmp of doubles
        assert u_g.min() >= 0.0 and u_g.max() < 1.0


def test_points_empty_window():
    r, u = binding.qmc_lattice_points(65537, np.array([1, 3], dtype=np.uint64), np.zeros(2), 10, 0)
    assert r.shape == (0, 2) and u.shape == (0, 2)


# ------------------------------------------------------------------------------------------------
# S1-S8: per-shift means, estimate and error for every family x transform x fit
# ------------------------------------------------------------------------------------------------
SIDI, KA = synth.TRANSFORM_SIDI, synth.TRANSFORM_KOROBOV_ASYM


@pytest.mark.parametrize("fam", [0, 1, 2, 3])
@pytest.mark.parametrize("tr", [NONE, BAKER, K + 1, K + 2, K + 3, K + 4, K + 5, K + 6, SIDI + 1, SIDI + 2, SIDI + 3, SIDI + 4, SIDI + 5,
                                SIDI + 6, KA + 16 * 2 + 1, KA + 16 * 5 + 3, KA + 16 * 1 + 4, KA + 16 * 3 + 6, KA + 16 * 4 + 4])
def test_means_all_transforms(fam, tr):
    d = {0: 5, 1: 3, 2: 7, 3: 6}[fam]
    probs = [make(fam, d, 8191, 6, tr, 300 + 10 * fam + tr % 97, fit=False),
             make(fam, d, 8191, 6, tr, 400 + 10 * fam + tr % 97, fit=True)]
    check_against_oracle(probs)


@pytest.mark.parametrize("fam", [4, 5, 6, 7])
@pytest.mark.parametrize("tr", [NONE, BAKER, K + 3, K + 1, SIDI + 2, KA + 16 * 2 + 1])
def test_genz_families_3_to_6(fam, tr):
    """corner peak, Gaussian, C^0, discontinuous (row f-4): every transform kind, with and without fit map"""
    d = {4: 5, 5: 8, 6: 10, 7: 5}[fam]                       # the dimensions of the paper's protocol (L728)
    check_against_oracle([make(fam, d, 8191, 6, tr, 3100 + 13 * fam + tr % 83), make(fam, d, 8191, 6, tr, 3200 + 13 * fam + tr % 83, fit=True),
                          make(fam, d, 8191, 5, tr, 3300 + fam, fit="full")])


@pytest.mark.parametrize("fam,d", [(4, 1), (4, 12), (4, 17), (5, 2), (5, 16), (6, 3), (6, 32), (7, 1), (7, 2), (7, 9), (7, 24)])
def test_genz_families_3_to_6_dimension_slots(fam, d):
    n = 65537 if d <= 16 else 8191
    check_against_oracle([make(fam, d, n, 5, K + 3 if fam in (4, 5) else BAKER, 3400 + 31 * fam + d)])


@pytest.mark.parametrize("fam,d", [(0, 3), (0, 16), (1, 8), (2, 5), (2, 12), (3, 6), (3, 9)])
@pytest.mark.parametrize("tr", [NONE, BAKER, K + 3, K + 2, SIDI + 2])
def test_means_full_fit_map(fam, d, tr):
    """the complete fit function of Eq. 19: two pole terms + cubic, Jacobian p'(y) (row f-2)"""
    p = make(fam, d, 8191, 5, tr, 2100 + 17 * fam + d + tr % 89, fit="full", a_hi=0.6)
    assert binding.qmc_validate_problem_host(p) == 0
    assert np.any(p["fit_coeffs"][:, 2] > 0) or d < 2
    check_against_oracle([p, make(fam, d, 8191, 5, tr, 2200 + d, fit=True, a_hi=0.6)])      # a pole-free problem in the same launch


@pytest.mark.parametrize("fam,d", [(0, 1), (0, 4), (0, 6), (0, 9), (0, 12), (0, 16), (0, 17), (0, 32), (1, 2), (1, 5), (1, 8),
                                   (1, 11), (1, 13), (1, 24), (2, 1), (2, 4), (2, 6), (2, 10), (2, 12), (2, 16), (2, 29),
                                   (3, 1), (3, 3), (3, 5), (3, 6), (3, 8), (3, 11), (3, 16)])
def test_means_all_dimension_slots(fam, d):
    """every register-slot count (4, 6, 8, 12, 16, 32) and dims that leave padded slots; several tiles + ragged tail"""
    n = 65537 if d <= 16 else 8191
    tr = K + 3 if fam != 1 else BAKER
    a_hi = 1.0 if d <= 16 else 0.3
    check_against_oracle([make(fam, d, n, 5, tr, 700 + 31 * fam + d, fit=(d % 2 == 0), a_hi=a_hi)])


@pytest.mark.parametrize("n", [2, 3, 7, 127, 128, 129, 1021, 4099, 65537, 262147, 1048573])
def test_means_lattice_sizes_and_tails(n):
    """n below one CTA, exactly one CTA, ragged tails, and many tiles"""
    z = synth.korobov_form_vector(n, 3, 1 + n // 3) if n > 3 else np.array([1, 1, 1], dtype=np.uint64)
    probs = [make(0, 3, n, 4, K + 3, 900 + n % 89, z=z), make(2, 3, n, 3, BAKER, 901 + n % 89, z=z)]
    check_against_oracle(probs)


@pytest.mark.parametrize("m", [2, 3, 4, 5, 8, 33, 64])
def test_means_shift_counts(m):
    """shift groups: m below, equal to and not a multiple of the group size"""
    check_against_oracle([make(1, 4, 8191, m, BAKER, 1200 + m), make(2, 5, 8191, m, K + 3, 1300 + m)])


@pytest.mark.parametrize("fam,d,m", [(0, 20, 40), (1, 4, 301), (2, 12, 70), (3, 6, 130), (3, 16, 50)])
def test_means_many_shifts_uncached(fam, d, m):
    """more shifts than the shared-memory shift cache holds (768 doubles per CTA): the per-group staging path"""
    n = 2053 if m > 100 else 8191
    check_against_oracle([make(fam, d, n, m, K + 3 if fam != 1 else BAKER, 5100 + d + m, a_hi=0.4)])


def test_maximum_shift_count():
    """m = QMC_MAX_M = 4096 shifts (include/qmc_lattice.h): 1024 groups, 8192 rows in the finalize stage for the complex family"""
    check_against_oracle([make(2, 2, 127, 4096, K + 3, 61), make(0, 3, 257, 4096, BAKER, 62)])


def test_large_mixed_batch_of_all_families():
    """300 small problems of all eight families, mixed transforms / fit modes / sizes in ONE call: every kernel variant's
    queue, the cost-sorted tile lists and the binary search of the tile prefix"""
    rng = synth.MT19937_64(9001)
    trs = [NONE, BAKER, K + 3, K + 1, SIDI + 3, KA + 16 * 2 + 3]
    probs = []
    for i in range(300):
        fam = i % 8
        d = 1 + rng.next_u64() % (6 if fam == 3 else 9)
        n = [127, 509, 1021, 2053, 4099][rng.next_u64() % 5]
        m = 2 + rng.next_u64() % 9
        fit = [False, True, "full"][rng.next_u64() % 3] if i % 5 == 0 else False
        probs.append(make(fam, int(d), n, int(m), trs[rng.next_u64() % len(trs)], 9100 + i, fit=fit, a_hi=0.5))
    check_against_oracle(probs)


def test_wide_residue_path():
    """n >= 2^31 uses 64-bit residue registers; n >= 2^32 needs the 128-bit product (the
    paper ships n = 15173222401).  The oracle can only afford one cheap full run above 2^31, so the 64-bit
    kernels are also driven at small n through qmc_plan_options.force_wide; their results are bit-identical
    to those of the 32-bit kernels."""
    probs = [make(0, 4, 65537, 5, K + 3, 71), make(1, 8, 8191, 5, BAKER, 72), make(2, 12, 8191, 5, K + 3, 73),
             make(3, 6, 8191, 5, K + 3, 74), make(0, 16, 8191, 4, K + 3, 75, fit=True), make(2, 20, 2053, 3, NONE, 76)]
    sms_wide, _, _ = check_against_oracle(probs, force_wide=True)
    sms_narrow, _, _ = run_gpu(probs)
    for a, b, p in zip(sms_wide, sms_narrow, probs):
        if p["dim"] <= 16:                              # dim > 16 always runs the 64-bit kernels
            assert np.array_equal(a, b), p["name"]
    n = 2147483659
    p = make(0, 1, n, 2, K + 3, 77)
    sms, _, _ = run_gpu([p])
    sm_or, _, _ = oracle.integrate(p)
    assert_means(sms[0], sm_or, p["name"])


def test_paper_largest_lattice_full_size():
    """n = 15173222401 > 2^33, the largest lattice the paper ships: 64-bit residues and the 128-bit first
    product of every thread, at full size.  The oracle cannot afford 3e10 evaluations, but in one dimension the residues
    k z mod n are a permutation of 0..n-1 for any z coprime to n, so with the trivial transform the rule is the equispaced
    sum  (1/n) sum_j cos(phi + a (j + theta)/n),  theta = frac(n Delta),  a geometric series with the closed form
    sin(a/2) / (n sin(a/(2n))) * cos(phi + a (theta - 1/2)/n + a/2): an exact value (to rounding) that any wrong or
    repeated residue would miss."""
    from fractions import Fraction
    n, m = 15173222401, 2
    prm = np.array([0.3125, 1.75])                            # u0, a
    sh = np.array([[0.6180339887498949], [0.1415926535897932]])
    z = np.array([5546223817], dtype=np.uint64)               # any z coprime to n
    assert np.gcd(int(z[0]), n) == 1
    p = synth.problem(0, prm, n, z, sh, NONE, name="paper.nmax.d1")
    sms, means, errs = run_gpu([p])
    phi, a = 2 * np.pi * prm[0], prm[1]
    for s_, delta in enumerate(sh[:, 0]):
        theta = float((Fraction(delta) * n) % 1)              # exact: Delta is a dyadic rational
        want = np.sin(a / 2) / (n * np.sin(a / (2 * n))) * np.cos(phi + a * (theta - 0.5) / n + a / 2)
        assert abs(sms[0][s_, 0] - want) <= 1e-13 * abs(want), (sms[0][s_, 0], want)


def test_mixed_batch_one_call():
    """problems of different family, dimension, n, m, transform in one stream-ordered call (S9)"""
    probs = [make(0, 4, 65537, 10, K + 3, 1), make(1, 8, 8191, 5, BAKER, 2), make(2, 12, 4099, 7, K + 3, 3),
             make(3, 6, 16381, 4, K + 3, 4), make(3, 6, 16381, 4, NONE, 5), make(0, 16, 8191, 3, K + 2, 6, fit=True),
             make(1, 3, 1021, 9, K + 1, 7), make(3, 2, 1021, 16, BAKER, 8, fit=True), make(2, 20, 2053, 2, NONE, 9)]
    check_against_oracle(probs)


def test_determinism_bitwise():
    """same inputs twice -> identical bits (fixed result slots; PAPER.md L883 motivates reproducibility)"""
    probs = synth.config(3, n_override=65537, count_override=24) + [make(2, 12, 65537, 8, K + 3, 5)]
    a = run_gpu(probs)
    b = run_gpu(probs)
    for x, y in zip(a[0], b[0]):
        assert x.tobytes() == y.tobytes()
    assert a[1].tobytes() == b[1].tobytes() and a[2].tobytes() == b[2].tobytes()


def test_cuda_graph_replay_is_bitwise_the_direct_call():
    """a single-problem call is stream-ordered and capturable: graph replays reproduce the direct call bit for bit"""
    p = make(2, 12, 65537, 8, K + 3, 4711)
    direct = run_gpu([p])
    batch = binding.DeviceBatch([p])
    graph = batch.capture()
    batch.means.zero_(); batch.errs.zero_(); batch.shift_means.zero_()
    for _ in range(3):
        graph.replay()
    sms, means, errs = batch.results()
    assert sms[0].tobytes() == direct[0][0].tobytes()
    assert means.tobytes() == direct[1].tobytes() and errs.tobytes() == direct[2].tobytes()


def test_minimal_example_one_eighth():
    """Fig. 2: f = x0 x1 x2, Korobov weight 3 -> 1/8, through the synchronous HOST entry."""
    d = 3
    prm = np.array([0, 0, 1, 1, 1, 1, 1, 1.0, 0, 0, 0, 1.0, 0, 0, 0], dtype=np.float64)   # a=b=0, U=F=1, nu=(1,1,1)
    rng = synth.MT19937_64(5)
    sh = synth.draw_shifts(rng, 8, d)
    z = synth.korobov_form_vector(65537, d, 25016)
    mean, err = binding.qmc_lattice_integrate(3, prm, d, 65537, z, sh, 8, K + 3)
    assert abs(mean[0] - 0.125) < 1e-9 and err[0] < 1e-9
    p = synth.problem(3, prm, 65537, z, sh, K + 3)
    sm_or, mean_or, err_or = oracle.integrate(p)
    sm, mean2, err2 = binding.qmc_lattice_integrate_ex(p)
    assert_means(sm, sm_or, "fig2")
    assert mean2[0] == mean[0] and err2[0] == err[0]


def test_synchronous_entry_nonfinite_status():
    """F without constant term and an unshifted first coordinate: f(0) = 1/0 -> QMC_ERR_NONFINITE, results written"""
    d = 2
    prm = np.array([0, 1, 1, 1, 0, 0, 1.0, 0, 0, 1.0, 1, 0], dtype=np.float64)            # U = 1, F = x0, b = 1
    sh = np.array([[0.0, 0.25], [0.0, 0.5]])
    with pytest.raises(binding.QmcError) as e:
        binding.qmc_lattice_integrate(3, prm, d, 1021, np.array([1, 5], dtype=np.uint64), sh, 2, NONE)
    assert e.value.status == binding.QMC_ERR_NONFINITE


def test_finalize_stage_hand_made():
    """Eq. 3 on Q_s = 1..m: err = sqrt((m+1)/12); device finalize vs closed form and oracle"""
    for m in (2, 10, 33):
        q = np.arange(1, m + 1, dtype=np.float64)
        mean, err = binding.qmc_finalize_means(q)
        assert abs(mean[0] - (m + 1) / 2) < 1e-14 and abs(err[0] - np.sqrt((m + 1) / 12.0)) < 1e-14
    rng = np.random.default_rng(1)
    q = 3.0 + 1e-9 * rng.standard_normal((32, 2))
    mean, err = binding.qmc_finalize_means(q)
    mean_or, err_or = oracle.finalize(q)
    np.testing.assert_allclose(err, err_or, rtol=1e-12)
    np.testing.assert_allclose(mean, mean_or, rtol=1e-15)


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs
# ------------------------------------------------------------------------------------------------
def test_config0_full():
    check_against_oracle(synth.config(0))


def test_config1_full():
    check_against_oracle(synth.config(1))


def test_config3_reduced_batch():
    """256 sectors at an oracle-friendly lattice: same parameters, same persistent-grid tile queue"""
    check_against_oracle(synth.config(3, n_override=8191))


def test_config4_reduced_with_nontrivial_fit():
    p = synth.config(4, n_override=1048573)[0]
    p = dict(p, fit_coeffs=synth.cubic_fit_coeffs(16, a4=0.6, a5=0.3), name="cfg4.n1048573.fit")
    check_against_oracle([p])


def _golden():
    if not os.path.exists(GOLDEN):
        pytest.skip("tests/golden/fullsize_oracle.json not generated")
    with open(GOLDEN) as f:
        return json.load(f)


def _golden_arrays(rec, nc):
    un = lambda xs: np.array([float.fromhex(x) for x in xs])
    return un(rec["shift_means"]).reshape(-1, nc), un(rec["mean"]), un(rec["err"])


def _check_full(p, rec):
    nc = oracle.ncomp(p["family"])
    sm_or, mean_or, err_or = _golden_arrays(rec, nc)
    assert rec["n"] == p["n"] and rec["m"] == p["m"] and rec["dim"] == p["dim"]
    sms, means, errs = run_gpu([p])
    assert_means(sms[0], sm_or, p["name"] + " (full size)")
    assert_err(errs[0, :nc], err_or, sm_or, p["name"])
    _, err_st = oracle.finalize(sms[0])
    np.testing.assert_allclose(errs[0, :nc], err_st, rtol=1e-12)


def test_config2_full_size_vs_stored_oracle():
    g = _golden()
    if "2" not in g:
        pytest.skip("config 2 not in golden file")
    _check_full(synth.config(2)[0], g["2"])


def test_config3_full_size_all_sectors():
    """the full 256-sector batch in bench.py's launch configuration: EVERY sector against the oracle's stored full-size record"""
    g = _golden()
    if "3" not in g:
        pytest.skip("config 3 not in golden file")
    probs = synth.config(3)
    assert sorted(int(k) for k in g["3"]["sectors"]) == list(range(len(probs))), "the golden file must hold every sector of configs[3]"
    sms, means, errs = run_gpu(probs)
    for key, rec in g["3"]["sectors"].items():
        i = int(key)
        assert rec["n"] == probs[i]["n"] and rec["m"] == probs[i]["m"] and rec["dim"] == probs[i]["dim"]
        sm_or, mean_or, err_or = _golden_arrays(rec, 1)
        assert_means(sms[i], sm_or, probs[i]["name"] + " (full size)")
        assert_err(errs[i, :1], err_or, sm_or, probs[i]["name"])
    # properties that hold for every sector: positive integrand -> positive means; finite; err consistent
    for i in range(len(probs)):
        assert np.all(np.isfinite(sms[i])) and np.all(sms[i] > 0)
        _, err_st = oracle.finalize(sms[i])
        np.testing.assert_allclose(errs[i, :1], err_st, rtol=1e-12)


def test_config4_full_size_vs_stored_oracle():
    g = _golden()
    if "4" not in g:
        pytest.skip("config 4 not in golden file")
    rec = g["4"]
    fit = np.array([float.fromhex(x) for x in rec["fit_coeffs"]]).reshape(16, 6)
    p = dict(synth.config(4)[0], fit_coeffs=fit)
    _check_full(p, rec)


# ------------------------------------------------------------------------------------------------
# S10: projection pass and fit (Eq. 20; reading C-8)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("fam,d,n,bins", [(0, 16, 65537, 256), (1, 8, 65537, 256), (2, 12, 16381, 64), (3, 6, 16381, 256),
                                          (4, 5, 8191, 128), (5, 8, 8191, 128), (6, 10, 8191, 256), (7, 5, 8191, 64),
                                          (1, 5, 8191, 1024), (0, 32, 4099, 1024), (1, 2, 127, 2)])
def test_projection_histogram(fam, d, n, bins):
    p = make(fam, d, n, 2, NONE, 1500 + fam + d)
    H_or = oracle.project(p, bins)
    batch = binding.DeviceBatch([p])
    H = batch.project(0, bins).cpu().numpy()
    assert H.shape == H_or.shape
    np.testing.assert_allclose(H, H_or, rtol=1e-12, atol=0)
    assert np.array_equal(H == 0.0, H_or == 0.0)            # bin membership is decided by bit-exact coordinates
    H2 = batch.project(0, bins).cpu().numpy()
    assert H.tobytes() == H2.tobytes()                       # deterministic
    np.testing.assert_allclose(binding.qmc_fit_cubic(H), oracle.fit_cubic(H_or), rtol=0, atol=1e-9)


def test_config4_projection_and_fit():
    """the projection pass of configs[4]: n_fit = 1048573, d = 16, 256 bins; against the live oracle and, when
    present, the stored full-size record"""
    p = synth.config(4)[0]
    proj = dict(p, n=synth.CONFIG4_NFIT, z=synth.genvec(synth.CONFIG4_NFIT, 16), transform=NONE)
    H_or = oracle.project(proj, synth.PROJECTION_BINS)
    H = binding.DeviceBatch([proj]).project(0, synth.PROJECTION_BINS).cpu().numpy()
    np.testing.assert_allclose(H, H_or, rtol=1e-12, atol=0)
    fit_gpu, fit_or = binding.qmc_fit_cubic(H), oracle.fit_cubic(H_or)
    np.testing.assert_allclose(fit_gpu, fit_or, rtol=0, atol=1e-9)
    if os.path.exists(GOLDEN):
        g = json.load(open(GOLDEN))
        if "4" in g:
            stored = np.array([float.fromhex(x) for x in g["4"]["fit_coeffs"]]).reshape(16, 6)
            assert stored.tobytes() == fit_or.tobytes()


def test_projection_to_full_fit_to_integration():
    """row f-2 end to end: device projection pass (Eq. 20) -> qmc_fit_polysingular (Eq. 19, bounds PAPER.md L231) -> fused
    integration with the fitted map; the fitted coefficients are an input of both sides, so parity holds at the usual bars,
    and for this peaked integrand the fitted map reduces the error estimate (the purpose of section 2.4)"""
    d, n = 3, 16381
    rng = synth.MT19937_64(31337)
    prm = np.array([9.0, 7.0, 8.0] + [0.02, 0.97, 0.03])                               # narrow peaks at the boundary
    sh = synth.draw_shifts(rng, 8, d)
    z = synth.korobov_form_vector(n, d, 1 + n // 3)
    base = synth.problem(1, prm, n, z, sh, BAKER, name="peaked")
    H = binding.DeviceBatch([dict(base, transform=NONE)]).project(0, 256).cpu().numpy()
    fit = binding.qmc_fit_polysingular(H)
    assert np.any(fit[:, 2:4] > 0)                          # the pole terms are used for this integrand
    fitted = dict(base, fit_coeffs=fit, name="peaked.fitted")
    assert binding.qmc_validate_problem_host(fitted) == 0
    sms, means, errs = check_against_oracle([base, fitted])
    cc, w = prm[:d], prm[d:]
    exact = np.prod(cc * (np.arctan(cc * (1 - w)) + np.arctan(cc * w)))                # Genz product peak
    for i in range(2):
        assert abs(means[i, 0] - exact) <= 6 * errs[i, 0]
    assert errs[1, 0] < 0.2 * errs[0, 0]                    # (the CPU experiment behind this test saw a factor 40)


# ------------------------------------------------------------------------------------------------
# boundary behaviour on the device
# ------------------------------------------------------------------------------------------------
def test_workspace_errors():
    import torch
    p = make(0, 4, 8191, 4, K + 3, 1)
    b = binding.DeviceBatch([p])
    L = binding.lib()
    s = torch.cuda.current_stream().cuda_stream
    st = L.qmc_lattice_integrate_batch(1, b.arr, b.means.data_ptr(), b.errs.data_ptr(), None, b.ws_ptr, b.ws_bytes - 1, s)
    assert st == -11
    st = L.qmc_lattice_integrate_batch(1, b.arr, b.means.data_ptr(), b.errs.data_ptr(), None, b.ws_ptr + 8, b.ws_bytes, s)
    assert st == -11
    st = L.qmc_lattice_integrate_batch(1, b.arr, None, b.errs.data_ptr(), None, b.ws_ptr, b.ws_bytes, s)
    assert st == -1
    st = L.qmc_lattice_integrate_batch(1, b.arr, b.means.data_ptr(), b.errs.data_ptr(), None, b.ws_ptr, b.ws_bytes, s)
    assert st == 0                                          # out_shift_means may be NULL
    torch.cuda.synchronize()
    sm_or, mean_or, _ = oracle.integrate(p)
    assert abs(b.means.cpu().numpy()[0, 0] - mean_or[0]) <= 1e-13 * abs(mean_or[0])


# ------------------------------------------------------------------------------------------------
# log factors of the sector family: f (lu log U + lf log F)^p (reading C-15)
# ------------------------------------------------------------------------------------------------
def make_log(d, n, m, tr, seed, fit=False, pw=None):
    p = make(3, d, n, m, tr, seed, fit=fit)
    rng = synth.MT19937_64(seed)
    prm = synth.sector_log(rng, d)                            # the same leading block as make() draws + [lu, lf, p]
    assert np.array_equal(prm[:-3], p["params"])
    if pw is not None:
        prm[-1] = float(pw)
    return dict(p, params=prm, name=p["name"] + f".log{int(prm[-1])}")


@pytest.mark.parametrize("d", [1, 3, 4, 6, 8, 9, 16])
@pytest.mark.parametrize("tr,fit", [(K + 3, False), (K + 3, True), (NONE, False), (BAKER, "full"), (SIDI + 2, False), (KA + 16 * 2 + 1, True)])
def test_sector_log_factor_means(d, tr, fit):
    probs = [make_log(d, 8191, 6, tr, 2600 + d, fit=fit, pw=pw) for pw in (1, 2, 3, 4)]
    check_against_oracle(probs)


def test_sector_log_factor_in_a_mixed_batch_and_tails():
    """plain and log sectors of several sizes share one launch; the log factor of one problem never leaks into the next"""
    probs = []
    for i, n in enumerate([127, 1021, 4099, 65537, 262147]):
        probs.append(make(3, 6, n, 5, K + 3, 2700 + i))
        probs.append(make_log(6, n, 5, K + 3, 2700 + i))
        probs.append(make(3, 6, n, 5, K + 3, 2750 + i))
    sms, _, _ = check_against_oracle(probs)
    assert not np.array_equal(sms[0], sms[1])


def test_sector_log_factor_many_shifts():
    check_against_oracle([make_log(6, 4099, 130, K + 3, 2800), make_log(16, 4099, 50, K + 3, 2801, fit=True)])


def test_sector_log_factor_projection():
    p = make_log(6, 16381, 2, NONE, 2810)
    H_or = oracle.project(p, 128)
    H = binding.DeviceBatch([p]).project(0, 128).cpu().numpy()
    np.testing.assert_allclose(H, H_or, rtol=1e-12, atol=0)
    H_plain = oracle.project(dict(p, params=p["params"][:-3]), 128)
    assert not np.allclose(H_or, H_plain)


def test_sector_log_factor_arguments_outside_the_series():
    """the kernel's own logarithm serves normal positive arguments; a subnormal U takes the library routine (same bar), and a
    negative U gives NaN on both sides (include/qmc_lattice.h: U, F > 0 is the caller's responsibility)"""
    n, d = 1021, 2
    rng = synth.MT19937_64(2830)
    z, sh = synth.korobov_form_vector(n, d, 341), synth.draw_shifts(rng, 4, d)

    def prob(cU0, name):
        # U = cU0 (constant), F = 2 + x0 + 0.5 x1, a = 0, b = 1, nu = (1, 0); log factor (log U + 0.5 log F)^2
        prm = [0, 1, 1, 3, 1, 0, cU0, 0, 0, 2.0, 1.0, 0.5, 0, 0, 1, 0, 0, 1, 1.0, 0.5, 2]
        return synth.problem(3, np.array(prm, dtype=np.float64), n, z, sh, K + 3, name=name)

    probs = [prob(1e-310, "subnormal U"), prob(3.0, "normal U"), prob(-1.0, "negative U")]
    sms, means, errs = run_gpu(probs)
    for i in (0, 1):
        sm_or, _, err_or = oracle.integrate(probs[i])
        assert np.all(np.isfinite(sm_or))
        assert_means(sms[i], sm_or, probs[i]["name"])
        assert_err(errs[i, :1], err_or, sm_or, probs[i]["name"])
    assert np.all(np.isnan(oracle.integrate(probs[2])[0])) and np.all(np.isnan(sms[2]))


def test_sector_log_factor_bad_power_yields_nan():
    good = make_log(3, 1021, 3, K + 3, 2820)
    bad = dict(good, params=good["params"].copy(), name="bad")
    bad["params"][-1] = 5.0                                  # p outside 1..4
    sms, _, _ = run_gpu([good, bad])
    sm_or, _, _ = oracle.integrate(good)
    assert_means(sms[0], sm_or, "good")
    assert np.all(np.isnan(sms[1]))


def test_bad_sector_block_yields_nan_not_garbage():
    """a parameter block the device-side compiler rejects (exponent > 8) poisons that problem's results only"""
    good = make(3, 3, 1021, 3, K + 3, 11)
    bad = dict(good, params=good["params"].copy(), name="bad")
    d = 3
    nU = int(bad["params"][2])
    bad["params"][4 + d + nU + d] = 9.0                      # exponent of U's second monomial, first variable
    sms, means, errs = run_gpu([good, bad])
    sm_or, _, _ = oracle.integrate(good)
    assert_means(sms[0], sm_or, "good")
    assert np.all(np.isnan(sms[1]))


def test_fp64_peak_probe_sane():
    rate, ms = binding.qmc_fp64_peak_probe(4000)
    assert 1e12 < rate < 4e13 and ms > 0


# ------------------------------------------------------------------------------------------------
# sector family: the device-side compiler and its program (qmc_sector_compile), the HOST-pointer batch entry
# ------------------------------------------------------------------------------------------------
def _interpret(steps, slots, c0, x):
    """the machine of gen_sector_interp.py / include/qmc_lattice.h, in Python: -> (U(x), F(x))"""
    S, A, si, out = c0[0], 0.0, 0, []
    for code in steps:
        if code == 0:
            continue
        if code == 2:
            break
        if code == 1:
            out.append(S); S = slots[si][0]; si += 1
            continue
        j, kind = divmod(int(code) - 3, 5)
        if kind == 0: S = A * x[j] + S
        elif kind == 1: S = slots[si][0] * x[j] + S; si += 1
        elif kind == 2: A = slots[si][0] * x[j] + A; si += 1
        elif kind == 3: A = slots[si][0] * x[j] + slots[si][1]; si += 1
        else: A = A * x[j]
    out.append(S)
    return out


def _sector_polys(p):
    prm, d = p["params"], p["dim"]
    nU, nF = int(prm[2]), int(prm[3])
    off, out = 4 + d, []
    for cnt in (nU, nF):
        out.append((prm[off:off + cnt], prm[off + cnt:off + cnt + cnt * d].reshape(cnt, d)))
        off += cnt * (1 + d)
    return out


def test_sector_programs_evaluate_their_polynomials():
    """Every program the device-side compiler makes of configs[3]'s 256 sectors, run by a Python model of the machine,
    reproduces U and F as written (sum of coefficient times monomial) at random points; the mean program length is the
    30.61 steps DESIGN.md and bench.py quote (the flat monomial-by-monomial count is sum of degrees = 44.44)."""
    rng = np.random.default_rng(7)
    lengths, flat = [], []
    for p in synth.config(3):
        steps, slots, c0 = binding.qmc_sector_compile(p["params"], p["dim"])
        x = rng.random(p["dim"])
        got = _interpret(steps, slots, c0, x)
        polys = _sector_polys(p)
        for (c, e), g in zip(polys, got):
            want = float(np.sum(c * np.prod(x[None, :] ** e, axis=1)))
            assert abs(g - want) <= 1e-14 * abs(want), p["name"]
        lengths.append(int(np.sum(steps >= 3)))
        flat.append(int(sum(e.sum() for _, e in polys)))
    assert abs(np.mean(flat) - 44.4375) < 1e-9
    assert abs(np.mean(lengths) - 30.61) < 0.01, np.mean(lengths)


def test_sector_compiler_limits():
    """the largest block the header allows (64 + 64 monomials of total degree 16 in 16 variables) compiles and integrates;
    repeated and high powers take the multiply steps"""
    rng = synth.MT19937_64(4242)
    d = 16
    def poly(cnt):
        c = np.array([rng.uniform_range(0.5, 2.0) for _ in range(cnt)])
        e = np.zeros((cnt, d))
        for t in range(1, cnt):
            for _ in range(16):
                j = rng.next_u64() % d
                if e[t, j] < 8: e[t, j] += 1
        return c, e
    cu, eu = poly(64); cf, ef = poly(64)
    prm = np.concatenate([[1, 1, 64, 64], np.zeros(d), cu, eu.ravel(), cf, ef.ravel()])
    steps, slots, c0 = binding.qmc_sector_compile(prm, d)
    x = np.array([0.3 + 0.04 * j for j in range(d)])
    U, F = _interpret(steps, slots, c0, x)
    assert abs(U - np.sum(cu * np.prod(x[None, :] ** eu, axis=1))) <= 1e-13 * abs(U)
    assert abs(F - np.sum(cf * np.prod(x[None, :] ** ef, axis=1))) <= 1e-13 * abs(F)
    p = synth.problem(3, prm, 1021, synth.genvec(1021, 16), synth.draw_shifts(rng, 4, d), K + 3, name="sector.max")
    check_against_oracle([p])


def test_host_pointer_batch_entry():
    """qmc_lattice_integrate_batch_host: mixed families in one synchronous call, bit-identical to the device-pointer entry"""
    probs = [make(3, 6, 8191, 16, K + 3, 9300 + i) for i in range(5)] + [make(1, 8, 8191, 7, BAKER, 9310), make(2, 12, 4099, 3, K + 3, 9311),
                                                                        make(0, 16, 4099, 4, K + 3, 9312, fit=True)]
    sms_h, means_h, errs_h = binding.qmc_lattice_integrate_batch_host(probs)
    sms_d, means_d, errs_d = run_gpu(probs)
    for a, b in zip(sms_h, sms_d):
        assert np.array_equal(a, b)
    assert np.array_equal(means_h, means_d) and np.array_equal(errs_h, errs_d)
    sm1, mean1, err1 = binding.qmc_lattice_integrate_ex(probs[5])
    assert np.array_equal(sm1, sms_d[5]) and mean1[0] == means_d[5, 0]
    binding.qmc_release_thread_resources()
    sms_h2, _, _ = binding.qmc_lattice_integrate_batch_host(probs[:2])       # the arena is rebuilt on demand
    assert np.array_equal(sms_h2[0], sms_d[0])


def test_projection_rejects_a_malformed_sector_block():
    """the projection pass validates a sector block on the device before it reads an exponent: NaN histograms,
    no out-of-range read; the struct-level limits are those of the integration entries"""
    p = make(3, 6, 4099, 2, NONE, 9400)
    bad = dict(p, params=p["params"].copy())
    bad["params"][4 + 6 + int(p["params"][2]) + 3] = 40.0          # an exponent out of range
    H = binding.DeviceBatch([bad]).project(0, 64).cpu().numpy()
    assert np.all(np.isnan(H))
    bad2 = dict(p, params=p["params"].copy())
    bad2["params"][2] = 3.0                                          # nU inconsistent with n_params
    H2 = binding.DeviceBatch([bad2]).project(0, 64).cpu().numpy()
    assert np.all(np.isnan(H2))
    good = binding.DeviceBatch([p]).project(0, 64).cpu().numpy()
    assert np.all(np.isfinite(good))


# ------------------------------------------------------------------------------------------------
# family 8: sector polynomials with complex coefficients (contour-deformed shape, reading C-16)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d", [1, 2, 3, 4, 5, 6, 7, 8, 11, 16])
def test_complex_sector_all_slot_counts(d):
    """every dimension-slot variant of the complex sector kernels (4 / 6 / 8 / 16 slots; groups of 4 or 2 shifts), m not a
    multiple of the group, against the oracle at 1e-13 of the modulus"""
    check_against_oracle([make(8, d, 8191, 7, K + 3, 9500 + d), make(8, d, 4099, 2, K + 3, 9520 + d)])


@pytest.mark.parametrize("tr,fit", [(NONE, False), (BAKER, False), (K + 1, False), (K + 3, True), (K + 3, "full"), (SIDI + 2, False),
                                    (KA + 16 * 2 + 1, True)])
def test_complex_sector_transforms_and_fit(tr, fit):
    check_against_oracle([make(8, 6, 8191, 9, tr, 9540 + tr % 89, fit=fit), make(8, 3, 8191, 5, tr, 9560 + tr % 89, fit=fit)])


def test_complex_sector_log_factors_and_mixed_batch():
    """principal-branch log factors (p = 1..3) and a batch mixing both sector families with closed-form ones"""
    rng = synth.MT19937_64(9580)
    probs = []
    for i, d in enumerate((2, 4, 6, 6, 8)):
        prm = synth.sector_complex(rng, d, log_block=True)
        probs.append(synth.problem(8, prm, 8191, synth.korobov_form_vector(8191, d, 2731), synth.draw_shifts(rng, 6, d), K + 3,
                                   name=f"csector.log.d{d}"))
    probs += [make(3, 6, 8191, 16, K + 3, 9590), make(8, 6, 8191, 16, K + 3, 9591), make(2, 12, 4099, 4, K + 3, 9592),
              make(1, 8, 4099, 5, BAKER, 9593)]
    check_against_oracle(probs)


def test_complex_sector_contour_deformation_value():
    """the Cauchy pin of the oracle, end to end on the GPU: the deformed one- and two-dimensional integrals keep their real
    values for every lambda"""
    c = 0.7
    rng = synth.MT19937_64(9600)
    def block(a, b, nu, U, F):
        d = len(nu)
        out = [float(a), float(b), float(len(U)), float(len(F))] + [float(v) for v in nu]
        for poly in (U, F):
            out += [complex(cc).real for cc, _ in poly] + [complex(cc).imag for cc, _ in poly]
            for _, e in poly:
                out += [float(v) for v in e]
        return np.array(out)
    for lam in (0.0, 0.6, 2.0):
        prm = block(1, 2, [0, 0], [(1.0 - 1j * lam, (0, 0)), (2j * lam, (1, 0))],
                    [(c, (0, 0)), (1.0 - 1j * lam, (1, 0)), (1j * lam, (2, 0)), (1.0, (0, 1))])
        p = synth.problem(8, prm, 1048573, synth.genvec(1048573, 8)[:2], synth.draw_shifts(rng, 8, 2), K + 3, name=f"cauchy.lam{lam}")
        sms, means, errs = check_against_oracle([p])
        exact = np.log((c + 1.0) ** 2 / (c * (c + 2.0)))
        assert abs(means[0, 0] - exact) < 1e-9 and abs(means[0, 1]) < 1e-9


def test_complex_sector_projection_and_adaptive():
    """projection histogram of |f| (modulus) against the oracle; qmc_integrate with both error modes ends on the oracle's (n, m)"""
    p = make(8, 5, 8191, 2, NONE, 9610)
    H_or = oracle.project(p, 128)
    H = binding.DeviceBatch([p]).project(0, 128).cpu().numpy()
    assert np.all(np.abs(H - H_or) <= 1e-12 * np.maximum(np.abs(H_or), 1e-300))
    q = make(8, 4, 8191, 8, K + 3, 9611)
    ln, lz = synth.ladder(4, 65521)
    for errormode in (0, 1):
        res, st = binding.qmc_integrate(8, q["params"], 4, K + 3, ln, lz, q["shifts"], min_n=1000, min_m=8, epsrel=1e-6, epsabs=0.0,
                                        maxeval=10 ** 9, errormode=errormode)
        i = list(ln).index(res["n"])
        ref = synth.problem(8, q["params"], res["n"], lz[i], q["shifts"][:res["m"]], K + 3)
        sm_or, mean_or, err_or = oracle.integrate(ref)
        assert np.all(np.abs(res["integral"] - mean_or) <= 1e-13 * np.hypot(*mean_or))


# ------------------------------------------------------------------------------------------------
# S10b: the paper's sort-based CDF sampling without a sort (reading C-8b)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("fam,d,n,step", [(0, 16, 65537, 10), (1, 8, 65537, 10), (2, 12, 16381, 7), (3, 6, 16381, 10), (8, 6, 8191, 10),
                                          (4, 5, 8191, 3), (5, 8, 8191, 1), (1, 2, 127, 5), (7, 5, 1021, 1021), (0, 32, 4099, 10),
                                          (1, 3, 1048573, 10)])
def test_cdf_samples_match_the_oracle_sort(fam, d, n, step):
    """kept coordinates bit-exact (the lattice's cyclic residue order IS the sorted order), CDF values at 1e-12, twice the same bits"""
    p = make(fam, d, n, 2, NONE, 9700 + fam + d)
    x_or, c_or = oracle.cdf_samples(p, step)
    batch = binding.DeviceBatch([p])
    x, c = batch.cdf_samples(0, step)
    x, c = x.cpu().numpy(), c.cpu().numpy()
    assert x.shape == x_or.shape == (d, n // step)
    assert x.tobytes() == x_or.tobytes()
    assert np.all(np.abs(c - c_or) <= 1e-12 * c_or)
    x2, c2 = batch.cdf_samples(0, step)
    assert c2.cpu().numpy().tobytes() == c.tobytes()


def test_cdf_samples_shift_edge_cases():
    """shift 0 (nothing wraps), a shift just below 1 (almost everything wraps) and the paper's n = 55 lattice of Fig. 1"""
    for n, z, sh in [(55, [1, 34], [0.0, 0.999999]), (1021, [1, 374], [1e-300, 0.5]), (8191, [1, 2731], [0.25, 1.0 - 2.0 ** -53])]:
        p = synth.problem(1, np.array([2.0, 3.0, 0.3, 0.6]), n, z, np.array([sh, sh]), NONE)
        x_or, c_or = oracle.cdf_samples(p, 5)
        x, c = binding.DeviceBatch([p]).cdf_samples(0, 5)
        assert x.cpu().numpy().tobytes() == x_or.tobytes()
        assert np.all(np.abs(c.cpu().numpy() - c_or) <= 1e-12 * c_or)


def test_fit_from_cdf_samples():
    """cubic fit from the sampled pairs against the oracle's (same closed form on the same pairs), and the projection -> fit ->
    integration chain with the sort-based samples: the error estimate of a boundary-peaked integrand drops"""
    p = make(1, 4, 65537, 8, K + 3, 9750)
    proj = dict(p, transform=NONE)
    x, c = binding.DeviceBatch([proj]).cdf_samples(0, 10)
    x, c = x.cpu().numpy(), c.cpu().numpy()
    fit = binding.qmc_fit_from_cdf(x, c)
    fit_or = oracle.fit_cubic_cdf(x, c)
    assert np.allclose(fit, fit_or, rtol=0, atol=1e-10)
    full = binding.qmc_fit_from_cdf(x, c, with_poles=True)
    assert binding.qmc_validate_problem_host(dict(p, fit_coeffs=full)) == 0
    _, _, err0 = run_gpu([p])
    _, _, err1 = run_gpu([dict(p, fit_coeffs=full)])
    assert err1[0, 0] < err0[0, 0]
    check_against_oracle([dict(p, fit_coeffs=full, name="cdf-fit")])


# ------------------------------------------------------------------------------------------------
# specialised sector kernels (qmc_sector_module_*): the sectors of a batch as compiled straight-line code,
# PAPER.md L427-L438 (the paper compiles every integrand); the interpreting kernel is the default
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d", [1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16])
def test_module_means_against_the_oracle(d):
    """every dimension-slot kind (4, 6, 8, 16), ragged tile tails, several sectors per kernel and one per kernel"""
    probs = [make(3, d, n, 5, K + 3, 9800 + 7 * d + i) for i, n in enumerate([127, 1021, 8191, 65537])]
    for per_kernel in (0, 1):
        mod = binding.SectorModule(probs, per_kernel)
        assert mod.info["specialised"] == 4 and mod.info["kernels"] == (4 if per_kernel else 1)
        check_against_oracle(probs, module=mod)
        mod.close()


@pytest.mark.parametrize("d", [3, 6, 8, 13])
def test_module_returns_the_bits_of_the_interpreting_kernel(d):
    """one problem per call: both routes tile alike, evaluate the same operations in the same order and must agree in every bit
    (with and without a log factor, whose U goes through shared memory on both routes)"""
    for p in (make(3, d, 262147, 9, K + 3, 9850 + d), make_log(d, 65537, 6, K + 3, 9860 + d, pw=2)):
        mod = binding.SectorModule([p])
        a = run_gpu([p])
        b = run_gpu([p], module=mod)
        assert a[0][0].tobytes() == b[0][0].tobytes() and a[1].tobytes() == b[1].tobytes() and a[2].tobytes() == b[2].tobytes()


@pytest.mark.parametrize("d", [1, 3, 4, 5, 6, 8, 9, 16])
def test_module_complex_sectors(d):
    """family 8 (reading C-16) through specialised kernels: oracle parity on every slot kind, with log factors (principal branch),
    and the bits of the interpreting kernel where the arithmetic is written with explicit roundings (no log factor)"""
    probs = [make(8, d, n, 5, K + 3, 9970 + 5 * d + i) for i, n in enumerate([127, 1021, 8191])]
    rng = synth.MT19937_64(9990 + d)
    logp = synth.problem(8, synth.sector_complex(rng, d, log_block=True), 4099, synth.korobov_form_vector(4099, d, 1 + 4099 // 3),
                         synth.draw_shifts(rng, 4, d), K + 3, name=f"csector.log.d{d}")
    mod = binding.SectorModule(probs + [logp])
    assert mod.info["specialised"] == 4 and mod.info["kernels"] == 1
    check_against_oracle(probs + [logp], module=mod)
    one = make(8, d, 65537, 6, K + 3, 9980 + d)
    a = run_gpu([one])
    b = run_gpu([one], module=binding.SectorModule([one]))
    assert a[0][0].tobytes() == b[0][0].tobytes() and a[1].tobytes() == b[1].tobytes() and a[2].tobytes() == b[2].tobytes()


def test_module_mixed_batch_routes_only_what_it_covers():
    """closed-form families, other transforms, fit maps and a rejected block stay on the default kernels in the same call;
    a and b = 0, nu up to 8, log factors and complex sectors run specialised"""
    probs = [make(3, 6, 8191, 5, K + 3, 9900), make(0, 5, 4099, 4, K + 3, 9901), make(8, 4, 4099, 4, K + 3, 9902),
             make(3, 6, 8191, 5, BAKER, 9903), make(3, 4, 8191, 5, K + 3, 9904, fit=True), make(3, 6, 8191, 5, K + 2, 9905),
             make_log(6, 8191, 5, K + 3, 9906, pw=3), make_log(8, 4099, 4, K + 3, 9907, pw=4), make(3, 16, 4099, 4, K + 3, 9908)]
    zero_powers = make(3, 5, 8191, 5, K + 3, 9909)
    prm = zero_powers["params"].copy()
    prm[0] = prm[1] = 0.0                                    # a = b = 0: the integrand is the monomial alone
    prm[4:9] = [8.0, 0.0, 3.0, 1.0, 0.0]
    probs.append(dict(zero_powers, params=prm, name="a=b=0"))
    bad = make(3, 6, 8191, 5, K + 3, 9910)
    prm = bad["params"].copy()
    prm[4 + 6 + int(prm[2])] = 2.5                           # a fractional exponent in U
    bad = dict(bad, params=prm, name="bad")
    mod = binding.SectorModule(probs + [bad])
    assert mod.info["specialised"] == 9                      # every sector but the rejected one (routing is decided per call)
    sms, means, errs = run_gpu(probs + [bad], module=mod)
    assert np.isnan(means[-1, 0]) and np.isnan(errs[-1, 0])
    ref = run_gpu(probs + [bad])
    assert np.isnan(ref[1][-1, 0])
    for i, p in enumerate(probs):
        sm_or, mean_or, err_or = oracle.integrate(p)
        assert_means(sms[i], sm_or, p["name"])
        assert_err(errs[i, :sm_or.shape[1]], err_or, sm_or, p["name"])


def test_module_serves_other_lattices_and_rejects_other_batches():
    """the module depends on the integrands only: new n, z, shifts and m reuse it; a batch of another shape is refused"""
    probs = [make(3, 6, 4099, 4, K + 3, 9950 + i) for i in range(5)]
    mod = binding.SectorModule(probs)
    other = [dict(make(3, 6, 65537, 7, K + 3, 9950 + i), name=f"relattice{i}") for i in range(5)]
    for a, b in zip(probs, other):
        assert np.array_equal(a["params"], b["params"])
    check_against_oracle(other, module=mod)
    with pytest.raises(binding.QmcError):
        binding.DeviceBatch(probs[:4], module=mod)           # count differs: the workspace query fails
    swapped = [probs[0], make(3, 5, 4099, 4, K + 3, 9960)] + probs[2:]
    with pytest.raises(binding.QmcError):
        binding.DeviceBatch(swapped, module=mod)


def test_module_config3_full_size():
    """BASELINE.json configs[3] at full size through the specialised kernels, bench.py's second launch configuration for that
    workload: EVERY sector against the oracle's stored full-size record"""
    g = _golden()
    probs = synth.config(3)
    mod = binding.SectorModule(probs)
    assert mod.info["specialised"] == 256 and mod.info["kernels"] == 8
    batch = binding.DeviceBatch(probs, module=mod)
    assert batch.integrate() == 1 + 8 + 1                    # prepare, one launch per kernel of the module, finalize
    sms, means, errs = batch.results()
    for key, rec in g["3"]["sectors"].items():
        i = int(key)
        sm_or, mean_or, err_or = _golden_arrays(rec, 1)
        assert_means(sms[i], sm_or, probs[i]["name"] + " (full size, specialised)")
        assert_err(errs[i, :1], err_or, sm_or, probs[i]["name"])


# ------------------------------------------------------------------------------------------------
# prepared batches (qmc_batch_*): plan / upload / prepare once, then kernel launches only
# ------------------------------------------------------------------------------------------------
def _prepared_problems():
    return [make(3, 6, 8191, 5, K + 3, 9990), make(0, 5, 4099, 4, K + 3, 9991), make(8, 4, 4099, 4, K + 3, 9992),
            make(3, 6, 65537, 6, BAKER, 9993), make(3, 4, 8191, 5, K + 3, 9994, fit=True), make_log(6, 8191, 5, K + 3, 9995, pw=2),
            make(2, 12, 4099, 4, SIDI + 2, 9996), make(1, 8, 262147, 8, BAKER, 9997)]


@pytest.mark.parametrize("with_module", [False, True])
def test_prepared_batch_returns_the_bits_of_the_direct_call(with_module):
    probs = _prepared_problems()
    module = binding.SectorModule(probs) if with_module else None
    direct = binding.DeviceBatch(probs, module=module)
    n_direct = direct.integrate()
    ref = direct.results()
    prepared = binding.DeviceBatch(probs, module=module).prepare()
    for call in range(3):
        prepared.shift_means.fill_(float("nan"))
        n_launch = prepared.launch()
        assert n_launch == n_direct - 1                     # no prepare kernel, no upload: fused kernels + finalize
        out = prepared.results()
        assert all(a.tobytes() == b.tobytes() for a, b in zip(out[0], ref[0])), call
        assert out[1].tobytes() == ref[1].tobytes() and out[2].tobytes() == ref[2].tobytes()


def test_prepared_batch_reads_shifts_at_launch():
    """fresh random shifts written into the same device buffers need no new batch"""
    import torch
    probs = _prepared_problems()
    prepared = binding.DeviceBatch(probs).prepare()
    prepared.launch()
    first = prepared.results()
    rng = synth.MT19937_64(424242)
    fresh = [dict(p, shifts=synth.draw_shifts(rng, p["m"], p["dim"])) for p in probs]
    for i in range(len(probs)):
        prepared._keep[4 * i + 2].copy_(torch.from_numpy(fresh[i]["shifts"]))      # the shifts tensor of problem i (DeviceBatch.__init__)
    prepared.launch()
    second = prepared.results()
    ref = run_gpu(fresh)
    assert all(a.tobytes() == b.tobytes() for a, b in zip(second[0], ref[0]))
    assert not all(a.tobytes() == b.tobytes() for a, b in zip(second[0], first[0]))


@pytest.mark.parametrize("with_module", [False, True])
def test_prepared_batch_launch_is_graph_capturable(with_module):
    """a whole sector batch -- tile queues, several kernel variants, finalize -- captured once and replayed"""
    import torch
    probs = _prepared_problems()
    module = binding.SectorModule(probs) if with_module else None
    ref = run_gpu(probs, module=module)
    batch = binding.DeviceBatch(probs, module=module).prepare()
    binding.qmc_profile_enable(False)
    try:
        batch.launch()
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            batch.launch()
        for rep in range(3):
            batch.shift_means.fill_(float("nan"))
            batch.means.fill_(float("nan"))
            graph.replay()
            out = batch.results()
            assert all(a.tobytes() == b.tobytes() for a, b in zip(out[0], ref[0])), rep
            assert out[1].tobytes() == ref[1].tobytes()
    finally:
        binding.qmc_profile_enable(False)                   # the default


def test_prepared_batch_argument_checks():
    L = binding.lib()
    probs = _prepared_problems()[:2]
    b = binding.DeviceBatch(probs)
    import ctypes as C
    handle = C.c_void_p()
    assert L.qmc_batch_create(b.count, b.arr, None, b.ws_ptr, 256, None, C.byref(handle)) == -11      # workspace too small
    assert L.qmc_batch_create(0, b.arr, None, b.ws_ptr, b.ws_bytes, None, C.byref(handle)) == -3
    assert L.qmc_batch_create(b.count, b.arr, None, b.ws_ptr, b.ws_bytes, None, None) == -1
    assert L.qmc_batch_launch(None, None, None, None, None) == -1
    b.prepare()
    assert L.qmc_batch_launch(b.prepared, None, b.errs.data_ptr(), None, None) == -1
    L.qmc_batch_destroy(None)


@pytest.mark.parametrize("d", [1, 3, 4, 5, 6, 8])
@pytest.mark.parametrize("m", [2, 5, 8, 11, 16, 32])
def test_product_peak_group_of_8_shifts(d, m):
    """the product-peak kernels of <= 8 slots exist with 4 and 8 shifts per lattice index (the plan chooses from m): per-shift
    results are the same bits either way, ragged last groups included, and match the oracle"""
    for tr in (BAKER, K + 3, NONE):
        p = make(1, d, 8191, m, tr, 9700 + 10 * d + m)
        a = run_gpu([p], group=4)
        b = run_gpu([p], group=8)
        c = run_gpu([p])
        assert a[0][0].tobytes() == b[0][0].tobytes() == c[0][0].tobytes()
        assert a[1].tobytes() == b[1].tobytes() and a[2].tobytes() == b[2].tobytes()
    check_against_oracle([p], group=8)


@pytest.mark.parametrize("fam", [0, 1, 2, 5])
@pytest.mark.parametrize("d", [2, 4, 6, 8, 11, 16])
def test_dedicated_korobov_kernels_and_the_generic_call_path(fam, d):
    """Korobov r != 3 without a fit map runs in kernels of its own (the transform kind fixed at compile time); the generic loop
    inside the family's kernel still serves it on request -- both against the oracle, every r, ragged tiles"""
    probs = [make(fam, d, n, 5, K + r, 9600 + 7 * d + r) for r, n in ((1, 8191), (2, 127), (4, 65537), (5, 4099), (6, 1021))]
    check_against_oracle(probs)
    check_against_oracle(probs, generic_call=True)
    a = run_gpu(probs)
    b = run_gpu(probs)
    assert all(x.tobytes() == y.tobytes() for x, y in zip(a[0], b[0]))


def test_prepared_batch_of_one_closed_form_problem_and_an_empty_module():
    """the degenerate ends: one closed-form problem (its plan travels in the kernel parameter, nothing to set up) as a prepared
    batch, and a module that found nothing to specialise (no kernels) in a batch call"""
    p = make(1, 8, 262147, 8, BAKER, 9401)
    ref = run_gpu([p])
    one = binding.DeviceBatch([p]).prepare()
    for _ in range(2):
        assert one.launch() == 2                              # fused kernel + finalize
        out = one.results()
        assert out[0][0].tobytes() == ref[0][0].tobytes() and out[2].tobytes() == ref[2].tobytes()
    probs = [p, make(0, 4, 4099, 4, K + 3, 9402)]
    empty = binding.SectorModule(probs)
    assert empty.info["kernels"] == 0 and empty.info["specialised"] == 0
    a = run_gpu(probs)
    b = run_gpu(probs, module=empty)
    assert all(x.tobytes() == y.tobytes() for x, y in zip(a[0], b[0]))
