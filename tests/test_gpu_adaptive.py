"""GPU tests of qmc_integrate: the paper's `integrate` iteration (section 3.3.1; fields L887-L920;
result struct L988-L995) around the fused hot path.  Whatever lattice / shift count the iteration ends on, its result
must equal the CPU oracle's result for that (n, m) at the parity bars of test_gpu_parity.py."""
import numpy as np
import pytest

import oracle
from paper_1811_11720_b200 import binding, synth

pytestmark = pytest.mark.gpu
K = synth.TRANSFORM_KOROBOV


def _oracle_at(p, res, ladder_n, ladder_z):
    i = int(np.where(ladder_n == res["n"])[0][0])
    q = dict(p, n=res["n"], z=ladder_z[i], shifts=p["shifts"][:res["m"]], m=res["m"])
    return oracle.integrate(q)


def _problem(c, max_m):
    p = synth.config(c)[0]
    rng = synth.MT19937_64(4242 + c)
    return dict(p, shifts=synth.draw_shifts(rng, max_m, p["dim"]), m=max_m)


def test_reaches_goal_by_enlarging_the_lattice():
    """configs[0] shape, eps_rel = 1e-8 (the paper's Genz setting): the iteration climbs the ladder,
    discards the earlier results (L357) and stops on a lattice whose estimate matches the oracle and the closed form"""
    p = _problem(0, 10)
    ln, lz = synth.ladder(4, 65537)
    res, st = binding.qmc_integrate(0, p["params"], 4, K + 3, ln, lz, p["shifts"], min_n=1000, min_m=10, epsrel=1e-8, epsabs=0.0,
                                    maxeval=10**9)
    assert st == 0 and res["m"] == 10 and res["n"] in ln.tolist() and res["iterations"] >= 2
    assert res["error"][0] <= 1e-8 * abs(res["integral"][0])
    sm_or, mean_or, err_or = _oracle_at(p, res, ln, lz)
    assert abs(res["integral"][0] - mean_or[0]) <= 1e-13 * abs(mean_or[0])
    assert abs(res["error"][0] - err_or[0]) <= 1e-12 * err_or[0] + 1e-13 * np.max(np.abs(sm_or)) / 3.0
    prm = p["params"]                                       # closed form of Genz oscillatory
    a = prm[1:]
    exact = np.cos(2 * np.pi * prm[0] + 0.5 * a.sum()) * np.prod(np.sin(a / 2) / (a / 2))
    assert abs(res["integral"][0] - exact) <= 6 * res["error"][0] + 1e-14
    assert res["evaluations"] >= res["n"] * res["m"]        # discarded iterations are counted (L995)


def test_maxeval_terminates_and_returns_the_last_result():
    p = _problem(1, 8)
    ln, lz = synth.ladder(8, 1048573)
    res, st = binding.qmc_integrate(1, p["params"], 8, synth.TRANSFORM_BAKER, ln, lz, p["shifts"], min_n=1000, min_m=8, epsrel=1e-12,
                                    epsabs=0.0, maxeval=200000)
    assert st == binding.QMC_ERR_MAXEVAL
    assert res["evaluations"] <= 200000 + res["n"] * res["m"]   # "approximate" maximum (L903-L905)
    sm_or, mean_or, err_or = _oracle_at(p, res, ln, lz)
    assert abs(res["integral"][0] - mean_or[0]) <= 1e-13 * abs(mean_or[0])


def test_exhausted_ladder_adds_shifts():
    """one available lattice: the iteration keeps it and adds random shifts (Monte Carlo scaling)"""
    p = dict(_problem(0, 64), transform=synth.TRANSFORM_NONE)
    ln, lz = synth.ladder(4, 1021)
    assert ln.tolist() == [1021]
    first, _ = binding.qmc_integrate(0, p["params"], 4, synth.TRANSFORM_NONE, ln, lz, p["shifts"][:4], min_n=1, min_m=4, epsrel=0.0,
                                     epsabs=0.0, maxeval=1)
    eps = float(first["error"][0] / abs(first["integral"][0])) / 2.5      # needs ~6x the shifts under m^-1/2 scaling
    res, st = binding.qmc_integrate(0, p["params"], 4, synth.TRANSFORM_NONE, ln, lz, p["shifts"], min_n=1, min_m=4, epsrel=eps,
                                    epsabs=0.0, maxeval=10**8)
    assert res["n"] == 1021 and res["m"] > 4 and res["iterations"] >= 2
    assert res["evaluations"] == 1021 * res["m"]            # extensions sample only the new shifts
    sm_or, mean_or, err_or = _oracle_at(p, res, ln, lz)
    assert abs(res["integral"][0] - mean_or[0]) <= 1e-13 * abs(mean_or[0])
    assert abs(res["error"][0] - err_or[0]) <= 1e-9 * err_or[0]
    assert (st == 0) == (res["error"][0] <= eps * abs(res["integral"][0]))


@pytest.mark.parametrize("errormode", [0, 1])
def test_complex_error_modes(errormode):
    """`all` needs every component within its own goal, `largest` compares with the largest component"""
    p = synth.config(2, n_override=1021)[0]
    rng = synth.MT19937_64(77)
    sh = synth.draw_shifts(rng, 16, 12)
    ln, lz = synth.ladder(12, 262139)
    res, st = binding.qmc_integrate(2, p["params"], 12, K + 3, ln, lz, sh, min_n=1000, min_m=16, epsrel=0.05, epsabs=0.0,
                                    maxeval=10**9, errormode=errormode)
    E, err = res["integral"], res["error"]
    if errormode == 0:
        met = all(err[c] <= 0.05 * abs(E[c]) for c in range(2))
    else:
        met = max(err) <= 0.05 * max(abs(E[0]), abs(E[1]))
    assert (st == 0) == met
    q = dict(p, shifts=sh, m=16)
    sm_or, mean_or, err_or = _oracle_at(q, res, ln, lz)
    assert np.all(np.abs(E - mean_or) <= 1e-13 * np.hypot(*mean_or))


def test_sector_with_log_factor_through_the_iteration():
    """an eps-expansion term of a sector (trailing [lu, lf, p] block, reading C-15) through qmc_integrate: the
    result equals the oracle's at the lattice the iteration stops on"""
    d = 6
    rng = synth.MT19937_64(5150)
    prm = synth.sector_log(rng, d)
    sh = synth.draw_shifts(rng, 16, d)
    ln, lz = synth.ladder(d, 262139)
    res, st = binding.qmc_integrate(synth.FAMILY_SECTOR, prm, d, K + 3, ln, lz, sh, min_n=1000, min_m=16, epsrel=1e-6, epsabs=0.0,
                                    maxeval=10**9)
    assert st == 0 and res["m"] == 16 and res["error"][0] <= 1e-6 * abs(res["integral"][0])
    p = synth.problem(synth.FAMILY_SECTOR, prm, int(ln[0]), lz[0], sh, K + 3)
    sm_or, mean_or, err_or = _oracle_at(p, res, ln, lz)
    assert abs(res["integral"][0] - mean_or[0]) <= 1e-13 * abs(mean_or[0])
    assert abs(res["error"][0] - err_or[0]) <= 1e-12 * err_or[0] + 1e-13 * np.max(np.abs(sm_or)) / np.sqrt(15.0)
    # without the block the same call integrates a different function
    res0, st0 = binding.qmc_integrate(synth.FAMILY_SECTOR, prm[:-3], d, K + 3, ln, lz, sh, min_n=1000, min_m=16, epsrel=1e-6,
                                      epsabs=0.0, maxeval=10**9)
    assert st0 == 0 and abs(res0["integral"][0] - res["integral"][0]) > 1e-3 * abs(res0["integral"][0])


def test_argument_errors():
    p = _problem(0, 10)
    ln, lz = synth.ladder(4, 65537)
    with pytest.raises(binding.QmcError) as e:
        binding.qmc_integrate(0, p["params"], 4, K + 3, ln[::-1].copy(), lz[::-1].copy(), p["shifts"], min_m=10)
    assert e.value.status == -3                             # ladder must ascend
    with pytest.raises(binding.QmcError) as e:
        binding.qmc_integrate(0, p["params"], 4, K + 3, ln, lz, p["shifts"], min_m=1)
    assert e.value.status == -6
    bad = lz.copy()
    bad[2, 1] = ln[2]                                       # z_j = n is not coprime to n
    with pytest.raises(binding.QmcError) as e:
        binding.qmc_integrate(0, p["params"], 4, K + 3, ln, bad, p["shifts"], min_m=10)
    assert e.value.status == -4
