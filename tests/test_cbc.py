"""The generating-vector tool (paper_1811_11720_b200/cbc.py; setup, off the hot path): component-by-component
construction in a weighted Korobov space.  SURVEY 8(c): the O(n^2) literal
construction and the FFT construction over the multiplicative group must pick the same vector, and the worst-case
error they report must be the criterion written out."""
import json
import os

import numpy as np
import pytest

from paper_1811_11720_b200 import cbc


def literal_e2(n, z, gamma):
    """e^2 = -1 + (1/n) sum_k prod_j (1 + gamma omega({k z_j / n})), omega(x) = 2 pi^2 (x^2 - x + 1/6) (Table A.3's kernel)"""
    k = np.arange(n, dtype=np.int64)
    p = np.ones(n)
    for zj in z:
        x = ((k * int(zj)) % n) / n
        p *= 1.0 + gamma * 2.0 * np.pi ** 2 * (x * x - x + 1.0 / 6.0)
    return -1.0 + p.sum() / n


@pytest.mark.parametrize("n,d", [(1021, 4), (4093, 6), (8191, 8)])
@pytest.mark.parametrize("gamma_rule", ["1", "1/d"])
def test_cbc_direct_equals_cbc_fft(n, d, gamma_rule):
    gamma = 1.0 if gamma_rule == "1" else 1.0 / d
    z_direct, e_direct = cbc.cbc_direct(n, d, gamma)
    z_fft, e_fft = cbc.cbc_fft(n, d, gamma)
    assert z_direct == z_fft
    assert all(1 <= zj <= n // 2 for zj in z_fft)            # folded to min(z, n - z): omega is symmetric
    lit = literal_e2(n, z_fft, gamma)
    assert abs(e_direct - lit) <= 1e-9 * max(1.0, abs(lit))
    assert abs(e_fft - lit) <= 1e-9 * max(1.0, abs(lit))


def test_cbc_first_components_minimise_the_criterion_by_brute_force():
    """n = 127: the second component must be the global minimiser of the two-dimensional criterion (all candidates tried)"""
    n, gamma = 127, 1.0
    z, _ = cbc.cbc_fft(n, 2, gamma)
    best = min(range(1, n), key=lambda c: (round(literal_e2(n, [1, c], gamma), 12), min(c, n - c)))
    assert z == [1, min(best, n - best)]


def test_committed_vectors_reproduce_their_stored_criterion():
    """data/genvecs.json: the small committed vectors give the e^2 stored beside them (literal sum over all n points)"""
    with open(cbc.DATA) as f:
        table = json.load(f)
    checked = 0
    for rec in table.values() if isinstance(table, dict) else table:
        if not isinstance(rec, dict) or "z" not in rec or rec["n"] > 1100000:
            continue
        gamma = 1.0 if rec["gamma"] == "1" else 1.0 / rec["d"]
        lit = literal_e2(rec["n"], rec["z"], gamma)
        assert abs(lit - rec["e2"]) <= 1e-7 * max(1.0, abs(lit)), (rec["n"], rec["d"])
        checked += 1
    assert checked >= 3
