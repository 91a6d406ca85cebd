"""Component-by-component (CBC) construction of rank-1 lattice generating vectors.

SETUP TOOL, not on the timed hot path: the generating vector z is an *input* of the C-ABI
library (include/qmc_lattice.h).  The vectors the paper ships (Table A.1)
are not available, so the vectors used by tests and bench.py are produced once by this tool and
committed under ``paper_1811_11720_b200/data/genvecs.json``.

Criterion (PAPER.md A.3, L1038-L1042, Korobov space, smoothness alpha = 2, beta_j = 1):
    e_s^2(z) = -1 + (1/n) sum_{k=0}^{n-1} prod_{j<=s} (1 + gamma_j * omega({k z_j / n})),
    omega(x) = 2 pi^2 (x^2 - x + 1/6)       (the paper's text is garbled: "x^2 x + 1/6").
For prime n, component s is the z in [1, n-1] minimising that sum given z_1..z_{s-1}
(section 2.2).  The fast variant (Nuyens-Cools, the paper's Ref. [47]) orders
candidates and points by powers of a primitive root g so that all candidate sums are one cyclic
convolution, evaluated by FFT; omega is symmetric so the group is folded to (n-1)/2 elements.

Ties (reading C-9): z and n-z always tie; candidates within 1e-9*(Emax-Emin) of the
minimum are treated as tied and the smallest min(z, n-z) is taken.
"""
from __future__ import annotations

import json
import math
import os
import sys
import time

import numpy as np

try:  # multi-threaded pocketfft when scipy is present (only matters for n ~ 1e9)
    import scipy.fft as _fft
    _FFT_KW = {"workers": -1}
except ImportError:  # pragma: no cover
    _fft, _FFT_KW = np.fft, {}

TWO_PI2 = 2.0 * math.pi * math.pi


def omega(x):
    """Kernel of the alpha=2 Korobov space."""
    return TWO_PI2 * (x * x - x + 1.0 / 6.0)


def is_prime(n: int) -> bool:
    if n < 2:
        return False
    for p in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):
        if n % p == 0:
            return n == p
    d, s = n - 1, 0
    while d % 2 == 0:
        d //= 2
        s += 1
    for a in (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37):  # deterministic for n < 3.3e24
        x = pow(a, d, n)
        if x in (1, n - 1):
            continue
        for _ in range(s - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def _factorize(m: int):
    f, p = [], 2
    while p * p <= m:
        if m % p == 0:
            f.append(p)
            while m % p == 0:
                m //= p
        p += 1 if p == 2 else 2
    if m > 1:
        f.append(m)
    return f


def primitive_root(n: int) -> int:
    fac = _factorize(n - 1)
    for g in range(2, n):
        if all(pow(g, (n - 1) // q, n) != 1 for q in fac):
            return g
    raise ValueError("no primitive root")


def _powers_mod(g: int, count: int, n: int) -> np.ndarray:
    """[g^0, g^1, ..., g^(count-1)] mod n by doubling; needs n < 2^32 (products < 2^64)."""
    assert n < (1 << 32)
    out = np.empty(count, dtype=np.uint64)
    out[0] = 1
    filled = 1
    nn = np.uint64(n)
    while filled < count:
        step = min(filled, count - filled)
        mult = np.uint64(pow(g, filled, n))
        np.multiply(out[:step], mult, out=out[filled:filled + step])
        np.remainder(out[filled:filled + step], nn, out=out[filled:filled + step])
        filled += step
    return out


def cbc_direct(n: int, d: int, gamma: float):
    """O(d n^2) reference CBC (small n only): literal evaluation of the criterion."""
    k = np.arange(n, dtype=np.int64)
    p = np.ones(n)
    z = []
    for s in range(d):
        if s == 0:
            zs = 1
        else:
            cand = np.arange(1, n // 2 + 1, dtype=np.int64)      # z and n-z tie: fold
            E = np.empty(len(cand))
            for i, c in enumerate(cand):
                E[i] = np.sum(p * omega(((k * c) % n) / n))
            tol = 1e-9 * (E.max() - E.min())
            zs = int(cand[np.nonzero(E <= E.min() + tol)[0]].min())
        z.append(zs)
        p = p * (1.0 + gamma * omega(((k * zs) % n) / n))
    return z, float(-1.0 + p.sum() / n)


def cbc_fft(n: int, d: int, gamma: float, verbose: bool = False, stop_on_repeat: bool = False):
    """Fast CBC for prime n < 2^32.  Returns (z, e2) with z_j folded to min(z, n-z)."""
    assert is_prime(n) and n > 3
    half = (n - 1) // 2
    g = primitive_root(n)
    ginv = pow(g, -1, n)
    # c[a] = omega(g^a / n), a in [0, half): g^(a+half) = -g^a and omega(1-x) = omega(x)
    pw = _powers_mod(g, half, n)
    c = omega(pw.astype(np.float64) / float(n))
    del pw
    # linear-convolution embedding of the length-`half` cyclic convolution in a smooth FFT size
    N = 1 << int(math.ceil(math.log2(2 * half)))
    cc = np.zeros(N)
    cc[:half] = c
    cc[half:2 * half] = c
    Fc = _fft.rfft(cc, **_FFT_KW)
    del cc
    P = np.ones(half)            # P[b] = p[g^(-b)], p = running product over chosen components
    z = [1]
    # component 1: z = 1 = g^0  ->  factor at point g^(-b) is omega(g^(-b)/n) = c[(-b) mod half]
    idx0 = (-np.arange(half, dtype=np.int64)) % half
    P *= 1.0 + gamma * c[idx0]
    for s in range(1, d):
        t0 = time.time()
        buf = np.zeros(N)
        buf[:half] = P
        Fp = _fft.rfft(buf, **_FFT_KW)
        del buf
        Fp *= Fc
        conv = _fft.irfft(Fp, n=N, **_FFT_KW)
        del Fp
        E = conv[half:2 * half].copy()     # E[a] = sum_b P[b] c[(a-b) mod half], candidate g^a
        del conv
        tol = 1e-9 * float(E.max() - E.min())
        ties = np.nonzero(E <= E.min() + tol)[0]
        best = None
        for a in ties[:4096]:
            zc = pow(g, int(a), n)
            zc = min(zc, n - zc)
            if best is None or zc < best[0]:
                best = (zc, int(a))
        zs, a_star = best
        del E
        z.append(zs)
        idx = (a_star + idx0) % half          # (a* - b) mod half
        P *= 1.0 + gamma * c[idx]
        del idx
        if verbose:
            print(f"  n={n} s={s + 1} z={zs} ties={len(ties)} ({time.time() - t0:.1f}s)", flush=True)
        if stop_on_repeat and len(set(z)) != len(z):
            return z, float("nan")
    # sum over k=1..n-1 is twice the folded sum; k=0 contributes prod(1+gamma*omega(0))
    p0 = 1.0
    for _ in range(d):
        p0 *= 1.0 + gamma * omega(0.0)
    e2 = -1.0 + (p0 + 2.0 * float(np.sum(P))) / n
    del ginv
    return z, e2


def build(n: int, d: int, verbose: bool = True):
    """gamma_j = 1 as BASELINE.json says; if components repeat, the paper's gamma_j = 1/d (L165)."""
    z, e2 = cbc_fft(n, d, 1.0, verbose=verbose, stop_on_repeat=True)
    gamma = "1"
    if len(set(z)) != len(z):
        if verbose:
            print(f"  n={n} d={d}: gamma=1 repeats components -> rebuilding with gamma=1/d", flush=True)
        z, e2 = cbc_fft(n, d, 1.0 / d, verbose=verbose)
        gamma = "1/d"
        assert len(set(z)) == len(z)
    return {"n": n, "d": d, "gamma": gamma, "z": z, "e2": e2}


DATA = os.path.join(os.path.dirname(os.path.abspath(__file__)), "data", "genvecs.json")


def main(argv):
    """python -m paper_1811_11720_b200.cbc n:d [n:d ...]  -> merges into data/genvecs.json"""
    table = {}
    if os.path.exists(DATA):
        with open(DATA) as f:
            table = json.load(f)
    for spec in argv:
        n, d = (int(v) for v in spec.split(":"))
        print(f"CBC n={n} d={d}", flush=True)
        rec = build(n, d)
        table[f"{n}:{d}"] = rec
        with open(DATA, "w") as f:
            json.dump(table, f, indent=1, sort_keys=True)
        print(f"  -> {rec}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
