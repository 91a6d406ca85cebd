"""CPU-side checks of the C-ABI boundary (no compute launches): the library loads, exports every symbol
include/qmc_lattice.h declares, validates arguments as the header states, and its host-only pieces
(launch plan, cubic fit) behave.  Runs with -m "not gpu"."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
from paper_1811_11720_b200 import binding, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
K3 = synth.TRANSFORM_KOROBOV + 3


@pytest.fixture(scope="module")
def L():
    from paper_1811_11720_b200 import build
    build.build()
    return binding.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "qmc_lattice.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qmc_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    names = _declared_symbols()
    assert len(names) >= 16
    for name in names:
        assert hasattr(L, name), f"{name} declared in include/qmc_lattice.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_status_strings_and_components(L):
    assert L.qmc_status_string(0) == b"ok"
    for st in range(-13, 0):
        assert L.qmc_status_string(st) not in (b"ok", b"unknown status")
    assert [L.qmc_num_components(f) for f in range(4)] == [1, 1, 2, 1]
    assert L.qmc_num_components(9) < 0


def _cfg0():
    return synth.config(0)[0]


def test_validate_problem_host_accepts_all_configs():
    for c in range(5):
        n_over = None if c < 4 else 1048573           # config 4's CBC vector is large; same code path
        for p in synth.config(c, n_override=n_over, count_override=4 if c == 3 else None):
            assert binding.qmc_validate_problem_host(p) == 0, p["name"]


@pytest.mark.parametrize("mutate,status", [
    (lambda p: p.update(dim=0), -2),
    (lambda p: p.update(n=1), -3),
    (lambda p: p.update(n=1 << 53), -3),
    (lambda p: p["z"].__setitem__(1, 0), -4),
    (lambda p: p["z"].__setitem__(1, 65537), -4),
    (lambda p: p["shifts"].__setitem__((0, 0), 1.0), -5),
    (lambda p: p["shifts"].__setitem__((1, 2), -1e-9), -5),
    (lambda p: p["shifts"].__setitem__((1, 2), float("nan")), -5),
    (lambda p: p.update(m=1), -6),
    (lambda p: p.update(transform=107), -7),
    (lambda p: p.update(transform=2), -7),
    (lambda p: p.update(transform=207), -7),                 # Sidi weight outside 1..6
    (lambda p: p.update(transform=1000 + 16 * 0 + 3), -7),   # asymmetric Korobov weights outside 1..6
    (lambda p: p.update(transform=1000 + 16 * 3 + 7), -7),
    (lambda p: p.update(family=9), -8),
    (lambda p: p.update(family=7), -9),                      # a valid family now, but the block has the wrong length
    (lambda p: p.update(params=p["params"][:-1]), -9),
    (lambda p: p.update(fit_coeffs=synth.cubic_fit_coeffs(4, a4=-0.2, a5=0.3)), -10),
    (lambda p: p.update(fit_coeffs=synth.cubic_fit_coeffs(4, a4=2.0, a5=-5.0)), -10),
    (lambda p: p.update(fit_coeffs=np.array([[1.0005, -0.5, 0.1, 0.0, 0.6, 0.2]] * 4)), -10),   # a0 below 1.001
    (lambda p: p.update(fit_coeffs=np.array([[1.5, 0.2, 0.0, 0.1, 0.6, 0.2]] * 4)), -10),       # a1 above -0.001
    (lambda p: p.update(fit_coeffs=np.array([[1.5, -0.5, -0.1, 0.0, 0.6, 0.2]] * 4)), -10),     # a2 negative
    (lambda p: p.update(fit_coeffs=np.array([[1.5, -0.5, 0.05, 0.05, 3.0, -6.0]] * 4)), -10),   # not increasing
])
def test_validate_problem_host_rejects(mutate, status):
    p = _cfg0()
    p = dict(p, z=p["z"].copy(), shifts=p["shifts"].copy(), params=p["params"].copy())
    mutate(p)
    assert binding.qmc_validate_problem_host(p) == status


@pytest.mark.parametrize("d", [1, 2, 3, 6])
def test_validate_sector_log_block(d):
    """The sector block takes an optional trailing [lu, lf, p] (p an integer in 1..4); d = 2 is the case where three more
    doubles could be mistaken for one more monomial."""
    rng = synth.MT19937_64(90 + d)
    prm = synth.sector_log(rng, d)
    n = 1021
    p = synth.problem(synth.FAMILY_SECTOR, prm, n, synth.korobov_form_vector(n, d, 341), synth.draw_shifts(rng, 4, d),
                      synth.TRANSFORM_KOROBOV + 3)
    assert binding.qmc_validate_problem_host(p) == 0
    assert binding.qmc_validate_problem_host(dict(p, params=prm[:-3])) == 0               # the plain block
    for bad_p in (0.0, 5.0, 1.5, -1.0):
        q = prm.copy(); q[-1] = bad_p
        assert binding.qmc_validate_problem_host(dict(p, params=q)) == -9
    for cut in (1, 2):
        assert binding.qmc_validate_problem_host(dict(p, params=prm[:-cut])) == -9
    assert binding.qmc_validate_problem_host(dict(p, params=np.concatenate([prm, [1.0]]))) == -9


def test_z_must_be_coprime_to_n():
    """'integers coprime to n'; n itself need not be prime (Fig. 1 uses 55, L108)."""
    p = _cfg0()
    p = dict(p, n=55, z=np.array([1, 34, 13, 21], dtype=np.uint64))
    assert binding.qmc_validate_problem_host(p) == 0
    p["z"][2] = 15                                        # gcd(15, 55) = 5
    assert binding.qmc_validate_problem_host(p) == -4


def test_synchronous_entry_rejects_before_touching_the_device(L):
    """Argument errors are reported without any launch, so this works without a GPU."""
    p = _cfg0()
    with pytest.raises(binding.QmcError) as e:
        binding.qmc_lattice_integrate(p["family"], p["params"], p["dim"], p["n"], p["z"], p["shifts"], 1, p["transform"])
    assert e.value.status == -6
    with pytest.raises(binding.QmcError) as e:
        binding.qmc_lattice_integrate(9, p["params"], p["dim"], p["n"], p["z"], p["shifts"], p["m"], p["transform"])
    assert e.value.status == -8


def _host_struct(p):
    keep = [np.ascontiguousarray(p["params"]), np.ascontiguousarray(p["z"]), np.ascontiguousarray(p["shifts"])]
    s = binding.qmc_problem(p["family"], p["dim"], p["m"], p["transform"], p["n"], keep[0].ctypes.data, len(keep[0]),
                            keep[1].ctypes.data, keep[2].ctypes.data, None)
    return s, keep


def test_plan_is_a_pure_function_of_the_problem(L):
    """Tiles and workspace size depend on the problem structs only (not on the device): the fixed
    result slots are what makes the reduction deterministic."""
    for c in (0, 1, 2):
        p = synth.config(c)[0]
        s, keep = _host_struct(p)
        arr = (binding.qmc_problem * 1)(s)
        tiles, tl0 = C.c_longlong(), C.c_longlong()
        assert L.qmc_plan_info(1, arr, C.byref(tiles), None, C.byref(tl0)) == 0
        assert tiles.value * tl0.value >= p["n"] > (tiles.value - 1) * tl0.value
        assert 128 <= tl0.value <= 128 * 1024          # >= one index per thread; fp64 chains of at most 1024 terms
        ws = L.qmc_workspace_bytes(1, arr)
        assert ws >= tiles.value * p["m"] * oracle.ncomp(p["family"]) * 8
        assert ws == L.qmc_workspace_bytes(1, arr)
    bad = (binding.qmc_problem * 1)(binding.qmc_problem(0, 0, 2, 0, 7, None, 0, None, None, None))
    assert L.qmc_workspace_bytes(1, bad) == 0
    assert L.qmc_plan_info(1, bad, None, None, None) == -2


def test_fit_cubic_matches_oracle_and_recovers_a_cubic():
    """qmc_fit_cubic is host code of the product; the oracle's fit is independent code (reading C-8)."""
    rng = np.random.default_rng(7)
    bins, d = 256, 5
    H = np.empty((d, bins))
    edges = np.arange(bins + 1) / bins
    truth = []
    for j in range(d):
        a4, a5 = 0.5 + 0.4 * rng.random(), 0.6 * rng.random() - 0.1
        a6 = 1 - a4 - a5
        pinv = lambda y: y * (a4 + y * (a5 + y * a6))          # p = CDF^-1, so CDF(e) = p^-1(e)
        ys = np.linspace(0, 1, 200001)
        cdf = np.interp(edges, pinv(ys), ys)
        H[j] = np.diff(cdf)
        truth.append((a4, a5))
    got = binding.qmc_fit_cubic(H)
    ref = oracle.fit_cubic(H)
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-10)
    for j, (a4, a5) in enumerate(truth):
        assert abs(got[j, 4] - a4) < 1e-6 and abs(got[j, 5] - a5) < 1e-6
        assert got[j, 2] == 0.0 and got[j, 3] == 0.0
    flat = binding.qmc_fit_cubic(np.ones((2, 64)))
    np.testing.assert_allclose(flat[:, 4:], [[1.0, 0.0], [1.0, 0.0]], atol=1e-12)
    spike = np.zeros((1, 64)); spike[0, 3] = 1.0              # not fittable by a monotone cubic -> identity
    assert binding.qmc_fit_cubic(spike)[0, 4:].tolist() == [1.0, 0.0]


def test_product_never_imports_the_oracle():
    """The product path must not route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1811_11720_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "qmc_oracle" not in text and "libqmc_oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "qmc_oracle.cpp")).read()
    assert "#include \"" not in otext                         # the oracle includes no project header


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libqmc_lattice.so")
    with pytest.raises(ImportError):
        binding.lib()


def _hist_of_map(a, bins):
    """histogram whose CDF is the inverse of the increasing map p of PAPER.md Eq. 19: c_b = p^-1(b/bins) by bisection
    (p evaluated by the ORACLE's fit_map), H[b] = c_{b+1} - c_b"""
    edges = [0.0]
    for b in range(1, bins):
        lo, hi = 0.0, 1.0
        for _ in range(80):
            mid = 0.5 * (lo + hi)
            if oracle.fit_map(a, mid)[0] < b / bins:
                lo = mid
            else:
                hi = mid
        edges.append(0.5 * (lo + hi))
    edges.append(1.0)
    return np.diff(np.array(edges))


def test_fit_polysingular_recovers_a_map_with_poles():
    """row f-2: the bounded Levenberg-Marquardt fit of the complete fit function (bounds L231) reproduces
    an inverse CDF generated from known parameters far better than the cubic sub-family can, and returns a valid map"""
    truth = np.array([[1.05, -0.4, 0.35, 0.0, 0.30, 0.25], [1.6, -0.03, 0.0, 0.45, 0.35, 0.10], [1.001, -0.001, 0.0, 0.0, 0.7, 0.2]])
    bins = 256
    H = np.array([_hist_of_map(a, bins) for a in truth])
    full, cubic = binding.qmc_fit_polysingular(H), binding.qmc_fit_cubic(H)
    for j in range(3):
        c = np.cumsum(H[j])[:-1] / H[j].sum()
        e = np.arange(1, bins) / bins
        res_full = max(abs(oracle.fit_map(full[j], y)[0] - t) for y, t in zip(c, e))
        res_cub = max(abs(oracle.fit_map(cubic[j], y)[0] - t) for y, t in zip(c, e))
        assert res_full <= res_cub + 1e-15
        a = full[j]
        assert a[0] >= 1.001 and a[1] <= -0.001 and a[2] >= 0 and a[3] >= 0
        assert min(oracle.fit_map(a, y)[1] for y in np.linspace(0, 1, 513)) > 0          # increasing
        assert abs(oracle.fit_map(a, 1.0)[0] - 1.0) < 1e-14 and oracle.fit_map(a, 0.0)[0] == 0.0
        if j < 2:
            assert res_full < 2e-4 and res_full < 0.05 * res_cub                            # the poles matter and are found
            assert a[2] > 0 or a[3] > 0
        else:
            assert res_full < 1e-9                                                           # an exact cubic stays a cubic fit
    p = dict(_cfg0(), fit_coeffs=np.tile(full[0], (4, 1)))
    assert binding.qmc_validate_problem_host(p) == 0                                         # valid input of the compute entries
    flat = binding.qmc_fit_polysingular(np.ones((2, 64)))
    np.testing.assert_allclose(flat[:, 4:], [[1.0, 0.0]] * 2, atol=1e-12)
    assert np.all(flat[:, 2:4] == 0.0)


def test_fit_from_cdf_pairs_on_the_host():
    """qmc_fit_from_cdf (host code): the cubic from sampled pairs equals the oracle's on the same pairs and recovers an exact
    cubic; with_poles recovers a map with a pole term; argument errors"""
    a4, a5 = 0.55, 0.35
    c = np.linspace(0.0005, 0.9995, 2000)
    x = c * (a4 + c * (a5 + c * (1 - a4 - a5)))
    got = binding.qmc_fit_from_cdf(np.stack([x, x]), np.stack([c, c]))
    ref = oracle.fit_cubic_cdf(np.stack([x, x]), np.stack([c, c]))
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-10)
    assert abs(got[0, 4] - a4) < 1e-10 and abs(got[0, 5] - a5) < 1e-10
    a = np.array([1.05, -0.2, 0.3, 0.0, 0.4, 0.2])                     # Eq. 19 with one pole term
    a6 = 1 - a[2] - a[3] - a[4] - a[5]
    xp = a[2] * c * (a[0] - 1) / (a[0] - c) + c * (a[4] + c * (a[5] + c * a6))
    full = binding.qmc_fit_from_cdf(xp[None, :], c[None, :], with_poles=True)
    model = full[0, 2] * c * (full[0, 0] - 1) / (full[0, 0] - c) + full[0, 3] * c * (full[0, 1] - 1) / (full[0, 1] - c) + \
        c * (full[0, 4] + c * (full[0, 5] + c * (1 - full[0, 2:].sum())))
    assert np.max(np.abs(model - xp)) < 1e-6 and full[0, 2] > 0.05
    L = binding.lib()
    out = np.zeros(6)
    assert L.qmc_fit_from_cdf(None, None, 1, 100, 0, binding._d(out)) == -1
    assert L.qmc_fit_from_cdf(binding._d(x), binding._d(c), 1, 4, 0, binding._d(out)) == -3
    assert L.qmc_cdf_sample_count(1048573, 10) == 104857 and L.qmc_cdf_sample_count(100, 0) == 0 and L.qmc_cdf_sample_count(100, 101) == 0


def test_host_pointer_batch_rejects_before_touching_the_device(L):
    """qmc_lattice_integrate_batch_host validates every problem (values included) before it stages or launches anything"""
    p = _cfg0()
    def call(probs):
        arr = (binding.qmc_problem * len(probs))()
        keep = []
        for i, q in enumerate(probs):
            prm, sh, z = np.ascontiguousarray(q["params"]), np.ascontiguousarray(q["shifts"]), np.ascontiguousarray(q["z"], dtype=np.uint64)
            keep += [prm, sh, z]
            arr[i] = binding.qmc_problem(q["family"], q["dim"], q["m"], q["transform"], q["n"], prm.ctypes.data, len(prm), z.ctypes.data,
                                         sh.ctypes.data, None)
        means, errs = np.zeros((len(probs), 2)), np.zeros((len(probs), 2))
        return L.qmc_lattice_integrate_batch_host(len(probs), arr, binding._d(means), binding._d(errs), None)
    bad_shift = dict(p, shifts=p["shifts"].copy())
    bad_shift["shifts"][1, 0] = 1.0
    assert call([p, bad_shift]) == -5
    assert call([dict(p, z=np.array([2, 4, 6, 65537 - 1], dtype=np.uint64) * 0 + 65537)]) == -4
    assert L.qmc_lattice_integrate_batch_host(0, None, None, None, None) == -3
    assert L.qmc_lattice_integrate_batch_host(1, None, None, None, None) == -1


def test_sector_family_limits_in_the_struct_checks(L):
    """dim <= QMC_MAX_SECTOR_DIM for both sector families; the complex family has (2 + d) doubles per monomial"""
    rng = synth.MT19937_64(3)
    d = 6
    prm = synth.sector_complex(rng, d)
    sh = synth.draw_shifts(rng, 4, d)
    ok = synth.problem(8, prm, 8191, synth.korobov_form_vector(8191, d, 2731), sh, K3)
    assert binding.qmc_validate_problem_host(ok) == 0
    assert binding.qmc_validate_problem_host(dict(ok, params=prm[:-1])) == -9
    assert binding.qmc_validate_problem_host(dict(ok, family=3)) == -9                 # the real family reads (1 + d) per monomial
    d17 = 17
    big = synth.problem(3, np.concatenate([[1, 1, 1, 1], np.zeros(d17), [1.0], np.zeros(d17), [1.0], np.zeros(d17)]), 8191,
                        synth.korobov_form_vector(8191, d17, 2731), synth.draw_shifts(rng, 2, d17), K3)
    assert binding.qmc_validate_problem_host(big) == -2


# ---- modules of specialised sector kernels: built on the host, no GPU needed (compiled integrands) ----
def _sector_problem(d, seed, n=4099, m=4, family=3):
    rng = synth.MT19937_64(seed)
    prm = synth.sector(rng, d) if family == 3 else synth.sector_complex(rng, d)
    return synth.problem(family, prm, n, synth.korobov_form_vector(n, d, 1 + n // 3), synth.draw_shifts(rng, m, d),
                         synth.TRANSFORM_KOROBOV + 3, name=f"sector.d{d}.{seed}")


def test_sector_module_builds_without_a_gpu():
    """every dimension-slot kind is assembled for sm_100a; kernels hold at most `sectors_per_kernel` sectors of one kind"""
    probs = [_sector_problem(d, 500 + d) for d in (2, 4, 5, 6, 6, 6, 7, 8, 11, 16)]
    mod = binding.SectorModule(probs, sectors_per_kernel=2)
    info = mod.info
    assert info["specialised"] == 10
    assert info["kernels"] == 1 + 2 + 1 + 1                  # slots 4: d = 2, 4; 6: d = 5, 6, 6, 6 (2 kernels); 8: d = 7, 8; 16: d = 11, 16
    assert info["build_ms"] > 0 and info["image_bytes"] > 10000 and 1 <= info["host_threads"] <= info["kernels"]
    for k in range(info["kernels"]):
        image, log = mod.image(k)
        assert image[:4] == b"\x7fELF"
        assert "registers" in log and "qmc_spec_dp" in log
    with pytest.raises(binding.QmcError):
        mod.image(info["kernels"])
    mod.close()
    mod.close()                                              # idempotent


def test_sector_module_code_is_the_compiled_program():
    """the device code of one sector: no indexed branch per step -- one per evaluation -- and as many FP64 instructions in the
    case as the Horner program has steps (x G points), plus the tail's multiplications"""
    import shutil
    import subprocess
    import tempfile
    if shutil.which("cuobjdump") is None:
        pytest.skip("cuobjdump not on PATH")
    p = _sector_problem(6, 777)
    mod = binding.SectorModule([p])
    image, _ = mod.image(0)
    with tempfile.NamedTemporaryFile(suffix=".cubin") as f:
        f.write(image)
        f.flush()
        sass = subprocess.run(["cuobjdump", "-sass", f.name], capture_output=True, text=True, check=True).stdout
    assert "sm_100" in sass
    assert sass.count("BRX") == 0                            # one sector: no selector, and no indexed branch per step either
    three = binding.SectorModule([p, _sector_problem(6, 778), _sector_problem(6, 779)])
    with tempfile.NamedTemporaryFile(suffix=".cubin") as f:
        f.write(three.image(0)[0])
        f.flush()
        assert subprocess.run(["cuobjdump", "-sass", f.name], capture_output=True, text=True, check=True).stdout.count("BRX") == 1
    ref = binding.SectorModule([dict(p, family=0, params=np.ones(7))])       # a batch with nothing to specialise: no kernels
    assert ref.info["kernels"] == 0 and ref.info["specialised"] == 0
    # count the polynomial's operations from the parameter block with the oracle-side model of the Horner form: every monomial
    # of degree D costs between 1 and D steps, so the case holds at least (monomials - constants) and at most sum(D) steps per point
    prm = p["params"]
    nU, nF = int(prm[2]), int(prm[3])
    off, lo, hi = 4 + 6, 0, 0
    for cnt in (nU, nF):
        e = prm[off + cnt:off + cnt + cnt * 6].reshape(cnt, 6)
        deg = e.sum(axis=1)
        lo += int((deg > 0).sum())
        hi += int(deg.sum())
        off += cnt * 7
    fp64 = sass.count("DFMA") + sass.count("DMUL")
    base = binding.SectorModule([dict(p, params=_one_monomial_block(6))])
    img0, _ = base.image(0)
    with tempfile.NamedTemporaryFile(suffix=".cubin") as f:
        f.write(img0)
        f.flush()
        sass0 = subprocess.run(["cuobjdump", "-sass", f.name], capture_output=True, text=True, check=True).stdout
    extra = fp64 - (sass0.count("DFMA") + sass0.count("DMUL"))
    assert 8 * (lo - 2) <= extra <= 8 * (hi + 16), (extra, lo, hi)


def _one_monomial_block(d):
    """U = 1 + x_0, F = 1 + x_0, a = b = 1, nu = 0: the smallest valid sector"""
    e = [0.0] * d
    e1 = [1.0] + [0.0] * (d - 1)
    return np.array([1.0, 1.0, 2.0, 2.0] + [0.0] * d + [1.0, 1.0] + e + e1 + [1.0, 1.0] + e + e1)


def test_sector_module_skips_what_it_cannot_compile(L):
    """other families and blocks the validation rejects stay on the default kernels; complex sectors get kernels of their own"""
    good = _sector_problem(6, 900)
    bad = _sector_problem(6, 901)
    prm = bad["params"].copy()
    prm[4 + 6 + int(prm[2]) + 2] = 9.0                       # an exponent outside 0..8
    bad = dict(bad, params=prm)
    osc = synth.config(0)[0]
    cplx = _sector_problem(5, 902, family=8)
    mod = binding.SectorModule([good, bad, osc, cplx, good])
    assert mod.info["specialised"] == 3 and mod.info["kernels"] == 2
    assert "qmc_cspec_dp6" in mod.image(1)[1] and "qmc_spec_dp6" in mod.image(0)[1]
    # argument checks
    out = C.c_void_p()
    arr = (binding.qmc_problem * 1)()
    assert L.qmc_sector_module_create(0, arr, 0, C.byref(out)) == -3          # QMC_ERR_N
    assert L.qmc_sector_module_create(1, None, 0, C.byref(out)) == -1         # QMC_ERR_NULL
    assert L.qmc_sector_module_create(1, arr, 0, None) == -1
    assert L.qmc_sector_module_create(1, arr, 5000, C.byref(out)) == -3
    assert L.qmc_sector_module_info(None, None, None, None, None, None) == -1
    L.qmc_sector_module_destroy(None)                        # a no-op


def test_sector_module_is_bound_to_its_batch(L):
    """the workspace query (and with it the launch) refuses a batch that is not the one the module was built from"""
    probs = [_sector_problem(6, 950 + i) for i in range(3)]
    mod = binding.SectorModule(probs)

    def ws(batch):
        arr = (binding.qmc_problem * len(batch))()
        keep = []
        for i, p in enumerate(batch):
            z = np.ascontiguousarray(p["z"], dtype=np.uint64)
            keep += [z, p["params"], p["shifts"]]
            arr[i] = binding.qmc_problem(p["family"], p["dim"], p["m"], p["transform"], p["n"], p["params"].ctypes.data, len(p["params"]),
                                         z.ctypes.data, p["shifts"].ctypes.data, None)
        return L.qmc_sector_module_workspace_bytes(mod.handle, len(batch), arr), L.qmc_workspace_bytes(len(batch), arr)

    with_module, default = ws(probs)
    assert with_module > 0 and default > 0
    assert ws(probs[:2])[0] == 0                             # another count
    assert ws([probs[0], _sector_problem(5, 960), probs[2]])[0] == 0          # another dimension
    assert ws([probs[0], dict(probs[1], family=0, params=np.ones(7)), probs[2]])[0] == 0
    # another lattice, other shifts, another transform: the same module (the transform only changes the routing)
    relattice = [dict(_sector_problem(6, 950 + i, n=65537, m=9), transform=synth.TRANSFORM_BAKER) for i in range(3)]
    assert ws(relattice)[0] > 0


def test_integrate_batch_rejects_before_touching_the_device():
    """qmc_integrate_batch validates every integrand on every lattice on the host; these calls return before any CUDA call"""
    rng = synth.MT19937_64(31)
    good = dict(family=3, dim=4, transform=synth.TRANSFORM_KOROBOV + 3, params=synth.sector(rng, 4))
    ln, lz = synth.ladder(6, 4093)
    shifts = synth.draw_shifts(rng, 8, 6)
    kw = dict(min_n=1000, min_m=4, epsrel=1e-6, epsabs=0.0, maxeval=10**6)

    def status(integrands, ln=ln, lz=lz, shifts=shifts, **over):
        try:
            binding.qmc_integrate_batch(integrands, ln, lz, shifts, **dict(kw, **over))
        except binding.QmcError as e:
            return e.status
        return 0

    assert status([dict(good, dim=7)]) == -2                           # wider than the ladder
    assert status([dict(good, family=9)]) == -8
    assert status([dict(good, transform=77)]) == -7
    assert status([dict(good, params=good["params"][:-1])]) == -9
    bad_shift = shifts.copy()
    bad_shift[2, 3] = -0.25
    assert status([good], shifts=bad_shift) == -5
    bad_z = lz.copy()
    bad_z[1, 2] = 0
    assert status([good], lz=bad_z) == -4
    assert status([good], ln=ln[::-1].copy(), lz=lz[::-1].copy()) == -3          # the ladder must ascend
    assert status([good], min_m=1) == -6
    assert status([good], epsrel=-1.0) == -9
    # a shift of a component the integrand does not use is not its problem
    unused = shifts.copy()
    unused[2, 5] = 7.0
    assert status([dict(good, dim=7)], shifts=unused) == -2


def _peak_cdf_pairs(a, w, count=400):
    """marginal of the product peak 1 / (a^-2 + (x - w)^2) in closed form: pairs (CDF(x_t), x_t)"""
    x = np.linspace(0.0025, 0.9975, count)
    cdf = (np.arctan(a * (x - w)) + np.arctan(a * w)) / (np.arctan(a * (1 - w)) + np.arctan(a * w))
    return cdf, x


def test_polysingular_fit_against_the_library_solver():
    """the bounded Levenberg-Marquardt of the product (qmc_fit.cu) against the oracle's fit of the same function with the same
    bounds by scipy.optimize.least_squares: the same residual, and -- where both poles are active and the
    minimum is unique -- the same parameters; on data generated from the model both reach a zero residual"""
    def sse(a, c, e):
        return float(sum((oracle.fit_map(a, y)[0] - t) ** 2 for y, t in zip(c, e)))

    for truth in ([1.05, -0.4, 0.35, 0.0, 0.30, 0.25], [1.6, -0.03, 0.0, 0.45, 0.35, 0.10]):
        c = np.linspace(0.002, 0.998, 400)
        e = np.array([oracle.fit_map(np.array(truth), y)[0] for y in c])
        a_or, cost_or = oracle.fit_polysingular_pairs(c, e)
        assert cost_or < 1e-24                                # pins the oracle's model against the C++ oracle's fit_map
        full = binding.qmc_fit_from_cdf(e[None, :], c[None, :], with_poles=True)[0]
        assert sse(full, c, e) < 1e-24
    for a, w in ((6.0, 0.4), (12.0, 0.03), (40.0, 0.7), (3.0, 0.9)):
        c, e = _peak_cdf_pairs(a, w)
        cub = binding.qmc_fit_from_cdf(e[None, :], c[None, :], with_poles=False)[0]
        full = binding.qmc_fit_from_cdf(e[None, :], c[None, :], with_poles=True)[0]
        a_or, cost_or = oracle.fit_polysingular_pairs(c, e, start45=(cub[4], cub[5]))
        cost = sse(full, c, e)
        assert cost <= cost_or * (1 + 1e-3) + 1e-18, (a, w, cost, cost_or)
        assert cost_or <= cost * (1 + 1e-3) + 1e-18, (a, w, cost, cost_or)           # neither solver beats the other
        assert cost < 1e-3 * sse(cub, c, e)                   # the poles matter for a peak
        if full[2] > 1e-3 and full[3] > 1e-3:
            np.testing.assert_allclose(full, a_or, rtol=1e-4, atol=1e-6)
        assert binding.qmc_validate_problem_host(dict(_cfg0(), fit_coeffs=np.tile(full, (4, 1)))) == 0


def test_sector_module_sizes_its_kernels_for_large_batches():
    """with sectors_per_kernel = 0 a large batch shares kernels so that a batch call's variant limit (64) is not hit"""
    rng = synth.MT19937_64(1234)
    blocks = [synth.sector(rng, 3, n_lo=2, n_span=2) for _ in range(40)]
    probs = [synth.problem(3, blocks[i % 40], 1021, synth.korobov_form_vector(1021, 3, 341), synth.draw_shifts(rng, 2, 3),
                           synth.TRANSFORM_KOROBOV + 3, name=f"s{i}") for i in range(1600)]
    mod = binding.SectorModule(probs)
    info = mod.info
    assert info["specialised"] == 1600 and info["kernels"] <= 48 and info["kernels"] * 64 >= 1600
    assert binding.SectorModule(probs[:100], sectors_per_kernel=25).info["kernels"] == 4
