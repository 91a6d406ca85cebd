"""Thin ctypes binding of include/qmc_lattice.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libqmc_lattice.so; PyTorch supplies device
memory and streams.  There is no CPU fallback: if the library is missing or no CUDA device is
present the calls raise.  Function names mirror the C ABI.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqmc_lattice.so")

EXPORTS = [
    "qmc_lattice_integrate", "qmc_lattice_integrate_ex", "qmc_lattice_integrate_batch", "qmc_workspace_bytes",
    "qmc_validate_problem_host", "qmc_lattice_project", "qmc_project_workspace_bytes", "qmc_fit_cubic",
    "qmc_lattice_points", "qmc_finalize_means", "qmc_fp64_peak_probe", "qmc_last_launch_count", "qmc_plan_info",
    "qmc_profile_enable", "qmc_profile_last_fused_ms",
    "qmc_num_components", "qmc_status_string", "qmc_last_cuda_error", "qmc_integrate", "qmc_fit_polysingular",
    "qmc_lattice_integrate_batch_opts", "qmc_workspace_bytes_opts", "qmc_lattice_integrate_batch_host",
    "qmc_release_thread_resources", "qmc_sector_compile", "qmc_lattice_cdf_samples", "qmc_cdf_workspace_bytes",
    "qmc_cdf_sample_count", "qmc_fit_from_cdf", "qmc_sector_module_create", "qmc_sector_module_destroy", "qmc_sector_module_info",
    "qmc_sector_module_image", "qmc_lattice_integrate_batch_module", "qmc_sector_module_workspace_bytes",
    "qmc_lattice_integrate_batch_host_module", "qmc_static_scratch_bytes", "qmc_lattice_integrate_batch_static",
    "qmc_integrate_batch", "qmc_batch_create", "qmc_batch_launch", "qmc_batch_destroy",
]

QMC_OK = 0
QMC_ERR_NONFINITE = -13
QMC_ERR_MAXEVAL = -14


class QmcError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        L = lib()
        msg = L.qmc_status_string(status).decode()
        if status == -12:
            msg += ": " + L.qmc_last_cuda_error().decode()
        super().__init__(f"{where}: status {status} ({msg})")


class qmc_problem(C.Structure):
    _fields_ = [("family", C.c_int), ("dim", C.c_int), ("m", C.c_int), ("transform", C.c_int), ("n", C.c_uint64),
                ("params", C.c_void_p), ("n_params", C.c_int), ("z", C.c_void_p), ("shifts", C.c_void_p),
                ("fit_coeffs", C.c_void_p)]


class qmc_plan_options(C.Structure):
    _fields_ = [("tiles_target", C.c_int), ("force_wide", C.c_int), ("group", C.c_int), ("generic_call", C.c_int)]


class qmc_integrand(C.Structure):
    _fields_ = [("family", C.c_int), ("dim", C.c_int), ("transform", C.c_int), ("n_params", C.c_int), ("params", C.c_void_p),
                ("fit_coeffs", C.c_void_p)]


class qmc_result(C.Structure):
    _fields_ = [("integral", C.c_double * 2), ("error", C.c_double * 2), ("n", C.c_uint64), ("m", C.c_int),
                ("iterations", C.c_int), ("evaluations", C.c_uint64)]


_lib = None


def lib():
    """Loads libqmc_lattice.so (build it with `python -m paper_1811_11720_b200.build`); fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_1811_11720_b200.build` (nvcc, sm_100a)")
        L = C.CDLL(LIB_PATH)
        dp, up, vp = C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.c_void_p
        pp = C.POINTER(qmc_problem)
        L.qmc_lattice_integrate.argtypes = [C.c_int, dp, C.c_int, C.c_uint64, up, dp, C.c_int, C.c_int, dp, dp, dp]
        L.qmc_lattice_integrate_ex.argtypes = [C.c_int, dp, C.c_int, C.c_int, C.c_uint64, up, dp, C.c_int, C.c_int, dp, dp,
                                               dp, dp]
        L.qmc_lattice_integrate_batch.argtypes = [C.c_int, pp, vp, vp, vp, vp, C.c_size_t, vp]
        L.qmc_workspace_bytes.argtypes = [C.c_int, pp]
        L.qmc_workspace_bytes.restype = C.c_size_t
        po = C.POINTER(qmc_plan_options)
        L.qmc_lattice_integrate_batch_opts.argtypes = [C.c_int, pp, vp, vp, vp, vp, C.c_size_t, vp, po]
        L.qmc_workspace_bytes_opts.argtypes = [C.c_int, pp, po]
        L.qmc_workspace_bytes_opts.restype = C.c_size_t
        L.qmc_lattice_integrate_batch_host.argtypes = [C.c_int, pp, dp, dp, dp]
        L.qmc_sector_compile.argtypes = [dp, C.c_int, C.c_int, C.POINTER(C.c_ubyte), C.c_int, C.POINTER(C.c_int), dp, C.c_int,
                                         C.POINTER(C.c_int), dp]
        L.qmc_sector_module_create.argtypes = [C.c_int, pp, C.c_int, C.POINTER(vp)]
        L.qmc_sector_module_destroy.argtypes = [vp]
        L.qmc_sector_module_destroy.restype = None
        L.qmc_sector_module_info.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), dp, C.POINTER(C.c_size_t), C.POINTER(C.c_int)]
        L.qmc_sector_module_image.argtypes = [vp, C.c_int, vp, C.c_size_t, C.POINTER(C.c_size_t), C.c_char_p, C.c_size_t]
        L.qmc_lattice_integrate_batch_host_module.argtypes = [vp, C.c_int, pp, dp, dp, dp]
        L.qmc_integrate_batch.argtypes = [C.c_int, C.POINTER(qmc_integrand), vp, C.c_int, up, up, C.c_int, dp, C.c_uint64, C.c_int, C.c_int,
                                          C.c_double, C.c_double, C.c_uint64, C.c_int, C.POINTER(qmc_result), C.POINTER(C.c_int)]
        L.qmc_batch_create.argtypes = [C.c_int, pp, vp, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.qmc_batch_launch.argtypes = [vp, vp, vp, vp, vp]
        L.qmc_batch_destroy.argtypes = [vp]
        L.qmc_batch_destroy.restype = None
        L.qmc_static_scratch_bytes.restype = C.c_size_t
        L.qmc_lattice_integrate_batch_static.argtypes = [C.c_int, pp, vp, vp, vp, vp]
        L.qmc_sector_module_workspace_bytes.argtypes = [vp, C.c_int, pp]
        L.qmc_sector_module_workspace_bytes.restype = C.c_size_t
        L.qmc_lattice_integrate_batch_module.argtypes = [vp, C.c_int, pp, vp, vp, vp, vp, C.c_size_t, vp]
        L.qmc_validate_problem_host.argtypes = [pp]
        L.qmc_lattice_project.argtypes = [pp, C.c_int, vp, vp, C.c_size_t, vp]
        L.qmc_project_workspace_bytes.argtypes = [pp, C.c_int]
        L.qmc_project_workspace_bytes.restype = C.c_size_t
        L.qmc_fit_cubic.argtypes = [dp, C.c_int, C.c_int, dp]
        L.qmc_lattice_cdf_samples.argtypes = [pp, C.c_int, vp, vp, vp, C.c_size_t, vp]
        L.qmc_cdf_workspace_bytes.argtypes = [pp, C.c_int]
        L.qmc_cdf_workspace_bytes.restype = C.c_size_t
        L.qmc_cdf_sample_count.argtypes = [C.c_uint64, C.c_int]
        L.qmc_cdf_sample_count.restype = C.c_longlong
        L.qmc_fit_from_cdf.argtypes = [dp, dp, C.c_int, C.c_longlong, C.c_int, dp]
        L.qmc_fit_polysingular.argtypes = [dp, C.c_int, C.c_int, dp]
        L.qmc_lattice_points.argtypes = [C.c_uint64, C.c_int, up, dp, C.c_uint64, C.c_uint64, vp, vp, vp]
        L.qmc_finalize_means.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp]
        L.qmc_fp64_peak_probe.argtypes = [C.c_int, dp, dp, vp]
        L.qmc_plan_info.argtypes = [C.c_int, pp, C.POINTER(C.c_longlong), C.POINTER(C.c_int), C.POINTER(C.c_longlong)]
        L.qmc_num_components.argtypes = [C.c_int]
        L.qmc_profile_enable.argtypes = [C.c_int]
        L.qmc_profile_last_fused_ms.argtypes = [dp]
        L.qmc_integrate.argtypes = [C.c_int, dp, C.c_int, C.c_int, C.c_int, dp, C.c_int, up, up, dp, C.c_uint64, C.c_int, C.c_int,
                                    C.c_double, C.c_double, C.c_uint64, C.c_int, C.POINTER(qmc_result)]
        L.qmc_status_string.argtypes = [C.c_int]
        L.qmc_status_string.restype = C.c_char_p
        L.qmc_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(status, where, allow=()):
    if status != QMC_OK and status not in allow:
        raise QmcError(status, where)
    return status


def _d(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _u(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint64))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def qmc_num_components(family: int) -> int:
    return int(lib().qmc_num_components(int(family)))


def qmc_lattice_integrate(family, params, dim, n, z, shifts, m, transform, fit_coeffs=None):
    """Synchronous HOST-pointer call (north_star's signature) -> (mean, err) arrays of ncomp doubles."""
    params, shifts, fit = _f64(params), _f64(shifts), _f64(fit_coeffs)
    z = np.ascontiguousarray(z, dtype=np.uint64)
    nc = max(qmc_num_components(family), 1)
    mean, err = np.zeros(2), np.zeros(2)
    _check(lib().qmc_lattice_integrate(int(family), _d(params), int(dim), int(n), _u(z), _d(shifts), int(m), int(transform),
                                       _d(fit), _d(mean), _d(err)), "qmc_lattice_integrate")
    return mean[:nc].copy(), err[:nc].copy()


def qmc_lattice_integrate_ex(p: dict):
    """Synchronous HOST-pointer call on a problem dict (synth.problem) -> (shift_means (m, ncomp), mean, err)."""
    params, shifts, fit = _f64(p["params"]), _f64(p["shifts"]), _f64(p.get("fit_coeffs"))
    z = np.ascontiguousarray(p["z"], dtype=np.uint64)
    nc = max(qmc_num_components(p["family"]), 1)
    mean, err, sm = np.zeros(2), np.zeros(2), np.zeros((p["m"], nc))
    _check(lib().qmc_lattice_integrate_ex(p["family"], _d(params), len(params), p["dim"], p["n"], _u(z), _d(shifts), p["m"],
                                          p["transform"], _d(fit), _d(mean), _d(err), _d(sm)), "qmc_lattice_integrate_ex")
    return sm, mean[:nc].copy(), err[:nc].copy()


def qmc_lattice_integrate_batch_host(problems):
    """Synchronous HOST-pointer batch (one H2D copy of all inputs, one D2H copy of all results) ->
    (shift_means list of (m, ncomp), means (count, 2), errs (count, 2))."""
    count = len(problems)
    arr = (qmc_problem * count)()
    keep = []
    for i, p in enumerate(problems):
        params, shifts, fit = _f64(p["params"]), _f64(p["shifts"]), _f64(p.get("fit_coeffs"))
        z = np.ascontiguousarray(p["z"], dtype=np.uint64)
        keep += [params, shifts, fit, z]
        arr[i] = qmc_problem(p["family"], p["dim"], p["m"], p["transform"], p["n"], params.ctypes.data, len(params), z.ctypes.data,
                             shifts.ctypes.data, None if fit is None else fit.ctypes.data)
    max_m = max(p["m"] for p in problems)
    means, errs, sm = np.zeros((count, 2)), np.zeros((count, 2)), np.zeros((count, 2 * max_m))
    _check(lib().qmc_lattice_integrate_batch_host(count, arr, _d(means), _d(errs), _d(sm)), "qmc_lattice_integrate_batch_host")
    out = []
    for i, p in enumerate(problems):
        nc = qmc_num_components(p["family"])
        out.append(sm[i, : p["m"] * nc].reshape(p["m"], nc).copy())
    return out, means, errs


class HostBatch:
    """Problems marshalled once for repeated synchronous HOST-pointer calls (qmc_lattice_integrate_batch_host): the numpy
    arrays stay where they are, `integrate()` is the C call and nothing else."""

    def __init__(self, problems, module=None):
        self.problems = problems
        self.module = module                               # a SectorModule built from the same problems, or None
        self.count = len(problems)
        self.arr = (qmc_problem * self.count)()
        self._keep = []
        for i, p in enumerate(problems):
            params, shifts, fit = _f64(p["params"]), _f64(p["shifts"]), _f64(p.get("fit_coeffs"))
            z = np.ascontiguousarray(p["z"], dtype=np.uint64)
            self._keep += [params, shifts, fit, z]
            self.arr[i] = qmc_problem(p["family"], p["dim"], p["m"], p["transform"], p["n"], params.ctypes.data, len(params),
                                      z.ctypes.data, shifts.ctypes.data, None if fit is None else fit.ctypes.data)
        self.max_m = max(p["m"] for p in problems)
        self.means, self.errs = np.zeros((self.count, 2)), np.zeros((self.count, 2))
        self.shift_means = np.zeros((self.count, 2 * self.max_m))
        self._args = (self.count, self.arr, _d(self.means), _d(self.errs), _d(self.shift_means))
        self._fn = lib().qmc_lattice_integrate_batch_host
        if module is not None:
            self._args = (module.handle,) + self._args
            self._fn = lib().qmc_lattice_integrate_batch_host_module

    def integrate(self):
        _check(self._fn(*self._args), "qmc_lattice_integrate_batch_host")
        return self.means, self.errs


def qmc_sector_compile(params, dim):
    """The interpreter program of a sector parameter block, compiled on the device -> (steps uint8[], slots (n, 2), c0 (2,))."""
    params = _f64(params)
    nst, nsl, c0 = C.c_int(), C.c_int(), np.zeros(2)
    _check(lib().qmc_sector_compile(_d(params), len(params), int(dim), None, 0, C.byref(nst), None, 0, C.byref(nsl), _d(c0)),
           "qmc_sector_compile")
    steps = np.zeros(nst.value, dtype=np.uint8)
    slots = np.zeros((nsl.value, 2))
    _check(lib().qmc_sector_compile(_d(params), len(params), int(dim), steps.ctypes.data_as(C.POINTER(C.c_ubyte)), len(steps),
                                    C.byref(nst), _d(slots), len(slots), C.byref(nsl), _d(c0)), "qmc_sector_compile")
    return steps, slots, c0


class SectorModule:
    """qmc_sector_module_create: the real sectors of `problems` as straight-line sm_100a code (built on the host, no GPU needed).
    DeviceBatch(problems, module=...) runs them; `info` tells what was built."""

    def __init__(self, problems, sectors_per_kernel=0):
        count = len(problems)
        arr = (qmc_problem * count)()
        keep = []
        for i, p in enumerate(problems):
            params = _f64(p["params"])
            keep.append(params)
            arr[i] = qmc_problem(p["family"], p["dim"], p.get("m", 0), p.get("transform", 0), p.get("n", 0), params.ctypes.data,
                                 len(params), None, None, None)
        self.count = count
        self.handle = C.c_void_p()
        _check(lib().qmc_sector_module_create(count, arr, int(sectors_per_kernel), C.byref(self.handle)), "qmc_sector_module_create")

    @property
    def info(self):
        ns, nk, ms, nb, th = C.c_int(), C.c_int(), C.c_double(), C.c_size_t(), C.c_int()
        _check(lib().qmc_sector_module_info(self.handle, C.byref(ns), C.byref(nk), C.byref(ms), C.byref(nb), C.byref(th)),
               "qmc_sector_module_info")
        return {"specialised": ns.value, "kernels": nk.value, "build_ms": ms.value, "image_bytes": nb.value, "host_threads": th.value}

    def image(self, kernel=0):
        """(device image bytes, assembler report) of one kernel"""
        nb = C.c_size_t()
        log = C.create_string_buffer(1 << 16)
        _check(lib().qmc_sector_module_image(self.handle, int(kernel), None, 0, C.byref(nb), log, len(log)), "qmc_sector_module_image")
        buf = C.create_string_buffer(nb.value)
        _check(lib().qmc_sector_module_image(self.handle, int(kernel), buf, nb.value, None, None, 0), "qmc_sector_module_image")
        return buf.raw, log.value.decode(errors="replace")

    def close(self):
        if self.handle:
            lib().qmc_sector_module_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def qmc_release_thread_resources():
    _check(lib().qmc_release_thread_resources(), "qmc_release_thread_resources")


def qmc_integrate(family, params, dim, transform, ladder_n, ladder_z, shifts, min_n=8191, min_m=32, epsrel=0.01, epsabs=1e-7,
                  maxeval=1000000, errormode=0, fit_coeffs=None):
    """The paper's `integrate` iteration (defaults: PAPER.md L887-L905) -> (dict result, status); status is QMC_OK when the
    error goal was met and QMC_ERR_MAXEVAL when maxeval / the ladder / the shifts ran out (the last result is returned)."""
    params, shifts, fit = _f64(params), _f64(shifts), _f64(fit_coeffs)
    ln = np.ascontiguousarray(ladder_n, dtype=np.uint64)
    lz = np.ascontiguousarray(ladder_z, dtype=np.uint64).reshape(len(ln), int(dim))
    nc = max(qmc_num_components(family), 1)
    res = qmc_result()
    st = _check(lib().qmc_integrate(int(family), _d(params), len(params), int(dim), int(transform), _d(fit), len(ln), _u(ln), _u(lz),
                                    _d(shifts), int(min_n), int(min_m), int(shifts.shape[0]), float(epsrel), float(epsabs),
                                    int(maxeval), int(errormode), C.byref(res)), "qmc_integrate", allow=(QMC_ERR_MAXEVAL,))
    return {"integral": np.array(res.integral[:nc]), "error": np.array(res.error[:nc]), "n": int(res.n), "m": int(res.m),
            "iterations": int(res.iterations), "evaluations": int(res.evaluations)}, st


def qmc_integrate_batch(integrands, ladder_n, ladder_z, shifts, module=None, min_n=8191, min_m=32, epsrel=0.01, epsabs=1e-7,
                        maxeval=1000000, errormode=0):
    """qmc_integrate for many integrands at once (dicts with family, params, dim, transform[, fit_coeffs]); the lattice evaluations
    of a round share one batched launch -> (list of result dicts, list of statuses, overall status)."""
    count = len(integrands)
    arr = (qmc_integrand * count)()
    keep = []
    for i, g in enumerate(integrands):
        params, fit = _f64(g["params"]), _f64(g.get("fit_coeffs"))
        keep += [params, fit]
        arr[i] = qmc_integrand(int(g["family"]), int(g["dim"]), int(g["transform"]), len(params), params.ctypes.data,
                               None if fit is None else fit.ctypes.data)
    ln = np.ascontiguousarray(ladder_n, dtype=np.uint64)
    lz = np.ascontiguousarray(ladder_z, dtype=np.uint64)
    shifts = _f64(shifts)
    ladder_dim = int(shifts.shape[1])
    assert lz.shape == (len(ln), ladder_dim)
    res = (qmc_result * count)()
    sts = (C.c_int * count)()
    st = _check(lib().qmc_integrate_batch(count, arr, None if module is None else module.handle, len(ln), _u(ln), _u(lz), ladder_dim,
                                          _d(shifts), int(min_n), int(min_m), int(shifts.shape[0]), float(epsrel), float(epsabs),
                                          int(maxeval), int(errormode), res, sts), "qmc_integrate_batch",
                allow=(QMC_ERR_MAXEVAL, QMC_ERR_NONFINITE))
    out = []
    for i, g in enumerate(integrands):
        nc = max(qmc_num_components(g["family"]), 1)
        r = res[i]
        out.append({"integral": np.array(r.integral[:nc]), "error": np.array(r.error[:nc]), "n": int(r.n), "m": int(r.m),
                    "iterations": int(r.iterations), "evaluations": int(r.evaluations)})
    return out, [int(v) for v in sts], st


def qmc_validate_problem_host(p: dict) -> int:
    params, shifts, fit = _f64(p["params"]), _f64(p["shifts"]), _f64(p.get("fit_coeffs"))
    z = np.ascontiguousarray(p["z"], dtype=np.uint64)
    s = qmc_problem(p["family"], p["dim"], p["m"], p["transform"], p["n"], params.ctypes.data, len(params), z.ctypes.data,
                    shifts.ctypes.data, None if fit is None else fit.ctypes.data)
    return int(lib().qmc_validate_problem_host(C.byref(s)))


def qmc_fit_cubic(hist):
    H = _f64(hist)
    d, bins = H.shape
    out = np.zeros((d, 6))
    _check(lib().qmc_fit_cubic(_d(H), d, bins, _d(out)), "qmc_fit_cubic")
    return out


def qmc_fit_from_cdf(x, cdf, with_poles=False):
    """Fit of Eq. 19 (cubic sub-family, or complete with pole terms) to the sort-based CDF samples -> (dim, 6)."""
    X, Cd = _f64(x), _f64(cdf)
    d, K = X.shape
    out = np.zeros((d, 6))
    _check(lib().qmc_fit_from_cdf(_d(X), _d(Cd), d, K, 1 if with_poles else 0, _d(out)), "qmc_fit_from_cdf")
    return out


def qmc_fit_polysingular(hist):
    """Bounded Levenberg-Marquardt fit of the complete fit function of Eq. 19 -> (dim, 6) coefficients a_0..a_5."""
    H = _f64(hist)
    d, bins = H.shape
    out = np.zeros((d, 6))
    _check(lib().qmc_fit_polysingular(_d(H), d, bins, _d(out)), "qmc_fit_polysingular")
    return out


class DeviceBatch:
    """Device-resident batch of problems for the stream-ordered entry points (torch owns the memory).

    Uploads the inputs once; `integrate()` then issues qmc_lattice_integrate_batch on torch's current
    stream without synchronising.  Outputs are torch tensors: means/errs (count, 2), shift_means
    (count, 2*max_m).
    """

    def __init__(self, problems, device="cuda:0", tiles_target=0, force_wide=False, module=None, group=0, generic_call=False):
        import torch
        self.module = module                               # a SectorModule built from the same problems, or None
        self.opts = qmc_plan_options(int(tiles_target), 1 if force_wide else 0, int(group), 1 if generic_call else 0)
        self.torch = torch
        self.device = torch.device(device)
        self.problems = problems
        self.count = len(problems)
        self._keep = []
        arr = (qmc_problem * self.count)()
        for i, p in enumerate(problems):
            t_params = torch.from_numpy(_f64(p["params"])).to(self.device)
            t_z = torch.from_numpy(np.ascontiguousarray(p["z"], dtype=np.uint64).view(np.int64)).to(self.device)
            t_sh = torch.from_numpy(_f64(p["shifts"])).to(self.device)
            fit = p.get("fit_coeffs")
            t_fit = None if fit is None else torch.from_numpy(_f64(fit)).to(self.device)
            self._keep += [t_params, t_z, t_sh, t_fit]
            arr[i] = qmc_problem(p["family"], p["dim"], p["m"], p["transform"], p["n"], t_params.data_ptr(),
                                 t_params.numel(), t_z.data_ptr(), t_sh.data_ptr(),
                                 None if t_fit is None else t_fit.data_ptr())
        self.arr = arr
        self.max_m = max(p["m"] for p in problems)
        self.ws_bytes = int(lib().qmc_workspace_bytes_opts(self.count, arr, C.byref(self.opts)))
        if module is not None and self.ws_bytes:
            with_module = int(lib().qmc_sector_module_workspace_bytes(module.handle, self.count, arr))
            if with_module == 0:
                raise QmcError(-10, "qmc_sector_module_workspace_bytes (the module was built from another batch)")
            self.ws_bytes = max(self.ws_bytes, with_module)
        if self.ws_bytes == 0:
            st = lib().qmc_plan_info(self.count, arr, None, None, None)
            raise QmcError(st if st != 0 else -11, "qmc_workspace_bytes")
        self.workspace = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 256
        self.ws_ptr = self.workspace.data_ptr() + off
        self.means = torch.zeros(self.count, 2, dtype=torch.float64, device=self.device)
        self.errs = torch.zeros(self.count, 2, dtype=torch.float64, device=self.device)
        self.shift_means = torch.zeros(self.count, 2 * self.max_m, dtype=torch.float64, device=self.device)

    def plan_info(self):
        tiles, ctas, tl0 = C.c_longlong(), C.c_int(), C.c_longlong()
        _check(lib().qmc_plan_info(self.count, self.arr, C.byref(tiles), C.byref(ctas), C.byref(tl0)), "qmc_plan_info")
        return {"tiles": tiles.value, "ctas": ctas.value, "tile_len0": tl0.value}

    def integrate(self, stream=None):
        """qmc_lattice_integrate_batch on `stream` (default: torch's current stream); returns launch count."""
        s = self.torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        if self.module is not None:
            _check(lib().qmc_lattice_integrate_batch_module(self.module.handle, self.count, self.arr, self.means.data_ptr(),
                                                            self.errs.data_ptr(), self.shift_means.data_ptr(), self.ws_ptr,
                                                            self.ws_bytes, s), "qmc_lattice_integrate_batch_module")
            return int(lib().qmc_last_launch_count())
        _check(lib().qmc_lattice_integrate_batch_opts(self.count, self.arr, self.means.data_ptr(), self.errs.data_ptr(),
                                                      self.shift_means.data_ptr(), self.ws_ptr, self.ws_bytes, s, C.byref(self.opts)),
               "qmc_lattice_integrate_batch")
        return int(lib().qmc_last_launch_count())

    def prepare(self, stream=None):
        """qmc_batch_create on this batch's workspace: plan, upload and prepare once; launch() is then kernel launches only"""
        s = self.torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        self.release()
        handle = C.c_void_p()
        _check(lib().qmc_batch_create(self.count, self.arr, None if self.module is None else self.module.handle, self.ws_ptr,
                                      self.ws_bytes, s, C.byref(handle)), "qmc_batch_create")
        self.prepared = handle
        return self

    def launch(self, stream=None):
        """qmc_batch_launch (after prepare()); returns launch count"""
        s = self.torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        _check(lib().qmc_batch_launch(self.prepared, self.means.data_ptr(), self.errs.data_ptr(), self.shift_means.data_ptr(), s),
               "qmc_batch_launch")
        return int(lib().qmc_last_launch_count())

    def release(self):
        if getattr(self, "prepared", None):
            lib().qmc_batch_destroy(self.prepared)
        self.prepared = None

    def __del__(self):
        try:
            self.release()
        except Exception:
            pass

    def integrate_static(self, stream=None):
        """qmc_lattice_integrate_batch_static: the same call with the library's static scratch array as workspace (nothing is
        allocated; batches whose workspace exceeds qmc_static_scratch_bytes() are rejected); returns launch count."""
        s = self.torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        _check(lib().qmc_lattice_integrate_batch_static(self.count, self.arr, self.means.data_ptr(), self.errs.data_ptr(),
                                                        self.shift_means.data_ptr(), s), "qmc_lattice_integrate_batch_static")
        return int(lib().qmc_last_launch_count())

    def capture(self):
        """Captures one integrate() call in a CUDA graph and returns the torch.cuda.CUDAGraph (call .replay()).  A call for
        ONE closed-form problem is two kernel launches plus at most one 8-byte memset, all stream-ordered and capturable; a
        batch call uploads its plan from pageable host memory and cannot be captured (the library then returns QMC_ERR_CUDA)."""
        torch = self.torch
        qmc_profile_enable(False)                          # event records do not belong in a graph
        self.integrate()                                    # warm-up outside the capture (module load, occupancy cache)
        torch.cuda.synchronize(self.device)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            self.integrate()
        return graph

    def results(self):
        """Synchronises and returns numpy (shift_means list of (m, ncomp), means (count, ncomp_max), errs)."""
        self.torch.cuda.synchronize(self.device)
        sm = self.shift_means.cpu().numpy()
        means, errs = self.means.cpu().numpy(), self.errs.cpu().numpy()
        out = []
        for i, p in enumerate(self.problems):
            nc = qmc_num_components(p["family"])
            out.append(sm[i, : p["m"] * nc].reshape(p["m"], nc).copy())
        return out, means, errs

    def cdf_samples(self, index=0, fitstepsize=10, stream=None, sync=True):
        """qmc_lattice_cdf_samples for problem `index` -> torch tensors (x (dim, K), cdf (dim, K)) on the device."""
        torch = self.torch
        p = self.problems[index]
        one = (qmc_problem * 1)(self.arr[index])
        K = int(lib().qmc_cdf_sample_count(p["n"], int(fitstepsize)))
        need = int(lib().qmc_cdf_workspace_bytes(one, int(fitstepsize)))
        if K == 0 or need == 0:
            raise QmcError(-3, "qmc_cdf_workspace_bytes")
        ws = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        ptr = ws.data_ptr() + ((-ws.data_ptr()) % 256)
        xs = torch.zeros(p["dim"], K, dtype=torch.float64, device=self.device)
        cdf = torch.zeros(p["dim"], K, dtype=torch.float64, device=self.device)
        s = torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        _check(lib().qmc_lattice_cdf_samples(one, int(fitstepsize), xs.data_ptr(), cdf.data_ptr(), ptr, need, s), "qmc_lattice_cdf_samples")
        if sync:
            torch.cuda.synchronize(self.device)
        else:
            self._keep_ws = (ws, xs, cdf)
        return xs, cdf

    def project(self, index=0, bins=256, stream=None, sync=True):
        """qmc_lattice_project for problem `index` -> torch tensor (dim, bins) on the device."""
        torch = self.torch
        p = self.problems[index]
        one = (qmc_problem * 1)(self.arr[index])
        need = int(lib().qmc_project_workspace_bytes(one, int(bins)))
        if need == 0:
            raise QmcError(-11, "qmc_project_workspace_bytes")
        ws = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
        ptr = ws.data_ptr() + ((-ws.data_ptr()) % 256)
        hist = torch.zeros(p["dim"], bins, dtype=torch.float64, device=self.device)
        s = torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        _check(lib().qmc_lattice_project(one, int(bins), hist.data_ptr(), ptr, need, s), "qmc_lattice_project")
        if sync:
            torch.cuda.synchronize(self.device)
        else:
            self._keep_ws = (ws, hist)                      # stream-ordered: keep the buffers alive until the caller synchronises
        return hist


def qmc_lattice_points(n, z, shift, k0, count, device="cuda:0"):
    """Residues (count, dim) uint64 and coordinates (count, dim) float64 from the device generator."""
    import torch
    z = np.ascontiguousarray(z, dtype=np.uint64)
    shift = _f64(shift)
    d = len(z)
    r = torch.zeros(max(count, 1), d, dtype=torch.int64, device=device)
    u = torch.zeros(max(count, 1), d, dtype=torch.float64, device=device)
    s = torch.cuda.current_stream(torch.device(device)).cuda_stream
    _check(lib().qmc_lattice_points(int(n), d, _u(z), _d(shift), int(k0), int(count), r.data_ptr(), u.data_ptr(), s),
           "qmc_lattice_points")
    torch.cuda.synchronize()
    return r.cpu().numpy().view(np.uint64)[:count], u.cpu().numpy()[:count]


def qmc_finalize_means(shift_means, device="cuda:0"):
    """Eq. 3 on the device for given per-shift means (m, ncomp) -> (mean, err)."""
    import torch
    sm = _f64(shift_means)
    if sm.ndim == 1:
        sm = sm.reshape(-1, 1)
    m, nc = sm.shape
    t = torch.from_numpy(sm).to(device)
    mean = torch.zeros(nc, dtype=torch.float64, device=device)
    err = torch.zeros(nc, dtype=torch.float64, device=device)
    s = torch.cuda.current_stream(torch.device(device)).cuda_stream
    _check(lib().qmc_finalize_means(t.data_ptr(), m, nc, mean.data_ptr(), err.data_ptr(), s), "qmc_finalize_means")
    torch.cuda.synchronize()
    return mean.cpu().numpy(), err.cpu().numpy()


def qmc_fp64_peak_probe(iters=20000):
    """-> (thread-level FP64 instructions per second, kernel ms) from the DFMA-chain probe."""
    rate, ms = C.c_double(), C.c_double()
    _check(lib().qmc_fp64_peak_probe(int(iters), C.byref(rate), C.byref(ms), None), "qmc_fp64_peak_probe")
    return rate.value, ms.value


def qmc_profile_enable(on=True):
    """Bracket the fused-kernel launches of later batch calls (this host thread) with CUDA events."""
    _check(lib().qmc_profile_enable(1 if on else 0), "qmc_profile_enable")


def qmc_profile_last_fused_ms():
    """Device time (ms) of the fused kernels of the last batch call; synchronises on its closing event."""
    ms = C.c_double()
    _check(lib().qmc_profile_last_fused_ms(C.byref(ms)), "qmc_profile_last_fused_ms")
    return ms.value
