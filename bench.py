#!/usr/bin/env python
"""bench.py -- throughput of the rank-1 shifted lattice hot path on B200 (BASELINE.json metric:
fp64 lattice-point integrand evaluations per second, and the fraction of the FP64 issue-rate roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--main-only]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (prepare, fused persistent kernel,
finalize) over one batch of synthetic input through the C ABI (qmc_lattice_integrate_batch).  The headline
workload is the largest single-GPU configuration, BASELINE.json configs[4] (2.15e10 evaluations per step); configs[1],
[2], [3] carry the same roofline record under "roofline_all" (configs[0] is the small parity case) and every config is
timed under "others".  Inputs are seeded and synthetic (paper_1811_11720_b200.synth).

Multi-GPU: the path has no exchange step: every rank integrates its own
independent problems (same shapes, rank-specific seeds); weak scaling; the only communication is the
MAX-reduction of the measured time.  `python bench.py --gpus N` starts its own N ranks (torch.distributed.run,
127.0.0.1) when it is not already running under torchrun.  `--impl reference` times the CPU oracle (oracle/) on the
host cores, on a stated sub-range of the same workload's lattice indices.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1811_11720_b200 import synth  # noqa: E402

METRIC = "fp64 lattice-point integrand evaluations per second"
UNIT = "evals/s"
MAIN_CONFIG = 4
ORACLE_SAMPLE_DIV = 64          # the oracle legs run about 1/64 of the workload's evaluations (oracle_sample)

# Algorithmic FP64-pipe instructions per integrand evaluation (thread level; FMA, MUL, ADD each count 1), derived in
# DESIGN.md section 5 from the method itself.  Per dimension: coordinate (1 FMA) + wrap/centre (1 ADD) = 2; transform: none 0,
# baker 1, Korobov-3 7 (c^2, 1/4 - c^2, weight product, 3-term Horner, phi); cubic fit map 6; integrand term: oscillatory 1,
# product peak 3, complex exp*poly 3.  Per evaluation: Korobov weight 3 (+1 with the fit Jacobian); cos 14 / sincos 21
# (executed counts of the libdevice fast paths); reciprocal 5; accumulate 1 per component (+1 for the complex amplitude).
# Sector family: steps of the greedy Horner programs of U and F (mean 30.61 over the 256 seeded sectors, one fp64 instruction per
# point each: tests/test_gpu_parity.py::test_sector_programs_evaluate_their_polynomials; the monomial-by-monomial count of
# round 1 was 44.44) + prefactor (mean 3.04) + powers (a: mean 1.51, b: mean 1.50) + weight*numerator 1.  These are the
# numerators of roofline.achieved (the USEFUL fraction); EXECUTED_FP64_PER_EVAL below gives the issue fraction.
ALG_FP64_PER_EVAL = {
    0: 4 * (2 + 7 + 1) + 3 + 14 + 1,                                  # 58   d=4 osc, Korobov-3
    1: 8 * (2 + 1 + 3) + 5 + 1,                                       # 54   d=8 product peak, baker
    2: 12 * (2 + 7 + 3) + 3 + 21 + 1 + 2,                             # 171  d=12 complex, Korobov-3
    3: 6 * (2 + 7) + 3 + 30.61 + 3.04 + 1.51 + 1.50 + 1 + 5 + 1,      # 100.7 d=6 sector, Korobov-3
    4: 16 * (2 + 7 + 6 + 1) + 4 + 14 + 1,                             # 275  d=16 osc, Korobov-3 + cubic map
}
# thread-level FP64-pipe instructions per evaluation the fused kernels EXECUTE (ncu smsp__inst_executed_pipe_fp64 x 32 / evaluations;
# profiles/r2_dram_full.md): the conversion of the residues, padded slots and the interpreter's bookkeeping on top of the above
EXECUTED_FP64_PER_EVAL = {1: 55.03, 2: 171.4, 3: 101.42, "3s": 100.44, 4: 279.29}     # "3s": configs[3] through the specialised kernels (profiles/r2_spec_full.md)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the fused kernel at FULL size (ncu, profiles/r2_dram_full.md)
PROFILED_DRAM_BYTES_PER_LAUNCH = {1: 70400, 2: 244992, 3: 1072640, "3s": 328320, 4: 207872}   # "3s": mean of the 8 launches of a step
FP64_LANES_PER_SM = 64                        # B200 (sm_100): 64 FP64 FMA lanes per SM -> nominal peak


def workload_name(c):
    d, n, m = synth.CONFIG_SHAPES[c]
    return {0: f"configs[0] d=4 Genz oscillatory, n={n}, m={m}, Korobov r=3",
            1: f"configs[1] d=8 Genz product peak, n={n}, m={m}, baker",
            2: f"configs[2] d=12 complex exp*poly, n={n}, m={m}, Korobov r=3",
            3: f"configs[3] 256 sector-like integrands d=6, n={n}, m={m}, Korobov r=3",
            4: f"configs[4] d=16 Genz oscillatory + cubic ICDF fit map, n={n}, m={m}, Korobov r=3"}[c]


def evals_of(problems):
    return float(sum(p["n"] * p["m"] for p in problems))


SHRINK = 1        # --shrink S (profiling runs only): 1/S of the work of every config, same kernels and tile shapes


EXTRA_SHIFT_FACTOR = 4  # time-to-target: up to 4 m shifts on the largest lattice
SECTOR_LOG = False    # --sector-log: configs[3]'s sectors with the log factors of an eps-expansion term (reading C-15)
# per evaluation on top of configs[3]: 2 logarithms (26 FP64 each: DESIGN.md section 9) + combination 3 + power (mean p - 1 = 1) + product 1
ALG_FP64_SECTOR_LOG_EXTRA = 2 * 26 + 3 + 1 + 1


def with_log_factors(probs):
    out = []
    for i, p in enumerate(probs):
        rng = synth.MT19937_64(synth.SECTOR_SEED + 5000 + i)
        tail = np.array([rng.uniform_range(0.5, 2.0), rng.uniform_range(-3.0, -1.0), float(1 + rng.next_u64() % 3)])
        out.append(dict(p, params=np.concatenate([p["params"], tail]), name=p["name"] + ".log"))
    return out


def shrunk_config(c):
    if c == 3 and SECTOR_LOG:
        return with_log_factors(synth.config(3, count_override=max(1, 256 // SHRINK)))
    if SHRINK <= 1:
        return synth.config(c)
    if c == 3:
        return synth.config(3, count_override=max(1, 256 // SHRINK))
    from paper_1811_11720_b200 import cbc
    n = synth.CONFIG_SHAPES[c][1] // SHRINK
    while not cbc.is_prime(n):
        n -= 1
    return synth.config(c, n_override=n)


def rank_problems(c, rank):
    """Problems of BASELINE.json configs[c] for `rank`: rank 0 gets exactly the seeded config; other ranks
    get the same shapes with rank-specific shifts (independent problems -> no data-path collective)."""
    probs = shrunk_config(c)
    if rank == 0:
        return probs
    out = []
    for i, p in enumerate(probs):
        rng = synth.MT19937_64(synth.CONFIG_SEED + 7919 * rank + 104729 * c + i)
        out.append(dict(p, shifts=synth.draw_shifts(rng, p["m"], p["dim"]), name=f"{p['name']}.rank{rank}"))
    return out


def aggregate(per_rank_evals, max_seconds):
    """whole-job throughput: all ranks' evaluations over the slowest rank's time"""
    return float(sum(per_rank_evals)) / max_seconds


# ----------------------------------------------------------------------------------------------------
# clocks sampling during the timed region (NVML; nvidia-smi fallback)
# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index):
        self.samples, self.stop_flag, self.thread, self.h, self.sm_max = [], False, None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                self.samples.append((time.perf_counter(), nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM),
                                     nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0,
                                     nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                                     if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons")
                                     else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)))
            except Exception:
                pass
            time.sleep(0.01)

    def start(self):
        if self.nv is not None:
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()

    def stop(self):
        self.stop_flag = True
        if self.thread is not None:
            self.thread.join()

    def summary(self, windows):
        """median SM clock over the samples that fall inside the timed windows [(t0, t1), ...]"""
        inside = [s for s in self.samples if any(a <= s[0] <= b for a, b in windows)] or self.samples
        if not inside:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0}
        mask = 0
        for s in inside:
            mask |= int(s[3])
        reasons = [name for bit, name in self.REASONS.items() if mask & bit and name != "gpu_idle"]
        return {"sm_mhz": float(statistics.median(s[1] for s in inside)), "sm_max_mhz": self.sm_max,
                "power_w_max": max(s[2] for s in inside), "reasons": reasons, "samples": len(inside)}


# ----------------------------------------------------------------------------------------------------
# GPU arm
# ----------------------------------------------------------------------------------------------------
class L2Flusher:
    """writes a buffer larger than the 126 MB L2 between timed iterations (outside the timed events)"""

    def __init__(self, torch, device):
        self.buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=device)

    def __call__(self):
        self.buf.fill_(1)


def time_steps(torch, binding, batch, steps, warmup, flush):
    """-> (per-step ms list (CUDA events on the launching stream), fused-kernel ms list, launches per step)"""
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        flush()
        batch.integrate()
    torch.cuda.synchronize()
    step_ms, fused_ms, launches = [], [], 0
    for _ in range(steps):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        launches = batch.integrate()
        e1.record(stream)
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        fused_ms.append(binding.qmc_profile_last_fused_ms())
    return step_ms, fused_ms, launches


def config4_with_device_fit(binding, probs):
    """configs[4]: fit coefficients from the DEVICE projection pass + the library's host fit (no oracle)."""
    p = probs[0]
    proj = dict(p, n=synth.CONFIG4_NFIT, z=synth.genvec(synth.CONFIG4_NFIT, p["dim"]), transform=synth.TRANSFORM_NONE)
    H = binding.DeviceBatch([proj]).project(0, synth.PROJECTION_BINS).cpu().numpy()
    return [dict(p, fit_coeffs=binding.qmc_fit_cubic(H))]


def e2e_host_api(binding, probs, reps, module=None):
    """The same metric through the synchronous HOST-pointer C-ABI call (qmc_lattice_integrate_batch_host; one problem or a
    whole batch in ONE call): validation, the host->device copy of all inputs from pinned staging memory, the kernels, the
    device->host copy of the results and the synchronisation are all inside the timed region (host wall clock around a
    blocking call)."""
    h2d = d2h = 0
    for p in probs:
        h2d += p["params"].nbytes + p["z"].nbytes + p["shifts"].nbytes + (0 if p.get("fit_coeffs") is None else p["fit_coeffs"].nbytes)
    d2h = len(probs) * (4 + 2 * max(p["m"] for p in probs)) * 8
    hb = binding.HostBatch(probs, module=module)            # argument structs built once; the timed call is the C entry
    hb.integrate()                                          # warm-up (module load, staging arena)
    t0 = time.perf_counter()
    for _ in range(reps):
        hb.integrate()
    dt = (time.perf_counter() - t0) / reps
    return dt, h2d, d2h


def variant_workloads():
    """-> [(label, problems, algorithmic FP64 instructions per evaluation, timed steps)]: workloads outside BASELINE.json's configs
    that exercise the generic tile loop (every transform of Table A.2 other than none / baker / Korobov-3, pole-term fit, P:L1054-L1060,
    Eq. 19) and the complex sector family (reading C-16), on the shapes of configs[2], [4] (at n / 8) and [3]."""
    K, S, KA = synth.TRANSFORM_KOROBOV, synth.TRANSFORM_SIDI, synth.TRANSFORM_KOROBOV_ASYM
    out = []
    p2 = synth.config(2)[0]
    d = p2["dim"]
    fam2 = 3 * d + 21 + 1 + 2                           # integrand terms, sincos, accumulate, amplitude (as configs[2])
    for name, tr, per_coord, per_point in [("Korobov r=1", K + 1, 2 + 5, 1), ("Korobov r=2", K + 2, 2 + 6, 2),
                                           ("Korobov (5,3)", KA + 16 * 5 + 3, 2 + 21.5, 1), ("Sidi r=3", S + 3, 2 + 38, 1)]:
        out.append((f"configs[2] shape (d=12 complex exp*poly, n={p2['n']}, m={p2['m']}) with {name} [variant]",
                    [dict(p2, transform=tr, name=f"cfg2.{name}")], d * per_coord + per_point + fam2, 5))
    from paper_1811_11720_b200 import cbc
    n4 = synth.CONFIG_SHAPES[4][1] // 8
    while not cbc.is_prime(n4):
        n4 -= 1
    p4 = synth.config(4, n_override=n4)[0]
    rng = synth.MT19937_64(synth.CONFIG_SEED + 4040)
    fit = np.array([[1.001 + 0.5 * rng.uniform(), -0.001 - 0.5 * rng.uniform(), 0.25 * rng.uniform(), 0.25 * rng.uniform(),
                     0.45 + 0.3 * rng.uniform(), 0.2 * rng.uniform() - 0.05] for _ in range(p4["dim"])])
    # pole terms: two reciprocals (5 + 1 each), k q, y e, a e q: 2 x (6 + 1 + 1 + 2) = 20 on top of the cubic map's 6
    out.append((f"configs[4] shape at n/8 (d=16 oscillatory, n={n4}, m={p4['m']}) with the complete fit function of Eq. 19 (pole terms) [variant]",
                [dict(p4, fit_coeffs=fit, name="cfg4.polefit")], 16 * (2 + 7 + 6 + 20 + 1) + 4 + 14 + 1, 3))
    probs = []
    for i in range(256):
        rng = synth.MT19937_64(synth.SECTOR_SEED + 20000 + i)
        prm = synth.sector_complex(rng, 6)
        q = synth.config(3, count_override=1)[0]
        probs.append(dict(q, family=synth.FAMILY_SECTOR_COMPLEX, params=prm, shifts=synth.draw_shifts(rng, q["m"], 6), name=f"csector{i}"))
    # coordinates 6 x 9 + weight 3; complex Horner programs 2 x 30.6; prefactor 3; U^a 1.5 x 4; F^b 2.5 x 4; division 13; accumulate 2
    out.append(("configs[3] shape (256 sectors, d=6, n=4194301, m=16) with complex coefficients: family 8, contour-deformed shape [variant]",
                probs, 6 * 9 + 3 + 2 * 30.6 + 3 + 6 + 10 + 13 + 2, 3))
    return out


def closed_form(c, prm):
    """exact integrals of the closed-form configs (Genz families 1, 2: PAPER.md L709-L713; complex exp*poly): analysis only"""
    d = synth.CONFIG_SHAPES[c][0]
    if c in (0, 4):
        a = prm[1:]
        return complex(np.cos(2 * np.pi * prm[0] + 0.5 * a.sum()) * np.prod(np.sin(a / 2) / (a / 2)))
    if c == 1:
        cc, w = prm[:d], prm[d:]
        return complex(np.prod(cc * (np.arctan(cc * (1 - w)) + np.arctan(cc * w))))
    a, b = prm[:d].astype(complex), prm[d:]
    e = np.exp(1j * a)
    return complex(np.prod((e - 1) / (1j * a) + b * (e / (1j * a) - (e - 1) / (1j * a) ** 2)))


def genz_exact(fam, prm, d):
    """analytic integrals of the six Genz functions over the unit cube: analysis only"""
    from math import factorial
    from scipy.special import erf
    if fam == synth.FAMILY_GENZ_OSC:
        a = prm[1:]
        return float(np.cos(2 * np.pi * prm[0] + 0.5 * a.sum()) * np.prod(np.sin(a / 2) / (a / 2)))
    c = prm[:d]
    if fam == synth.FAMILY_GENZ_PRODPEAK:
        w = prm[d:]
        return float(np.prod(c * (np.arctan(c * (1 - w)) + np.arctan(c * w))))
    if fam == synth.FAMILY_GENZ_CORNER:
        tot = 0.0
        for mask in range(1 << d):
            sel = [j for j in range(d) if mask >> j & 1]
            tot += (-1.0) ** len(sel) / (1.0 + sum(c[j] for j in sel))
        return tot / (factorial(d) * np.prod(c))
    if fam == synth.FAMILY_GENZ_GAUSSIAN:
        w = prm[d:]
        return float(np.prod(np.sqrt(np.pi) / (2 * c) * (erf(c * (1 - w)) + erf(c * w))))
    if fam == synth.FAMILY_GENZ_C0:
        w = prm[d:]
        return float(np.prod((2.0 - np.exp(-c * w) - np.exp(-c * (1 - w))) / c))
    b = np.ones(d)
    b[:min(d, 2)] = prm[d:]
    return float(np.prod(np.expm1(c * b) / c))


def genz_table(binding, transform, dims=(5, 8, 10), sets=10, m=32, epsrel=1e-8, maxeval=7 * 10 ** 8):
    """The protocol of the paper's Table 1 / Table 2: per family and dimension, `sets` random parameter
    sets at the family's difficulty, eps_rel = 1e-8, at most 7e8 samples, 32 shifts; average correct digits
    (against the analytic result) and seconds per integration through qmc_integrate on the committed lattice ladder."""
    fams = [synth.FAMILY_GENZ_OSC, synth.FAMILY_GENZ_PRODPEAK, synth.FAMILY_GENZ_CORNER, synth.FAMILY_GENZ_GAUSSIAN,
            synth.FAMILY_GENZ_C0, synth.FAMILY_GENZ_DISCONT]
    rows = []
    for fi, fam in enumerate(fams):
        for d in dims:
            ln, lz = synth.ladder(d, 16777213)
            rng = synth.MT19937_64(1811117400 + 100 * fi + d)
            digits, secs, evals = [], [], []
            for k in range(sets + 1):                       # set 0 is the warm-up
                prm = synth.genz_protocol(rng, fam, d)
                sh = synth.draw_shifts(rng, m, d)
                t0 = time.perf_counter()
                res, st = binding.qmc_integrate(fam, prm, d, transform, ln, lz, sh, min_n=1000, min_m=m, epsrel=epsrel, epsabs=0.0,
                                                maxeval=maxeval)
                dt = time.perf_counter() - t0
                if k == 0:
                    continue
                exact = genz_exact(fam, prm, d)
                rel = abs(res["integral"][0] - exact) / abs(exact)
                digits.append(-np.log10(max(rel, 1e-16)))
                secs.append(dt)
                evals.append(res["evaluations"])
            rows.append({"family": fi + 1, "d": d, "digits": float(np.mean(digits)), "seconds": float(np.mean(secs)),
                         "evaluations": float(np.mean(evals))})
    return rows


def time_to_target(binding, c, probs, epsrel=1e-8):
    """BASELINE metric part 3: wall time of the paper's iteration (qmc_integrate) to an ESTIMATED relative
    error of 1e-8 on the committed lattice ladder, shifts and parameters of configs[c]; earlier lattices are discarded (L357)."""
    p = probs[0]
    ln, lz = synth.ladder(p["dim"], p["n"])
    # the config's m shifts first, then seeded extra shifts up to 4 m for the shift-extension leg of the iteration (the ladder
    # ends at the config's own n)
    rng = synth.MT19937_64(synth.CONFIG_SEED + 900 + c)
    shifts = np.concatenate([p["shifts"], synth.draw_shifts(rng, EXTRA_SHIFT_FACTOR * p["m"] - p["m"], p["dim"])])
    kw = dict(min_n=1000, min_m=p["m"], epsrel=epsrel, epsabs=0.0, maxeval=2 ** 62, fit_coeffs=p.get("fit_coeffs"))
    binding.qmc_integrate(p["family"], p["params"], p["dim"], p["transform"], ln[:1], lz[:1], p["shifts"], **kw)   # warm-up
    t0 = time.perf_counter()
    res, st = binding.qmc_integrate(p["family"], p["params"], p["dim"], p["transform"], ln, lz, shifts, **kw)
    dt = time.perf_counter() - t0
    exact = closed_form(c, p["params"])
    est = complex(*res["integral"]) if len(res["integral"]) == 2 else complex(res["integral"][0])
    return {"workload": workload_name(c), "target_rel_err": epsrel, "reached": st == 0, "seconds": dt, "n": res["n"], "m": res["m"],
            "iterations": res["iterations"], "evaluations": res["evaluations"],
            "estimated_rel_err": float(max(res["error"]) / abs(est)), "true_rel_err": abs(est - exact) / abs(exact),
            "max_m": int(shifts.shape[0]), "ladder": [int(v) for v in ln]}


def time_to_target_batch(binding, probs, epsrel=1e-8):
    """configs[3]: every sector through qmc_integrate on its own (estimate-only criterion, no closed form); the time is
    for the whole batch of 256 sectors, one after the other."""
    ln, lz = synth.ladder(probs[0]["dim"], probs[0]["n"])
    kw = dict(min_n=1000, min_m=probs[0]["m"], epsrel=epsrel, epsabs=0.0, maxeval=2 ** 62)
    p0 = probs[0]
    binding.qmc_integrate(p0["family"], p0["params"], p0["dim"], p0["transform"], ln[:1], lz[:1], p0["shifts"], **kw)   # warm-up
    reached, worst, evals = 0, 0.0, 0
    t0 = time.perf_counter()
    for p in probs:
        res, st = binding.qmc_integrate(p["family"], p["params"], p["dim"], p["transform"], ln, lz, p["shifts"], **kw)
        reached += int(st == 0)
        worst = max(worst, float(res["error"][0] / abs(res["integral"][0])))
        evals += res["evaluations"]
    dt = time.perf_counter() - t0
    return {"workload": workload_name(3), "target_rel_err": epsrel, "reached": reached == len(probs), "sectors_reached": reached,
            "sectors": len(probs), "seconds": dt, "evaluations": evals, "estimated_rel_err": worst, "true_rel_err": None,
            "n": int(ln[-1]), "m": p0["m"], "iterations": None, "ladder": [int(v) for v in ln]}


def time_to_target_batched(binding, probs, module, epsrel=1e-8):
    """configs[3] through qmc_integrate_batch: every sector follows the same iteration, the lattice evaluations of a round share one
    batched launch (with `module`: the specialised sector kernels).  The sectors share one set of shifts (sector 0's)."""
    ln, lz = synth.ladder(probs[0]["dim"], probs[0]["n"])
    kw = dict(min_n=1000, min_m=probs[0]["m"], epsrel=epsrel, epsabs=0.0, maxeval=2 ** 62)
    integrands = [dict(family=p["family"], dim=p["dim"], transform=p["transform"], params=p["params"]) for p in probs]
    shifts = probs[0]["shifts"]
    binding.qmc_integrate_batch(integrands, ln[:1], lz[:1], shifts, module=module, **kw)      # warm-up (module load)
    t0 = time.perf_counter()
    results, statuses, overall = binding.qmc_integrate_batch(integrands, ln, lz, shifts, module=module, **kw)
    dt = time.perf_counter() - t0
    reached = sum(int(s == 0) for s in statuses)
    return {"workload": workload_name(3) + (" [qmc_integrate_batch + specialised kernels]" if module is not None else " [qmc_integrate_batch]"),
            "target_rel_err": epsrel, "reached": reached == len(probs), "sectors_reached": reached, "sectors": len(probs), "seconds": dt,
            "evaluations": int(sum(r["evaluations"] for r in results)),
            "estimated_rel_err": max(float(r["error"][0] / abs(r["integral"][0])) for r in results), "true_rel_err": None,
            "n": int(max(r["n"] for r in results)), "m": int(max(r["m"] for r in results)),
            "iterations": int(max(r["iterations"] for r in results)), "ladder": [int(v) for v in ln],
            "module_build_s": None if module is None else module.info["build_ms"] * 1e-3}


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU fallback (use --impl reference for the oracle)")
    from paper_1811_11720_b200 import binding
    binding.lib()                                           # fails loudly if libqmc_lattice.so is missing

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(device))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    if args.genz_table:
        out = {"genz_protocol": {"korobov3": genz_table(binding, synth.TRANSFORM_KOROBOV + 3),
                                 "baker_d10": genz_table(binding, synth.TRANSFORM_BAKER, dims=(10,))},
               "note": "PAPER.md Table 1 / Table 2 protocol on one B200; averages over 10 seeded parameter sets"}
        if rank == 0:
            print(json.dumps(out))
        return

    binding.qmc_profile_enable(True)
    flush = L2Flusher(torch, device)
    sampler = ClockSampler(local)
    sampler.start()

    # FP64 issue-rate peak, measured in this process right before the timed runs (thread-level DFMA / s)
    binding.qmc_fp64_peak_probe(2000)
    peak_rate, peak_ms = binding.qmc_fp64_peak_probe(60000)
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count

    def measure(c, steps, warmup, specialised=False):
        """specialised (configs[3] only): the sectors as compiled straight-line code (qmc_sector_module_create, PAPER.md L427-L438:
        the paper compiles its integrands before integrating); the module is built once, outside the timed steps, and its
        build time is reported beside the line"""
        probs = rank_problems(c, rank)
        if c == 4:
            probs = config4_with_device_fit(binding, probs)
        alg = ALG_FP64_PER_EVAL[c] + (ALG_FP64_SECTOR_LOG_EXTRA if c == 3 and SECTOR_LOG else 0)
        key = "3s" if specialised else c
        executed = EXECUTED_FP64_PER_EVAL.get(key) if not (c == 3 and SECTOR_LOG) else None
        traffic = PROFILED_DRAM_BYTES_PER_LAUNCH.get(key) if SHRINK == 1 and not SECTOR_LOG else None
        label = bench_config(c)["workload"]
        if c == 3:
            label += " [specialised kernels: qmc_sector_module]" if specialised else " [interpreting kernel: the default entry]"
        module = binding.SectorModule(probs) if specialised else None
        rec, probs, w = measure_probs(label, probs, alg, executed, traffic, steps, warmup, module)
        if module is not None:
            info = module.info
            rec["sector_module"] = dict(info, note="built once per batch of integrands on the host (Horner compile -> PTX -> nvJitLink, "
                                        "kernels in parallel), outside the timed steps; reused for every lattice, shift set and sample count")
        return rec, probs, w

    def measure_probs(label, probs, alg, executed, traffic, steps, warmup, module=None):
        batch = binding.DeviceBatch(probs, device=device, module=module)
        barrier()
        w0 = time.perf_counter()
        step_ms, fused_ms, launches = time_steps(torch, binding, batch, steps, warmup, flush)
        barrier()
        w1 = time.perf_counter()
        total_s = max_over_ranks(sum(step_ms) * 1e-3)
        ev = evals_of(probs)
        fused_avg_s = statistics.fmean(fused_ms) * 1e-3
        achieved = alg * ev / fused_avg_s
        sms, means, errs = batch.results()
        rec = {"workload": label, "value": aggregate([ev * steps] * world, total_s), "unit": UNIT,
               "ms_per_step": total_s / steps * 1e3, "ms_per_step_best": min(step_ms), "steps": steps, "warmup": warmup,
               "evals_per_step_per_gpu": ev, "fused_kernel_ms": fused_avg_s * 1e3,
               "fused_kernel_share_of_step": fused_avg_s * 1e3 * steps / sum(step_ms),
               "gpu_launches_per_step": launches, "plan": batch.plan_info(),
               "roofline": {"bound": "alu", "achieved": achieved / 1e12, "peak": peak_rate / 1e12, "unit": "Tinst/s (thread-level FP64 instructions)",
                            "frac": achieved / peak_rate,
                            "frac_is": "USEFUL fraction: algorithmic FP64 instructions per evaluation x evaluations / fused-kernel time / peak",
                            "issue_frac": None if executed is None else executed * ev / fused_avg_s / peak_rate,
                            "issue_frac_is": "EXECUTED FP64-pipe instructions per evaluation (ncu, profiles/) x evaluations / fused-kernel time / peak",
                            "traffic": traffic,
                            "traffic_unit": "dram bytes per launch of the fused kernel at full size (ncu, profiles/r2_dram_full.md); the path is ALU bound, inputs are KBs",
                            "alg_fp64_inst_per_eval": alg, "executed_fp64_inst_per_eval": executed,
                            "peak_source": "qmc_fp64_peak_probe measured in this run (DFMA chains with one register multiplicand: FP64-pipe bound, not register-file bound)",
                            "peak_nominal": sm_count * FP64_LANES_PER_SM * 1.965e9 / 1e12},
               "result_mean": [float(v) for v in means[0]], "result_err": [float(v) for v in errs[0]]}
        return rec, probs, (w0, w1)

    windows = []
    main, main_probs, w = measure(args.main, args.steps, args.warmup, specialised=args.main == 3 and not args.interpret)
    windows.append(w)
    others = []
    interpreted3 = None
    if not args.main_only:
        for c, (k, wu) in {0: (50, 5), 1: (50, 5), 2: (10, 3), 3: (5, 3), 4: (3, 3)}.items():
            if c == args.main or (args.others is not None and c not in args.others):
                continue
            rec, _, w = measure(c, k, wu, specialised=c == 3 and not args.interpret)
            windows.append(w)
            others.append(rec)
            if c == 3 and not args.interpret:                # the same workload through the default entry, beside it
                interpreted3, _, w = measure(3, k, wu)
                windows.append(w)
    # variants beyond the BASELINE configs: the generic transforms and the pole-term fit on configs[2]'s / [4]'s shape, the
    # complex sector family on configs[3]'s shape.  alg counts: DESIGN.md section 5 ("variants").
    variants = []
    if rank == 0 and world == 1 and not args.main_only and (args.others is None or 9 in args.others):
        for label, probs, alg, k in variant_workloads():
            rec, _, w = measure_probs(label, probs, alg, None, None, k, 3)
            windows.append(w)
            variants.append(rec)
            if probs[0]["family"] == synth.FAMILY_SECTOR_COMPLEX and not args.interpret:       # the same batch as compiled code
                module = binding.SectorModule(probs)
                rec, _, w = measure_probs(label + " [specialised kernels: qmc_sector_module]", probs, alg, None, None, k, 3, module)
                rec["sector_module"] = module.info
                windows.append(w)
                variants.append(rec)

    # the roofline record of every config of the target (configs[1..4]) at top level
    roofline_all = {}
    for rec_c, rec in [(args.main, main)] + [(int(r["workload"].split("]")[0].split("[")[1]), r) for r in others]:
        if rec_c >= 1:
            roofline_all[f"configs[{rec_c}]"] = dict(rec["roofline"], fused_kernel_ms=rec["fused_kernel_ms"], ms_per_step=rec["ms_per_step"],
                                                     evals_per_s=rec["value"], workload=rec["workload"])
            if "sector_module" in rec:
                roofline_all[f"configs[{rec_c}]"]["sector_module"] = rec["sector_module"]
    if interpreted3 is not None:
        r = interpreted3
        roofline_all["configs[3] interpreted"] = dict(r["roofline"], fused_kernel_ms=r["fused_kernel_ms"], ms_per_step=r["ms_per_step"],
                                                      evals_per_s=r["value"], workload=r["workload"])

    # S10, the projection pass of configs[4] (n_fit lattice, one shift, 256 bins, all 16 dimensions): device time of the two kernels
    projection = None
    if rank == 0 and world == 1 and not args.main_only:
        p4 = rank_problems(4, 0)[0]
        proj = dict(p4, n=synth.CONFIG4_NFIT, z=synth.genvec(synth.CONFIG4_NFIT, p4["dim"]), transform=synth.TRANSFORM_NONE)
        pb = binding.DeviceBatch([proj], device=device)
        for _ in range(3):
            pb.project(0, synth.PROJECTION_BINS)
        tms = []
        for _ in range(10):
            flush()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            pb.project(0, synth.PROJECTION_BINS, sync=False)
            e1.record()
            e1.synchronize()
            tms.append(e0.elapsed_time(e1))
        pms = statistics.median(tms)
        projection = {"workload": f"projection pass of configs[4]: n_fit={synth.CONFIG4_NFIT}, d=16, 1 shift, {synth.PROJECTION_BINS} bins, transform none",
                      "ms": pms, "evals_per_s": synth.CONFIG4_NFIT / (pms * 1e-3), "histogram_updates_per_s": synth.CONFIG4_NFIT * 16 / (pms * 1e-3),
                      "note": "project_kernel + project_merge_kernel; shared-memory bound (warp-private histograms, lane-ordered merge), 0.2 % of a configs[4] step"}

    # the same step replayed from a CUDA graph (single-problem calls are capturable): launch overhead of small problems
    graphs = []
    if rank == 0 and world == 1 and not args.main_only:
        for c in (0, 1):
            if args.others is not None and c not in args.others and c != args.main:
                continue
            batch = binding.DeviceBatch(rank_problems(c, 0), device=device)
            g = batch.capture()
            for _ in range(5):
                g.replay()
            torch.cuda.synchronize()
            reps = 200
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                g.replay()
            e1.record()
            e1.synchronize()
            ms = e0.elapsed_time(e1) / reps
            graphs.append({"workload": workload_name(c), "ms_per_step_graph_replay": ms, "value": evals_of(batch.problems) / (ms * 1e-3),
                           "note": "back-to-back replays, no L2 flush in between (inputs are KBs)"})
        binding.qmc_profile_enable(True)

    ttt = []
    if rank == 0 and world == 1 and not args.main_only:
        for c in (0, 1, 2, 3, 4):
            if args.others is not None and c not in args.others and c != args.main:
                continue
            probs = rank_problems(c, 0)
            if c == 4:
                probs = config4_with_device_fit(binding, probs)
            ttt.append(time_to_target_batch(binding, probs) if c == 3 else time_to_target(binding, c, probs))
            if c == 3:                                      # the same 256 sectors iterated together, default and specialised kernels
                ttt.append(time_to_target_batched(binding, probs, None))
                if not args.interpret:
                    ttt.append(time_to_target_batched(binding, probs, binding.SectorModule(probs)))

    # end-to-end through the HOST-pointer entry (rank-local; max over ranks)
    barrier()
    e2e_reps = max(3, min(args.steps, 50 if main["ms_per_step"] < 10 else 5))
    main_module = binding.SectorModule(main_probs) if "sector_module" in main else None   # configs[3]: the route of the headline line
    e2e_s, h2d, d2h = e2e_host_api(binding, main_probs, e2e_reps, main_module)
    e2e_s = max_over_ranks(e2e_s)
    sampler.stop()
    clocks = sampler.summary(windows)

    out = {"metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": bench_config(args.main),
           "run": {"l2": "256 MiB buffer written between timed iterations (inputs are KB-sized and stay resident)",
                   "parallelism": f"replicas x{world} (independent problems per rank, no data-path collective)",
                   "plan": main["plan"], "timed_region_s": main["ms_per_step"] * args.steps * 1e-3},
           "e2e": {"value": aggregate([main["evals_per_step_per_gpu"]] * world, e2e_s), "unit": UNIT, "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3, "reps": e2e_reps,
                   "api": ("qmc_lattice_integrate_batch_host_module" if main_module is not None else "qmc_lattice_integrate_batch_host") + " (HOST pointers; validation + H2D from pinned staging + kernels + D2H + sync inside the timed call)"},
           "gpu_launches": main["gpu_launches_per_step"] * args.steps,
           "roofline": main["roofline"], "roofline_all": roofline_all, "projection_pass": projection,
           "fused_kernel_ms": main["fused_kernel_ms"],
           "fused_kernel_share_of_step": main["fused_kernel_share_of_step"],
           "fp64_peak_probe": {"thread_inst_per_s": peak_rate, "ms": peak_ms, "sm_count": sm_count,
                               "implied_clock_mhz_at_64_lanes": peak_rate / (sm_count * FP64_LANES_PER_SM) / 1e6},
           "clocks": clocks, "others": others, "variants": variants, "time_to_rel_err_1e-8": ttt, "cuda_graph": graphs}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.main)
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------------------------------
# CPU oracle arm (reported baseline; never tuned)
# ----------------------------------------------------------------------------------------------------
def oracle_problems(c):
    """the headline workload for the oracle legs; configs[4] takes the fit map the ORACLE derives from its own projection pass"""
    probs = shrunk_config(c)
    if c == 4:
        import oracle
        p = probs[0]
        proj = dict(p, n=synth.CONFIG4_NFIT, z=synth.genvec(synth.CONFIG4_NFIT, p["dim"]), transform=synth.TRANSFORM_NONE)
        probs = [dict(p, fit_coeffs=oracle.fit_cubic(oracle.project(proj, synth.PROJECTION_BINS)))]
    return probs


ORACLE_MIN_INDICES = 128 * 65536     # the oracle parallelises over 2^16-index chunks: a sample keeps every host core busy


def oracle_sample(probs, div):
    """The bounded sample of a workload, about 1/div of its evaluations: for a batch of at least div problems every div-th
    problem on its whole lattice; otherwise lattice indices [0, k_end) of every problem, all shifts, with
    k_end = min(n, max(ceil(n / div), 128 * 2^16)).  -> list of (problem, k_end)"""
    if len(probs) >= div:
        return [(p, p["n"]) for p in probs[::div]]
    return [(p, min(p["n"], max(-(-p["n"] // div), ORACLE_MIN_INDICES))) for p in probs]


def oracle_sample_pass(probs, div):
    """the oracle as it stands on the bounded sample -> evaluations done"""
    import oracle
    done = 0
    for p, k_end in oracle_sample(probs, div):
        oracle.shift_sums(p, 0, k_end)
        done += k_end * p["m"]
    return float(done)


def sample_text(c, div, done):
    probs = shrunk_config(c)
    smp = oracle_sample(probs, div)
    what = (f"every {div}-th problem ({len(smp)} of {len(probs)}) on its whole lattice" if len(probs) >= div
            else f"lattice indices [0, {smp[0][1]}) of n = {probs[0]['n']}")
    return (f"{what}, all shifts, of {workload_name(c)}: {done:.3g} of {evals_of(probs):.3g} evaluations per pass; "
            "throughput = evaluations done / wall time; OpenMP over 2^16-index chunks")


def cpu_baseline(c, budget_s=12.0):
    """The oracle timed on the host cores on a bounded sample of the SAME workload (about 10-30 s), plus the per-core figure of
    SURVEY 8(d): the same code with OMP_NUM_THREADS=1 on a 1/4096 sub-range, in a child process (the OpenMP runtime reads the
    variable once)."""
    import oracle
    import subprocess
    probs = oracle_problems(c)
    passes, done, t0 = 0, 0.0, time.perf_counter()
    while True:
        done += oracle_sample_pass(probs, ORACLE_SAMPLE_DIV)
        passes += 1
        dt = time.perf_counter() - t0
        if dt >= budget_s or passes >= 3:
            break
    rec = {"value": done / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
           "sample": sample_text(c, ORACLE_SAMPLE_DIV, done / passes) + f"; {passes} pass(es), {dt:.1f} s", "seconds": dt}
    try:
        env = dict(os.environ, OMP_NUM_THREADS="1")
        out = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-per-core", str(c)] +
                             (["--sector-log"] if SECTOR_LOG else []) + (["--shrink", str(SHRINK)] if SHRINK > 1 else []),
                             env=env, capture_output=True, text=True, timeout=600, check=True).stdout.strip().splitlines()[-1]
        rec["per_core"] = json.loads(out)
    except Exception as e:                                   # the per-core figure is an extra; never fail the bench line for it
        rec["per_core"] = {"unavailable": repr(e)[:200]}
    return rec


def run_oracle_per_core(c):
    import oracle
    probs = oracle_problems(c)
    p = probs[0]                                             # one problem, 4 chunks of 2^16 indices
    k_end = min(p["n"], 4 * 65536)
    t0 = time.perf_counter()
    oracle.shift_sums(p, 0, k_end)
    dt = time.perf_counter() - t0
    done = float(k_end * p["m"])
    print(json.dumps({"value": done / dt, "unit": UNIT, "cores": oracle.num_threads(), "seconds": dt,
                      "sample": f"lattice indices [0, {k_end}) of the first problem of {workload_name(c)}, all shifts ({done:.3g} evaluations); OMP_NUM_THREADS=1"}))


def bench_config(c):
    """the `config` object both arms print: it names the workload and nothing that differs between the arms"""
    return {"workload": workload_name(c) + (" + log factors (lu log U + lf log F)^p [variant, not a BASELINE config]" if c == 3 and SECTOR_LOG else "")
            + (f" [SHRUNK x1/{SHRINK} for profiling: not a bench value]" if SHRINK > 1 else ""),
            "evals_per_step_per_gpu": evals_of(shrunk_config(c))}


def run_reference(args):
    """The reference arm of this tier = the CPU oracle as it stands, on this arm's workload, metric and unit.  A step is one
    bounded sample of the workload (sample_text); the number of steps is cut so that the run ends within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    c = args.main
    probs = oracle_problems(c)
    for _ in range(min(args.warmup, 1)):
        oracle.shift_sums(probs[0], 0, min(probs[0]["n"], 8 * 65536))
    times, done, steps = [], 0.0, args.steps
    i = 0
    while i < steps:
        t0 = time.perf_counter()
        done += oracle_sample_pass(probs, ORACLE_SAMPLE_DIV)
        times.append(time.perf_counter() - t0)
        i += 1
        if i == 1:
            steps = max(1, min(steps, int(150.0 / max(times[0], 1e-3))))     # bounded: the whole run stays within minutes
    total = sum(times)
    value = done / total
    sample = sample_text(c, ORACLE_SAMPLE_DIV, done / len(times)) + f"; {len(times)} step(s) of one pass each"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": len(times), "warmup": min(args.warmup, 1), "ms_per_step": total / len(times) * 1e3,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": bench_config(c),
                      "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
                      "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start N ranks of this script on this node (127.0.0.1) and pass the line on"""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--main-only", action="store_true", help="time the headline config only (skip 'others', time-to-target, graphs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--interpret", action="store_true",
                    help="configs[3]: time the interpreting kernel only (no module of specialised sector kernels is built)")
    ap.add_argument("--genz-table", action="store_true",
                    help="run the Genz protocol of the paper's Table 1 / Table 2 through qmc_integrate instead of the throughput bench")
    ap.add_argument("--sector-log", action="store_true",
                    help="configs[3] with the log factors of an eps-expansion term on every sector (use with --main 3 --main-only)")
    ap.add_argument("--shrink", type=int, default=1,
                    help="profiling only: run 1/S of every config's work (fewer sectors / a smaller prime n)")
    ap.add_argument("--main", type=int, default=MAIN_CONFIG, choices=[0, 1, 2, 3, 4],
                    help="config reported as the headline line (default configs[4], the largest single-GPU configuration)")
    ap.add_argument("--others", type=lambda v: [int(x) for x in v.split(",") if x != ""], default=None,
                    help="comma-separated subset of the configs to time besides the headline (default: all)")
    ap.add_argument("--oracle-per-core", type=int, default=None, help=argparse.SUPPRESS)   # child process of cpu_baseline
    args = ap.parse_args()
    global SHRINK, SECTOR_LOG
    SHRINK = max(1, args.shrink)
    SECTOR_LOG = bool(args.sector_log)
    if args.oracle_per_core is not None:
        run_oracle_per_core(args.oracle_per_core)
        return
    world = int(os.environ.get("WORLD_SIZE", "0"))
    if world == 0 and args.gpus > 1:
        spawn_ranks(args)                                    # does not return
    if world > 0 and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if args.impl == "reference":
        run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3
        run_ours(args)


if __name__ == "__main__":
    main()
