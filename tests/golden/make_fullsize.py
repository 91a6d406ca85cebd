"""Writes tests/golden/fullsize_oracle.json: the CPU oracle's results at BASELINE.json's FULL sizes.

Calls only oracle/ and the seeded input generators (paper_1811_11720_b200.synth holds no arithmetic
of the method).  No value comes from the CUDA path.  Doubles are stored as C99 hex strings.

    python tests/golden/make_fullsize.py [2] [3] [4]        (hours of CPU time in total on 8 cores)

configs[2]: all 32 per-shift means (re, im), estimate and error (Eq. 2-3).
configs[3]: all 256 sectors (SECTOR_SAMPLE), one record each.
configs[4]: projection histogram (n_fit lattice, first shift; Eq. 20, reading C-8),
            the oracle's cubic fit of it, and the 20 per-shift means with that fit map applied.
"""
import hashlib
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1811_11720_b200 import synth  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "fullsize_oracle.json")
SECTOR_SAMPLE = list(range(256))        # every sector of configs[3] (about 25 minutes of oracle time on 8 cores)


def hexlist(a):
    return [float(v).hex() for v in np.asarray(a, dtype=np.float64).ravel()]


def record(p):
    t = time.time()
    sm, mean, err = oracle.integrate(p)
    return {"name": p["name"], "n": p["n"], "dim": p["dim"], "m": p["m"], "shift_means": hexlist(sm), "mean": hexlist(mean),
            "err": hexlist(err), "oracle_seconds": round(time.time() - t, 1), "oracle_threads": oracle.num_threads()}


def config4_problem():
    """configs[4] with the fit map the ORACLE derives from its own projection pass."""
    p = synth.config(4)[0]
    proj = dict(p, n=synth.CONFIG4_NFIT, z=synth.genvec(synth.CONFIG4_NFIT, p["dim"]), transform=synth.TRANSFORM_NONE)
    H = oracle.project(proj, synth.PROJECTION_BINS)
    fit = oracle.fit_cubic(H)
    return dict(p, fit_coeffs=fit), H, fit


def provenance():
    """Which oracle wrote the file: sha256 of oracle/qmc_oracle.cpp and the commit it was run from (informative; the
    binding check is tests/test_oracle_pins.py::test_fullsize_goldens_are_what_the_live_oracle_computes)."""
    with open(os.path.join(ROOT, "oracle", "qmc_oracle.cpp"), "rb") as f:
        sha = hashlib.sha256(f.read()).hexdigest()
    try:
        head = subprocess.run(["git", "-C", ROOT, "rev-parse", "HEAD"], capture_output=True, text=True, check=True).stdout.strip()
        dirty = bool(subprocess.run(["git", "-C", ROOT, "status", "--porcelain", "--", "oracle"], capture_output=True,
                                    text=True, check=True).stdout.strip())
    except Exception:
        head, dirty = "unknown", False
    return {"oracle_sha256": sha, "git_head": head, "oracle_dirty": dirty}


def main(argv):
    which = [int(a) for a in argv] or [2, 3, 4]
    table = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            table = json.load(f)
    prov = table.setdefault("provenance", {})
    for c in which:
        print(f"config {c} ...", flush=True)
        if c == 3:
            probs = synth.config(3)
            table["3"] = {"sectors": {str(i): record(probs[i]) for i in SECTOR_SAMPLE}}
        elif c == 4:
            p, H, fit = config4_problem()
            rec = record(p)
            rec["projection_hist"] = hexlist(H)
            rec["fit_coeffs"] = hexlist(fit)
            table["4"] = rec
        else:
            table[str(c)] = record(synth.config(c)[0])
        prov[str(c)] = provenance()
        with open(OUT, "w") as f:
            json.dump(table, f, indent=0, sort_keys=True)
        print(f"config {c} done", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
