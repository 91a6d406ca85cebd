"""Builds libqmc_lattice.so (the C-ABI library of include/qmc_lattice.h) in-tree with nvcc for sm_100a.

python -m paper_1811_11720_b200.build [--force]
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libqmc_lattice.so")
# (source, extra nvcc defines, object name): the closed-form fused kernels are one source compiled per (family, part)
SOURCES = [("qmc_host.cu", [], "qmc_host.o"), ("qmc_adaptive.cu", [], "qmc_adaptive.o"), ("qmc_fit.cu", [], "qmc_fit.o"),
           ("qmc_misc.cu", [], "qmc_misc.o"), ("qmc_project.cu", [], "qmc_project.o"), ("qmc_fused_f3.cu", [], "qmc_fused_f3.o"),
           ("qmc_fused_f8.cu", [], "qmc_fused_f8.o")]
SOURCES += [("qmc_fused_closed.cu", [f"-DQMC_FAM={f}", f"-DQMC_PART={q}"], f"qmc_fused_closed_f{f}_p{q}.o")
            for q in (3, 2, 1, 0) for f in (2, 4, 1, 0)]       # the slowest parts first
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]


def _deps(path, seen=None):
    """the files `path` includes with #include "...", recursively (paths relative to the including file)"""
    seen = set() if seen is None else seen
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line.startswith("#include \""):
                inc = os.path.normpath(os.path.join(os.path.dirname(path), line.split('"')[1]))
                if inc not in seen and os.path.exists(inc):
                    seen.add(inc)
                    _deps(inc, seen)
    return seen


def _compile(job, force: bool) -> str:
    src, defines, objname = job
    obj = os.path.join(OBJ, objname)
    path = os.path.join(CSRC, src)
    newest = max(os.path.getmtime(p) for p in [path, *_deps(path)])
    if force or not os.path.exists(obj) or os.path.getmtime(obj) < newest:
        subprocess.run(["nvcc", *NVCC_FLAGS, *defines, "-c", path, "-o", obj], check=True)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    jobs = [j for j in SOURCES if os.path.exists(os.path.join(CSRC, j[0]))]
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(os.cpu_count() or 4, len(jobs))) as ex:
        objs = list(ex.map(lambda j: _compile(j, force), jobs))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.run(["nvcc", "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"],
                       check=True)
        if verbose:
            print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
