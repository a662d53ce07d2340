"""Builds libpf.so (the C-ABI library of include/pf.h) in-tree with nvcc for sm_100a.

    python -m paper_2306_04322_b200.build [--force]
    PF_EXTRA_NVCC_FLAGS="-DPF_DBG_SKIP_COMPUTE" PF_BUILD_SUFFIX=nocomp python -m paper_2306_04322_b200.build
        -> libpf_nocomp.so beside libpf.so (an ablation / experiment build; load it with PF_LIBPF=<path>, see pf.py)
    PF_EXTRA_NVCC_FLAGS="-DPF_WCOL" PF_BUILD_SUFFIX=wcol ...   adds wcol_kernels.cu (persistent pipelined strided kernel, selected at
        run time with PF_WCOL=1); PF_EXTRA_NVCC_FLAGS="-DPF_WFFT" the warp-tile FFT. Neither is part of the default library.

The translation units are compiled in parallel and linked into
paper_2306_04322_b200/libpf.so (static cudart; no torch, no other dependency).
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SUFFIX = os.environ.get("PF_BUILD_SUFFIX", "")
OBJ = os.path.join(HERE, "csrc", "build" + ("_" + SUFFIX if SUFFIX else ""))
SO = os.path.join(HERE, "libpf" + ("_" + SUFFIX if SUFFIX else "") + ".so")
UNITS = ["row_kernels", "col_kernels", "col2d_kernels", "fd_kernels", "fd2d_kernels", "fd3d_kernels", "sgrid_kernels", "static_energy", "dsmem_probe", "pf"]
HEADERS = sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(os.path.dirname(HERE), "include", "pf.h")]
if "-DPF_WCOL" in os.environ.get("PF_EXTRA_NVCC_FLAGS", "").split():       # opt-in variant (profiles/r2_col_variants.md)
    UNITS.insert(3, "wcol_kernels")
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("PF_EXTRA_NVCC_FLAGS", "").split()


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(unit: str, force: bool) -> str:
    src = os.path.join(CSRC, unit + ".cu")
    obj = os.path.join(OBJ, unit + ".o")
    if force or _stale(obj, [src] + HEADERS):
        log = os.path.join(OBJ, unit + ".ptxas.log")
        with open(log, "w") as fh:
            r = subprocess.run([_nvcc()] + NVCC_FLAGS + ["-c", src, "-o", obj], stdout=fh, stderr=subprocess.STDOUT)
        if r.returncode != 0:
            sys.stderr.write(open(log).read()[-4000:])
            raise RuntimeError(f"nvcc failed on {unit}.cu (log: {log})")
    return obj


def build(force: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        objs = list(ex.map(lambda u: _compile(u, force), UNITS))
    if force or _stale(SO, objs):
        subprocess.run([_nvcc(), "-shared", "-o", SO] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"], check=True)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
