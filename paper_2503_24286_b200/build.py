"""Builds libpyro.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2503_24286_b200.build [--force] [-DNAME=VALUE ...]
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpyro.so")
SOURCES = ["pyro_kernels.cu", "pyro_jac_kernels.cu", "pyro_api.cpp", "pyro_pack.cpp", "pyro_jac_pack.cpp"]
HEADERS = ["pyro_kernels.h", "pyro_pack.h", "pyro_tables.h", "pyro_math.cuh", "pyro_point.cuh", "pyro_jac.cuh",
           "pyro_jac_tables.h",
           os.path.join("..", "..", "include", "pyro.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build_libpyro(force=False, defines=(), verbose=False):
    if not (force or _stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, *NVCC_FLAGS, *defines, "-o", LIB, *[os.path.join(CSRC, s) for s in SOURCES]]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libpyro.so")
    with open(os.path.join(_HERE, "libpyro.build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    args = sys.argv[1:]
    build_libpyro(force="--force" in args, defines=[a for a in args if a.startswith("-D")], verbose=True)
    print(LIB)
