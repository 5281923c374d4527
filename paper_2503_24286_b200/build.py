"""Builds libpyro.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2503_24286_b200.build [--force] [-DNAME=VALUE ...]

Every source is compiled to an object file of its own (in parallel), then linked.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libpyro.so")
SOURCES = ["pyro_kernels.cu", "pyro_fused_kernels.cu", "pyro_rates2_kernels.cu", "pyro_jac_kernels.cu", "pyro_jac_block_kernels.cu", "pyro_reactor_kernels.cu", "pyro_transport.cu", "pyro_probes.cu", "pyro_cn_kernels.cu", "pyro_api.cpp", "pyro_pack.cpp",
           "pyro_jac_pack.cpp"]
HEADERS = ["pyro_kernels.h", "pyro_pack.h", "pyro_tables.h", "pyro_math.cuh", "pyro_point.cuh", "pyro_rates_kernel.cuh",
           "pyro_jac.cuh", "pyro_jac_dev.cuh", "pyro_jac_tables.h", os.path.join("..", "..", "include", "pyro.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "-Xptxas", "-v"]


STAMP = os.path.join(OBJ, "defines.txt")   # the -D options the objects and the library on disk were built with


def _built_defines():
    try:
        return open(STAMP).read()
    except OSError:
        return None


def _stale(defines=()):
    if not os.path.exists(LIB) or _built_defines() != " ".join(defines):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build_libpyro(force=False, defines=(), verbose=False):
    if not (force or _stale(defines)):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    same_defines = _built_defines() == " ".join(defines)   # objects compiled with other -D options are never reused
    newest_header = max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)

    def compile_one(src):
        obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
        path = os.path.join(CSRC, src)
        if (not force and same_defines and os.path.exists(obj)
                and os.path.getmtime(obj) > max(os.path.getmtime(path), newest_header)):
            return obj, None, ""
        cmd = [nvcc, *NVCC_FLAGS, *defines, "-c", "-o", obj, path]
        res = subprocess.run(cmd, capture_output=True, text=True)
        return obj, res, " ".join(cmd) + "\n" + res.stdout + res.stderr

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as pool:
        results = list(pool.map(compile_one, SOURCES))
    log = "".join(r[2] for r in results)
    failed = [r for r in results if r[1] is not None and r[1].returncode != 0]
    link = None
    if not failed:
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-o", LIB, *[r[0] for r in results]]
        link = subprocess.run(cmd, capture_output=True, text=True)
        log += " ".join(cmd) + "\n" + link.stdout + link.stderr
    if verbose or failed or (link and link.returncode != 0):
        sys.stderr.write(log)
    if failed or link.returncode != 0:
        raise RuntimeError("nvcc failed building libpyro.so")
    with open(os.path.join(_HERE, "libpyro.build.log"), "w") as f:
        f.write(log)
    with open(STAMP, "w") as f:
        f.write(" ".join(defines))
    return LIB


if __name__ == "__main__":
    args = sys.argv[1:]
    build_libpyro(force="--force" in args, defines=[a for a in args if a.startswith("-D")], verbose=True)
    print(LIB)
