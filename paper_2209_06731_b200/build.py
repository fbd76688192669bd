"""Builds the C-ABI shared library (csrc/ -> libgx.so, in-tree) with nvcc for sm_100a.

``python -m paper_2209_06731_b200.build`` or ``build()``; nvcc cross-compiles without a GPU.  One translation unit
per kernel family, compiled in parallel, linked into one shared object.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgx.so")
OBJ = os.path.join(HERE, "build")
SOURCES = ["gx_api.cu", "sets_scalar.cu", "sets_scalar2.cu", "sets_row.cu", "sets_rx.cu", "ubench.cu"]
HEADERS = ["dft_regs.cuh", "dft_packed.cuh", "kernel_sets.h", "nl_rx_kernels.cuh", "nl_kernels.cuh", "nl_row_kernels.cuh",
           "linear_kernels.cuh"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--extended-lambda", "-Xcompiler", "-fPIC"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "gx.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=(), lib: str = LIB) -> str:
    if not force and lib == LIB and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    objdir = OBJ if lib == LIB else lib + ".build"
    os.makedirs(objdir, exist_ok=True)
    extra = (["-Xptxas", "-v"] if verbose else []) + ["-D" + d for d in defines]

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + extra + ["-c", "-o", obj, os.path.join(CSRC, src)]
        res = subprocess.run(cmd, capture_output=True, text=True)
        return src, obj, res

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    for src, obj, res in results:
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed on " + src)
        if verbose:
            sys.stderr.write(res.stderr)
    cmd = [nvcc, "-shared", "-o", lib] + [obj for _, obj, _ in results]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("link failed: " + " ".join(cmd))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
