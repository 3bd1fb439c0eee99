"""Build libs2b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1510_04068_b200.build [--force]

Each .cu is compiled to an object in csrc/build/ (parallel, incremental by mtime) and the
objects are linked into paper_1510_04068_b200/libs2b200.so with a static CUDA runtime, so the
library loads on a box without a GPU (symbol checks) and next to PyTorch's own runtime.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(PKG, "libs2b200.so")
HEADER = os.path.join(os.path.dirname(PKG), "include", "s2b200.h")
TEST_HEADER = os.path.join(os.path.dirname(PKG), "include", "s2b200_test.h")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-diag-suppress", "177"]


def _sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _deps_mtime():
    hdrs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))] + [HEADER, TEST_HEADER]
    return max(os.path.getmtime(h) for h in hdrs)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    hdr_m = _deps_mtime()
    jobs, objs = [], []
    for src in _sources():
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src[:-3] + ".o")
        objs.append(o)
        src_m = os.path.getmtime(s)
        for line in open(s):   # a .cu that includes another .cu (second instance of a module) depends on it
            if line.startswith('#include "') and line.rstrip().endswith('.cu"'):
                src_m = max(src_m, os.path.getmtime(os.path.join(CSRC, line.split('"')[1])))
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(src_m, hdr_m):
            jobs.append([NVCC, *FLAGS, "-c", s, "-o", o])

    def run(cmd):
        if verbose:
            print(" ".join(cmd), flush=True)
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
        return r

    if jobs:
        with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            list(ex.map(run, jobs))
    if jobs or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        run([NVCC, "-shared", "-o", LIB + ".tmp", *objs, "-cudart", "static",
             "-gencode", "arch=compute_100a,code=sm_100a"])
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
