"""Builds paper_2604_07617_b200/libcatapult.so (the C-ABI library of include/catapult.h) in-tree
with nvcc for sm_100a.  nvcc cross-compiles without a GPU."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
INC = os.path.join(ROOT, "include")
LIB = os.path.join(PKG, "libcatapult.so")
OBJ = os.path.join(PKG, "build")
SOURCES = ["api.cu", "field.cu", "tracer.cu", "estimate.cu", "peaks.cu", "mathprobe.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-I", INC, "-I", CSRC]


def _deps():
    out = [os.path.join(INC, "catapult.h")]
    for fn in os.listdir(CSRC):
        out.append(os.path.join(CSRC, fn))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in _deps())
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    extra += os.environ.get("CATAPULT_NVCC_FLAGS", "").split()     # e.g. -DCATAPULT_SPLIT_NREG_BOOZER=24 for sweeps

    def compile_one(src):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        if (not force and os.path.exists(obj) and os.path.getmtime(obj) >= newest):
            return obj
        cmd = [NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}")
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
