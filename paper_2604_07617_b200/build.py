"""Builds the two shared libraries in-tree with nvcc for sm_100a (nvcc cross-compiles without a GPU):

  paper_2604_07617_b200/libcatapult.so        the product: the C-ABI of include/catapult.h
  paper_2604_07617_b200/libcatapult_probe.so  measurement / test hooks of include/catapult_probe.h
                                              (DFMA and L2 peak micro-benchmarks, device math probe)
"""
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
PROBE_LIB = os.path.join(PKG, "libcatapult_probe.so")
OBJ = os.path.join(PKG, "build")
SOURCES = ["api.cu", "field.cu", "tracer.cu", "tracer_pair.cu", "estimate.cu", "measure.cu"]
PROBE_SOURCES = ["probe_api.cu", "peaks.cu", "mathprobe.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", *ARCH, "-lineinfo", "-Xcompiler", "-fPIC", "-I", INC, "-I", CSRC]


def _deps():
    out = [os.path.join(INC, fn) for fn in os.listdir(INC)]
    for fn in os.listdir(CSRC):
        out.append(os.path.join(CSRC, fn))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in _deps())
    if (not force and all(os.path.exists(l) and os.path.getmtime(l) >= newest for l in (LIB, PROBE_LIB))):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

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

    with ThreadPoolExecutor(max_workers=len(SOURCES) + len(PROBE_SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES + PROBE_SOURCES))
    n = len(SOURCES)
    subprocess.run([NVCC, "-shared", *ARCH, "-o", LIB, *objs[:n]], check=True)
    subprocess.run([NVCC, "-shared", *ARCH, "-o", PROBE_LIB, *objs[n:]], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
