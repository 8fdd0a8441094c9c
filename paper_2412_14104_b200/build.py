"""Builds libtatrg.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libtatrg.so")
CU = ["gemm.cu", "gemm_big.cu", "gemm_p.cu", "gemm_tma.cu", "ts.cu", "rng.cu", "reduce.cu", "qr.cu", "jacobi.cu", "jacobi_small.cu", "gauge.cu", "chol.cu", "sq_iter.cu", "cholqr_fused.cu"]
CPP = ["tensor.cpp", "step.cpp", "api.cpp"]
GAUSS = os.path.join(ROOT, "seeded_inputs", "gauss.c")   # the shared seeded INPUT generator
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _newer(target, sources):
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(s) <= t for s in sources)


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, f) for f in CU + CPP]
    deps = srcs + [GAUSS, os.path.join(ROOT, "include", "tatrg.h")] + \
        [os.path.join(CSRC, h) for h in ("common.h", "tensor.h", "ctx.h", "chol64.cuh", "sq_iter.h")]
    if not force and _newer(SO, deps):
        return SO
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s) + ".o")
        objs.append(o)
        cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-x", "cu", "-c", s, "-o", o]
        procs.append((cmd, subprocess.Popen(cmd)))
    og = os.path.join(objdir, "gauss.o")
    cmd = ["gcc", "-O2", "-fPIC", "-fopenmp", "-ffp-contract=off", "-c", GAUSS, "-o", og]
    procs.append((cmd, subprocess.Popen(cmd)))
    objs.append(og)
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("build failed: " + " ".join(cmd))
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", SO] + objs + ["-Xcompiler", "-fopenmp", "-lgomp", "-lcudart"]
    subprocess.run(cmd, check=True)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
