"""Seeded synthetic INPUT generators shared by the oracle tests and the CUDA path.

Holds none of the method's arithmetic: only the counter-based Gaussian stream
that feeds the RSVD sketches and the gauge
reference matrices (reading G12).  Implemented in C (gauss.c) and
loaded with ctypes; built on demand with gcc if the shared object is missing.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libseeded_inputs.so")
_SRC = os.path.join(_HERE, "gauss.c")

# `which` codes of the sub-seed recipe.
WHICH_SWAP, WHICH_A, WHICH_X, WHICH_Y, WHICH_D = 0, 1, 2, 3, 4
WHICH_REF_AD = 5          # gauge reference for the canonical A/D columns
WHICH_REF_SQ = (6, 7, 8)  # gauge references for the three squeezers (t1, t2, t3)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.si_splitmix64.restype = ctypes.c_uint64
        lib.si_splitmix64.argtypes = [ctypes.c_uint64]
        lib.si_subseed.restype = ctypes.c_uint64
        lib.si_subseed.argtypes = [ctypes.c_uint64] * 3
        lib.si_fill_gauss.restype = None
        lib.si_fill_gauss.argtypes = [ctypes.c_void_p, ctypes.c_uint64,
                                      ctypes.c_uint64, ctypes.c_uint64]
        _lib = lib
    return _lib


def subseed(seed: int, step: int, which: int) -> int:
    return int(_load().si_subseed(seed & (2**64 - 1), step, which))


def gauss(sub: int, n: int, offset: int = 0, out: np.ndarray | None = None) -> np.ndarray:
    """n consecutive N(0,1) doubles of stream `sub`, starting at element `offset`."""
    if out is None:
        out = np.empty(n, dtype=np.float64)
    assert out.dtype == np.float64 and out.flags.c_contiguous and out.size >= n
    _load().si_fill_gauss(out.ctypes.data, n, sub, offset)
    return out


def gauss_matrix(seed: int, step: int, which: int, rows: int, cols: int) -> np.ndarray:
    """Row-major rows x cols Gaussian matrix of sub-stream (seed, step, which)."""
    return gauss(subseed(seed, step, which), rows * cols).reshape(rows, cols)
