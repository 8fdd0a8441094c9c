"""The C-ABI boundary without a GPU: libtatrg.so builds in-tree, loads, and exports every function
include/tatrg.h declares; the Python binding lists exactly those; compute calls fail loudly (no CPU
fallback) when there is no CUDA device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "tatrg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)            # comments
    text = re.sub(r"^\s*#.*$", "", text, flags=re.M)              # preprocessor lines
    names = re.findall(r"\b([A-Za-z_][A-Za-z0-9_]*)\s*\([^;{}]*\)\s*;", text)
    return sorted(set(names))


def test_header_declares_the_three_calls_of_the_path():
    names = declared_functions()
    for n in ("init_ising_tensor", "coarse_grain", "log_Z_per_site", "coarse_grain_atrg"):
        assert n in names
    assert len(names) >= 30


def test_library_exports_every_declared_symbol():
    from paper_2412_14104_b200 import build as b
    so = b.build()
    L = ctypes.CDLL(so)
    missing = [n for n in declared_functions() if not hasattr(L, n)]
    assert not missing, missing


def test_binding_lists_exactly_the_declared_symbols():
    import paper_2412_14104_b200 as t
    assert sorted(t.EXPORTS) == declared_functions()
    L = t.lib()
    for n in t.EXPORTS:
        getattr(L, n)


def test_no_cpu_fallback():
    import torch
    import paper_2412_14104_b200 as t
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(t.TatrgError):
        t.init_ising_tensor(0.2, 0.0)
    with pytest.raises(t.TatrgError):
        t.set_workspace(nbytes=1 << 20)
    # the library itself refuses to work without a workspace / device
    assert t.lib().init_ising_tensor(ctypes.c_double(0.2), ctypes.c_double(0.0)) != 0
    assert t.lib().tatrg_last_error()
