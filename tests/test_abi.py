"""CPU-only checks of the boundary: the C-ABI library builds/loads and exports every symbol that
include/flatspin.h declares; without a device compute entry points fail loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    txt = open(os.path.join(ROOT, "include", "flatspin.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(fs_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    from paper_2002_11401_b200 import build
    from paper_2002_11401_b200.binding import EXPORTS
    lib = build.build()
    L = ctypes.CDLL(lib)
    syms = header_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(EXPORTS) == syms          # the binding mirrors the header one to one


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2002_11401_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f
                assert "flatspin_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "flatspin_oracle.cpp")).read()
    assert "flatspin.h" not in osrc.replace("include/flatspin.h", "") and "cuda" not in osrc.lower().replace("cuda path", "")


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    from paper_2002_11401_b200 import workloads as W
    from paper_2002_11401_b200.binding import Sim
    w = W.config("1")
    with pytest.raises(RuntimeError):
        Sim(w.pos, w.angle, w.hc, w.params)


def test_argument_errors_are_reported_not_thrown():
    from paper_2002_11401_b200.binding import load_library, FsParams, FS_ERR_ARG
    L = load_library()
    p = FsParams(0.001, 1, 1, 3, 3, 1.0)
    n = ctypes.c_size_t()
    assert L.fs_workspace_bytes(0, 1, None, ctypes.byref(p), ctypes.byref(n), None) == FS_ERR_ARG
    assert b"N=" in L.fs_last_error()
    bad = FsParams(0.001, 1, 1, -3, 3, 1.0)
    assert L.fs_workspace_bytes(10, 1, None, ctypes.byref(bad), ctypes.byref(n), None) == FS_ERR_ARG
    assert L.fs_relax(None, 0, None) == FS_ERR_ARG
    assert L.fs_destroy(None) == 0
