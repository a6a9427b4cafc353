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


def test_stencil_kernels_keep_their_weights_in_uniform_registers():
    """Compile-time property of the built library: every constant-table variant of k_gather_stencil must
    read its couplings through the uniform datapath (LDCU -> `DFMA R, R, UR, R`, 62 against 51 DFMA/clk/SM); ptxas
    drops that silently when the kernel's control flow changes shape (a loop inside a divergent branch in front of the
    main loop is enough).  The inversion-paired fp64 variants stage their tiles by TMA (UTMALDG)."""
    import shutil
    import subprocess
    from paper_2002_11401_b200 import build
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", build.build()], capture_output=True, text=True, check=True).stdout
    parts = re.split(r"\n\s*Function : ", sass)
    seen = 0
    for p in parts:
        name = p.split("\n")[0]
        m = re.search(r"k_gather_stencilILi(\d+)ELi(\d+)ELb(\d)ELi8ELb(\d)ELi(\d+)E([df])", name)
        if not m or m.group(3) != "1":                      # only the constant-table (CT) variants
            continue
        seen += 1
        vec = len(re.findall(r"LDC[.\w]* R\d+, c\[0x3\]", p))          # table reads with a vector-register index
        uni = len(re.findall(r"LDCU[.\w]* UR\d+, c\[0x3\]", p))       # ... through the uniform datapath
        assert uni >= 16 and vec <= 2, (name, vec, uni)
        if m.group(4) == "1" and m.group(6) == "d":
            assert "UTMALDG" in p, name
    assert seen >= 12
