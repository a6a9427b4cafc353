"""Build libflatspin_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "csrc", "flatspin.cu")
HDR = os.path.join(ROOT, "include", "flatspin.h")
LIB = os.path.join(HERE, "libflatspin_b200.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "550"]


def nvcc_path() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [HDR] + [os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc"))]
    newest = max(os.path.getmtime(f) for f in deps)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-I", os.path.join(ROOT, "include"), SRC, "-o", LIB]
        subprocess.check_call(cmd)
    return LIB


def build_profile(out_dir: str) -> str:
    """The same sources with the phase timers compiled in (-DFS_RELAX_PROFILE -DFS_BATCH_PROFILE): clock64 / %globaltimer
    per phase of k_relax and k_relax_batch, read back through fs_debug_relax_profile / fs_debug_batch_profile.
    Used by `bench.py --phase-profile` only; the shipped library has none of it."""
    os.makedirs(out_dir, exist_ok=True)
    lib = os.path.join(out_dir, "libflatspin_b200_profile.so")
    cmd = [nvcc_path()] + NVCC_FLAGS + ["-DFS_RELAX_PROFILE", "-DFS_BATCH_PROFILE", "-I", os.path.join(ROOT, "include"), SRC, "-o", lib]
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose=True))
