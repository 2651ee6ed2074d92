"""Build step of libgsr.so: nvcc for sm_100a only, in-tree (the .so travels with the snapshot).

``python -m paper_2308_00778_b200.build`` or ``build()`` from ``__graft_entry__``.
"""
from __future__ import annotations

import os
import shutil
import subprocess

_PKG = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_PKG)
SRC = [os.path.join(_PKG, "csrc", "gsr.cu"), os.path.join(_PKG, "csrc", "gsr_noalloc.cu")]
DEPS = SRC + [os.path.join(_PKG, "csrc", "gsr_kernels.cuh"), os.path.join(_ROOT, "include", "gsr.h"),
              os.path.join(_ROOT, "include", "gsr_bench.h"), os.path.join(_ROOT, "include", "gsr_noalloc.h")]
LIB = os.path.join(_PKG, "libgsr.so")
LIB_CHECK = os.path.join(_PKG, "libgsr_check.so")     # -DGSR_BOUNDS_CHECK: every gather / scatter index asserted

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libgsr.so cannot be built (there is no CPU fallback)")


def up_to_date(lib: str = LIB) -> bool:
    return os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False, check: bool = False) -> str:
    """check=True builds the bounds-checked variant (libgsr_check.so); point GSR_LIBRARY at it to run the tests on it."""
    lib = LIB_CHECK if check else LIB
    if force or not up_to_date(lib):
        tmp = lib + f".tmp{os.getpid()}"
        cmd = [_nvcc(), *NVCC_FLAGS, "-I", os.path.join(_ROOT, "include"), "-o", tmp, *SRC]
        if check:
            cmd.insert(1, "-DGSR_BOUNDS_CHECK")
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose=True, check="--check" in sys.argv))
