"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/gsr.h declares, the binding lists the same names, and without a GPU the product path
fails loudly instead of falling back."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols(name="gsr.h"):
    src = open(os.path.join(ROOT, "include", name)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gsr_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _header_symbols()
    for must in ("gsr_create", "gsr_upload", "gsr_aprod1", "gsr_aprod2", "gsr_lsqr", "gsr_destroy",
                 "gsr_precondition"):
        assert must in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2308_00778_b200 import build, gsr
    path = build.build()
    lib = ctypes.CDLL(path)
    names = _header_symbols()
    assert sorted(gsr.SYMBOLS) == names
    for n in names:
        assert hasattr(lib, n), n
    # the measurement hook lives in its own header, outside the product ABI
    bench_names = _header_symbols("gsr_bench.h")
    assert bench_names == sorted(gsr.BENCH_SYMBOLS) == ["gsr_bench_set", "gsr_time_aprod"]
    assert "gsr_time_aprod" not in names
    for n in bench_names:
        assert hasattr(lib, n), n


def test_binding_struct_sizes_match_header():
    # gsr_layout: 6*i64 + 5*i32 + u32 flags + pointer = 80 bytes; gsr_result: 2 ptr + i32(+4) + i64 + 5 f64 = 72
    from paper_2308_00778_b200 import gsr
    assert ctypes.sizeof(gsr._Layout) == 80
    assert ctypes.sizeof(gsr._Result) == 72


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_means_error_not_fallback():
    from paper_2308_00778_b200 import gsr
    with pytest.raises(gsr.GsrError) as e:
        gsr.Gsr(10, 2, 8, 8)
    assert e.value.code == gsr.GSR_ECUDA


def test_library_reads_no_environment_variables():
    """Kernel-path choices are gsr_layout.flags, per handle: nothing in the library calls getenv."""
    for f in ("gsr.cu", "gsr_kernels.cuh"):
        assert "getenv" not in open(os.path.join(ROOT, "paper_2308_00778_b200", "csrc", f)).read()


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2308_00778_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "gsr_oracle" not in txt, f
