"""gsr_norm2_noalloc (include/gsr_noalloc.h): the norm for callers that cannot allocate.

Who needs it: code that wants LSQR's |u| / |v| norm but must not call cudaMalloc -- a rank whose HBM
is already full (the Large system plus a framework's memory pool), a component that has to take all
device memory from its host application's pool, or a latency-critical path that cannot accept
cudaMalloc's device-wide synchronisation.  The entry point takes no handle and allocates nothing;
its partial sums go to a fixed 128 KiB array inside libgsr.so, shared by all calls on a GPU.

What is checked here: the new entry point returns what the EXISTING handle path computes for the same
vector -- gsr_lsqr with itnlim = 0 stops right after step 1 of LSQR and returns rnorm = beta_1 = |b|,
formed by the handle's k_sumsq + k_scalar on cudaMalloc'ed partial buffers -- on two calls in a row, the
second on a SHORTER vector, so that partial sums left in the shared scratch by the first call would
show up if the second call read them.  Tolerance: 1e-12 relative, the suite's aprod bound (for a sum of
squares sum|terms| is the sum itself); the two paths differ only in summation order.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  It passes alone in a fresh process (the first call then
does the per-device set-up) and after the other GPU tests (which never touch the built-in scratch).
"""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

from paper_2308_00778_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NORM_TOL = 1e-12


def test_noalloc_header_export_binding_agree():
    """CPU-side: libgsr.so exports what include/gsr_noalloc.h declares, the binding lists the same name and
    the same limits, and the source of the entry point contains no allocating call."""
    from paper_2308_00778_b200 import build, gsr
    src = open(os.path.join(ROOT, "include", "gsr_noalloc.h")).read()
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = sorted(set(re.findall(r"\b(gsr_[a-z0-9_]+)\s*\(", code)))
    assert names == sorted(gsr.NOALLOC_SYMBOLS) == ["gsr_norm2_noalloc"]
    lib = ctypes.CDLL(build.build())
    assert hasattr(lib, "gsr_norm2_noalloc")
    assert int(re.search(r"#define GSR_NOALLOC_CHUNK (\d+)", src).group(1)) == gsr.NOALLOC_CHUNK
    assert int(re.search(r"#define GSR_NOALLOC_MAX_PARTIALS (\d+)", src).group(1)) == gsr.NOALLOC_MAX_PARTIALS
    cu = open(os.path.join(ROOT, "paper_2308_00778_b200", "csrc", "gsr_noalloc.cu")).read()
    cu = re.sub(r"//.*", "", cu)
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cub::", "thrust::", "new ", "malloc("):
        assert banned not in cu, banned
    assert "cudaGetSymbolAddress" in cu


def _norm_on_handle_path(a):
    """|a| from the existing path: a Gaia-shaped system with len(a) rows whose known terms are a;
    gsr_lsqr(itnlim = 0) returns rnorm = beta_1 = |b| (k_sumsq + k_scalar on the handle's buffers)."""
    from paper_2308_00778_b200 import gsr
    obs = 100
    assert a.numel() % obs == 0
    cfg = synth.mini(seed=11, n_stars=a.numel() // obs, obs=obs, n_dof_att=500, n_instr=64)
    d = synth.generate(cfg, "cuda")
    with gsr.Gsr(a.numel(), cfg.n_stars, cfg.n_dof_att, cfg.n_instr) as G:
        G.gsr_upload(d["values"], d["matrixIndexAstro"], d["matrixIndexAtt"], d["instrCol"], a)
        r = G.gsr_lsqr(0, 0.0, 0.0, want_se=False)
    assert r.itn == 0
    return r.rnorm


@pytest.mark.gpu
def test_norm2_noalloc_matches_handle_path_on_two_calls_in_a_row():
    from paper_2308_00778_b200 import gsr
    rng = np.random.default_rng(2308)
    # 300,100 elements = 4 full chunks of 65,536 + a ragged one; then 70,000 = 1 full + a ragged one
    a_long = torch.from_numpy(rng.standard_normal(300_100) * 3.0).cuda()
    a_short = torch.from_numpy(rng.standard_normal(70_000) * 1e-3).cuda()
    want_long = _norm_on_handle_path(a_long)
    want_short = _norm_on_handle_path(a_short)
    assert want_long > 1e3 * want_short > 0.0     # stale partials of the long vector would swamp the short one

    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")   # the caller's output slots
    gsr.gsr_norm2_noalloc(a_long, out[0:1])
    gsr.gsr_norm2_noalloc(a_short, out[1:2])                           # second call, scratch still dirty
    got_long, got_short = out.tolist()
    assert abs(got_long - want_long) <= NORM_TOL * want_long, (got_long, want_long)
    assert abs(got_short - want_short) <= NORM_TOL * want_short, (got_short, want_short)
    # and against the definition, computed by torch in fp64 (not the oracle; a plain cross-check)
    assert abs(got_long - torch.linalg.vector_norm(a_long).item()) <= NORM_TOL * want_long
    assert abs(got_short - torch.linalg.vector_norm(a_short).item()) <= NORM_TOL * want_short

    # the summation order depends only on n: a repeat gives the same bits, whatever ran in between
    again = torch.empty(1, dtype=torch.float64, device="cuda")
    gsr.gsr_norm2_noalloc(a_long, again)
    assert again.item() == got_long
    # a prefix of a longer buffer (n passed explicitly), and the empty vector
    gsr.gsr_norm2_noalloc(a_long, again, n=70_000)
    ref = torch.linalg.vector_norm(a_long[:70_000]).item()
    assert abs(again.item() - ref) <= NORM_TOL * ref
    gsr.gsr_norm2_noalloc(a_long, again, n=0)
    assert again.item() == 0.0


@pytest.mark.gpu
def test_norm2_noalloc_rejects_what_the_scratch_cannot_hold():
    """n beyond GSR_NOALLOC_MAX_N is refused with GSR_EINVAL and a message naming the limit, before
    anything is launched (the pointer is never dereferenced: a one-element tensor stands in)."""
    from paper_2308_00778_b200 import gsr
    lib = gsr.load_library()
    a = torch.ones(1, dtype=torch.float64, device="cuda")
    out = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    err = ctypes.create_string_buffer(512)
    st = torch.cuda.current_stream().cuda_stream or None
    rc = lib.gsr_norm2_noalloc(a.data_ptr(), gsr.NOALLOC_MAX_N + 1, out.data_ptr(), 0, st, err, len(err))
    assert rc == gsr.GSR_EINVAL
    msg = err.value.decode()
    assert str(gsr.NOALLOC_MAX_N) in msg and str(gsr.NOALLOC_MAX_N + 1) in msg, msg
    assert lib.gsr_norm2_noalloc(a.data_ptr(), -1, out.data_ptr(), 0, st, err, len(err)) == gsr.GSR_EINVAL
    assert lib.gsr_norm2_noalloc(a.data_ptr(), 1, None, 0, st, None, 0) == gsr.GSR_EINVAL
    torch.cuda.synchronize()
    assert out.item() == 7.0            # untouched
    # the largest size is accepted as far as the check goes: here only n = 1 is run for real
    assert lib.gsr_norm2_noalloc(a.data_ptr(), 1, out.data_ptr(), 0, st, err, len(err)) == gsr.GSR_OK
    assert out.item() == 1.0
