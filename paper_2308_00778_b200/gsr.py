"""ctypes binding of libgsr.so (include/gsr.h) -- argument marshalling only.

Same names as the C ABI.  Tensors are torch CUDA (or CPU/numpy for the "host or device"
arguments); torch is used for device memory only.  There is no CPU fallback: if libgsr.so is
missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
# GSR_LIBRARY selects another build of the same ABI (the bounds-checked libgsr_check.so); read by this binding only
LIB_PATH = os.environ.get("GSR_LIBRARY") or os.path.join(_PKG, "libgsr.so")

GSR_OK, GSR_EINVAL, GSR_EINDEX, GSR_ENOMEM, GSR_ECUDA, GSR_ESTATE = 0, -1, -2, -3, -4, -5
TRACE_CAP = 4096
# gsr_layout.flags (include/gsr.h)
GSR_FLAG_NO_ATT_COPY, GSR_FLAG_NO_FUSE, GSR_FLAG_NO_TEX, GSR_FLAG_INS_COPY = 1, 2, 4, 8
# gsr_path_info bits
GSR_PATH_ATT_COPY, GSR_PATH_FUSED, GSR_PATH_INSTR_MATCH, GSR_PATH_TEX, GSR_PATH_IC16, GSR_PATH_UT, GSR_PATH_INS_COPY = 1, 2, 4, 8, 16, 32, 64
# gsr_time_aprod selectors (include/gsr_bench.h)
GSR_TIME_APROD1_GROUP, GSR_TIME_APROD2_GROUP = 1, 2
GSR_TIME_K_APROD1, GSR_TIME_K_APROD2_MAIN, GSR_TIME_K_APROD2_ATT, GSR_TIME_K_FUSED = 11, 12, 13, 21
GSR_TIME_K_INS_SCATTER, GSR_TIME_K_U_TO_TIME, GSR_TIME_OVERLAP_PROBE = 14, 15, 31

# every symbol include/gsr.h declares (tests check that the library exports each one)
SYMBOLS = [
    "gsr_create", "gsr_destroy", "gsr_last_error", "gsr_bad_row", "gsr_ncols", "gsr_nrows",
    "gsr_upload", "gsr_upload_rows", "gsr_upload_finish", "gsr_upload_constraints", "gsr_set_b",
    "gsr_get_star_rowptr", "gsr_precondition", "gsr_get_colscale", "gsr_get_values",
    "gsr_aprod1", "gsr_aprod2", "gsr_lsqr", "gsr_get_trace", "gsr_path_info", "gsr_last_timing",
    "gsr_set_cov_pairs", "gsr_get_cov",
]
# the measurement hook of include/gsr_bench.h
BENCH_SYMBOLS = ["gsr_bench_set", "gsr_time_aprod"]
# the allocation-free entry point of include/gsr_noalloc.h
NOALLOC_SYMBOLS = ["gsr_norm2_noalloc"]
NOALLOC_CHUNK, NOALLOC_MAX_PARTIALS = 65536, 16384
NOALLOC_MAX_N = NOALLOC_CHUNK * NOALLOC_MAX_PARTIALS


class GsrError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libgsr error {code}: {msg}")
        self.code = code


class _Layout(C.Structure):
    _fields_ = [("n_obs", C.c_int64), ("n_stars", C.c_int64), ("n_dof_att", C.c_int64),
                ("n_instr", C.c_int64), ("n_con", C.c_int64), ("n_con_nnz", C.c_int64),
                ("n_astro_par", C.c_int32), ("n_att_par", C.c_int32), ("n_instr_par", C.c_int32),
                ("n_glob_par", C.c_int32), ("device", C.c_int32), ("flags", C.c_uint32),
                ("stream", C.c_void_p)]


class _Result(C.Structure):
    _fields_ = [("x", C.c_void_p), ("se", C.c_void_p), ("istop", C.c_int32), ("itn", C.c_int64),
                ("anorm", C.c_double), ("acond", C.c_double), ("rnorm", C.c_double),
                ("arnorm", C.c_double), ("xnorm", C.c_double)]


_lib = None


def load_library():
    """dlopen libgsr.so (built in-tree by paper_2308_00778_b200.build).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    P, I64, I32, D = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    sig = {
        "gsr_create": (I32, [C.POINTER(_Layout), C.POINTER(P)]),
        "gsr_destroy": (I32, [P]),
        "gsr_last_error": (C.c_char_p, [P]),
        "gsr_bad_row": (I64, [P]),
        "gsr_ncols": (I64, [P]),
        "gsr_nrows": (I64, [P]),
        "gsr_upload": (I32, [P, P, P, P, P, P]),
        "gsr_upload_rows": (I32, [P, I64, I64, P, P, P, P, P]),
        "gsr_upload_finish": (I32, [P, P]),
        "gsr_upload_constraints": (I32, [P, P, P, P]),
        "gsr_set_b": (I32, [P, P]),
        "gsr_get_star_rowptr": (I32, [P, P]),
        "gsr_precondition": (I32, [P]),
        "gsr_get_colscale": (I32, [P, P]),
        "gsr_get_values": (I32, [P, P, P]),
        "gsr_aprod1": (I32, [P, P, P]),
        "gsr_aprod2": (I32, [P, P, P]),
        "gsr_lsqr": (I32, [P, I64, D, D, D, C.POINTER(_Result)]),
        "gsr_get_trace": (I32, [P, P, I64, C.POINTER(I64)]),
        "gsr_set_cov_pairs": (I32, [P, I64, P, P]),
        "gsr_get_cov": (I32, [P, P]),
        "gsr_path_info": (I32, [P]),
        "gsr_last_timing": (I32, [P, C.POINTER(D), C.POINTER(I64)]),
        "gsr_time_aprod": (I32, [P, I32, I32, C.POINTER(D)]),
        "gsr_bench_set": (I32, [P, C.c_char_p, I64]),
        "gsr_norm2_noalloc": (I32, [P, I64, P, I32, P, C.c_char_p, I64]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    _lib = lib
    return lib


def _ptr(a, dtype=None, what="array"):
    """Raw pointer of a contiguous torch tensor / numpy array (or None)."""
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        if dtype is not None and a.dtype != dtype:
            raise TypeError(f"{what}: expected {dtype}, got {a.dtype}")
        if not a.is_contiguous():
            raise ValueError(f"{what}: tensor must be contiguous")
        return a.data_ptr()
    if isinstance(a, np.ndarray):
        want = {torch.float64: np.float64, torch.int64: np.int64, torch.int32: np.int32}.get(dtype)
        if want is not None and a.dtype != want:
            raise TypeError(f"{what}: expected {want}, got {a.dtype}")
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError(f"{what}: array must be C-contiguous")
        return a.ctypes.data
    raise TypeError(f"{what}: torch tensor or numpy array expected")


def _dev(a, dtype, what, numel=None):
    if not (isinstance(a, torch.Tensor) and a.is_cuda):
        raise TypeError(f"{what}: CUDA tensor required")
    if numel is not None and a.numel() != numel:
        raise ValueError(f"{what}: expected {numel} elements, got {a.numel()}")
    return _ptr(a, dtype, what)


@dataclass
class LsqrResult:
    x: torch.Tensor
    se: torch.Tensor | None
    istop: int
    itn: int
    anorm: float
    acond: float
    rnorm: float
    arnorm: float
    xnorm: float
    loop_ms: float = 0.0
    kernel_launches: int = 0


class Gsr:
    """One system on one GPU.  Methods mirror the C entry points one to one."""

    def __init__(self, n_obs, n_stars, n_dof_att, n_instr, n_con=0, n_con_nnz=0, device=0, stream=None, flags=0,
                 n_glob=1, n_astro_par=5, n_att_par=12, n_instr_par=6):
        self.lib = load_library()
        self._h = C.c_void_p()
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream(device).cuda_stream
        L = _Layout(n_obs, n_stars, n_dof_att, n_instr, n_con, n_con_nnz, n_astro_par, n_att_par, n_instr_par, n_glob,
                    device, flags, stream or None)
        self.n_par = n_astro_par + n_att_par + n_instr_par + n_glob
        rc = self.lib.gsr_create(C.byref(L), C.byref(self._h))
        if rc != GSR_OK:
            msg = self.lib.gsr_last_error(self._h).decode() if self._h else "gsr_create failed"
            if self._h:
                self.lib.gsr_destroy(self._h)
                self._h = C.c_void_p()
            raise GsrError(rc, msg)
        self.device = torch.device("cuda", device)
        self.n = int(self.lib.gsr_ncols(self._h))
        self.m_tot = int(self.lib.gsr_nrows(self._h))
        self.n_obs, self.n_stars, self.n_con, self.n_con_nnz = n_obs, n_stars, n_con, n_con_nnz

    def _ck(self, rc):
        if rc != GSR_OK:
            raise GsrError(rc, self.lib.gsr_last_error(self._h).decode())

    def close(self):
        h = getattr(self, "_h", None)
        if h:
            self._h = None          # (no module globals here: close also runs from __del__ at interpreter exit)
            self.lib.gsr_destroy(h)

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- upload -----------------------------------------------------------------------
    def gsr_upload(self, values, matrixIndexAstro, matrixIndexAtt, instrCol, b):
        self._ck(self.lib.gsr_upload(self._h, _ptr(values, torch.float64, "values"),
                                     _ptr(matrixIndexAstro, torch.int64, "matrixIndexAstro"),
                                     _ptr(matrixIndexAtt, torch.int64, "matrixIndexAtt"),
                                     _ptr(instrCol, torch.int32, "instrCol"), _ptr(b, torch.float64, "b")))

    def gsr_upload_rows(self, row0, nrows, values, matrixIndexAstro, matrixIndexAtt, instrCol, b):
        self._ck(self.lib.gsr_upload_rows(self._h, row0, nrows, _ptr(values, torch.float64, "values"),
                                          _ptr(matrixIndexAstro, torch.int64, "matrixIndexAstro"),
                                          _ptr(matrixIndexAtt, torch.int64, "matrixIndexAtt"),
                                          _ptr(instrCol, torch.int32, "instrCol"), _ptr(b, torch.float64, "b")))

    def gsr_upload_finish(self, b_tail=None):
        self._ck(self.lib.gsr_upload_finish(self._h, _ptr(b_tail, torch.float64, "b_tail")))

    def gsr_upload_constraints(self, rowptr, col, val):
        self._ck(self.lib.gsr_upload_constraints(self._h, _ptr(rowptr, torch.int64, "rowptr"),
                                                 _ptr(col, torch.int64, "col"), _ptr(val, torch.float64, "val")))

    def gsr_set_b(self, b):
        self._ck(self.lib.gsr_set_b(self._h, _ptr(b, torch.float64, "b")))

    def gsr_bad_row(self):
        return int(self.lib.gsr_bad_row(self._h))

    # ---- derived data -----------------------------------------------------------------
    def gsr_get_star_rowptr(self):
        out = torch.empty(self.n_stars + 1, dtype=torch.int64, device=self.device)
        self._ck(self.lib.gsr_get_star_rowptr(self._h, out.data_ptr()))
        return out

    def gsr_precondition(self):
        self._ck(self.lib.gsr_precondition(self._h))

    def gsr_get_colscale(self):
        out = torch.empty(self.n, dtype=torch.float64, device=self.device)
        self._ck(self.lib.gsr_get_colscale(self._h, out.data_ptr()))
        return out

    def gsr_get_values(self):
        out = torch.empty((self.n_obs, self.n_par), dtype=torch.float64, device=self.device)
        con = torch.empty(self.n_con_nnz, dtype=torch.float64, device=self.device) if self.n_con_nnz else None
        self._ck(self.lib.gsr_get_values(self._h, out.data_ptr(), None if con is None else con.data_ptr()))
        return out, con

    # ---- products ---------------------------------------------------------------------
    def gsr_aprod1(self, x, y):
        """y += A x, in place on the CUDA tensor y."""
        self._ck(self.lib.gsr_aprod1(self._h, _dev(x, torch.float64, "x", self.n),
                                     _dev(y, torch.float64, "y", self.m_tot)))
        return y

    def gsr_aprod2(self, y, x):
        """x += A^T y, in place on the CUDA tensor x."""
        self._ck(self.lib.gsr_aprod2(self._h, _dev(y, torch.float64, "y", self.m_tot),
                                     _dev(x, torch.float64, "x", self.n)))
        return x

    # ---- solver -----------------------------------------------------------------------
    def gsr_lsqr(self, itnlim, atol, btol, conlim=0.0, want_se=True, host_out=False) -> LsqrResult:
        if host_out:
            x = torch.empty(self.n, dtype=torch.float64).pin_memory()
            se = torch.empty(self.n, dtype=torch.float64).pin_memory() if want_se else None
        else:
            x = torch.empty(self.n, dtype=torch.float64, device=self.device)
            se = torch.empty(self.n, dtype=torch.float64, device=self.device) if want_se else None
        R = _Result(x.data_ptr(), None if se is None else se.data_ptr(), 0, 0, 0.0, 0.0, 0.0, 0.0, 0.0)
        self._ck(self.lib.gsr_lsqr(self._h, int(itnlim), float(atol), float(btol), float(conlim), C.byref(R)))
        ms, nl = C.c_double(), C.c_int64()
        self._ck(self.lib.gsr_last_timing(self._h, C.byref(ms), C.byref(nl)))
        return LsqrResult(x, se, int(R.istop), int(R.itn), R.anorm, R.acond, R.rnorm, R.arnorm, R.xnorm,
                          ms.value, nl.value)

    def gsr_get_trace(self, max_itn=TRACE_CAP):
        out = np.zeros((max_itn, 5))
        nw = C.c_int64()
        self._ck(self.lib.gsr_get_trace(self._h, out.ctypes.data, max_itn, C.byref(nw)))
        return out[: nw.value]

    def gsr_set_cov_pairs(self, pi, pj):
        """Couples (pi[q], pj[q]) of unknowns whose covariance the following gsr_lsqr calls estimate (i64, host or device)."""
        npairs = 0 if pi is None else int(pi.shape[0])
        self._n_pairs = npairs
        self._ck(self.lib.gsr_set_cov_pairs(self._h, npairs, _ptr(pi, torch.int64, "pi"), _ptr(pj, torch.int64, "pj")))

    def gsr_get_cov(self):
        out = torch.empty(getattr(self, "_n_pairs", 0), dtype=torch.float64, device=self.device)
        self._ck(self.lib.gsr_get_cov(self._h, out.data_ptr()))
        return out

    def gsr_path_info(self):
        return int(self.lib.gsr_path_info(self._h))

    def gsr_bench_set(self, key, value):
        self._ck(self.lib.gsr_bench_set(self._h, key.encode(), int(value)))

    def gsr_time_aprod(self, which, reps):
        ms = C.c_double()
        self._ck(self.lib.gsr_time_aprod(self._h, which, reps, C.byref(ms)))
        return ms.value


def gsr_norm2_noalloc(a, out, n=None, stream=None):
    """out[0] = |a[:n]|_2 through gsr_norm2_noalloc (include/gsr_noalloc.h), the entry point for callers that
    cannot allocate device memory: no handle, and the library itself allocates nothing -- its scratch is a fixed
    array inside libgsr.so.  Both tensors are the CALLER's: `a` a float64 CUDA tensor, `out` a float64 CUDA
    tensor of one element on the same GPU (this binding does not create it, so that the call stays free of
    allocations end to end).  n defaults to a.numel(); the library rejects n > NOALLOC_MAX_N with GSR_EINVAL.
    Calls share the built-in scratch: never run two of them at the same time on one GPU."""
    lib = load_library()
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.numel() >= 1):
        raise TypeError("out: CUDA tensor with one element required")
    n = a.numel() if n is None else int(n)
    pa = _dev(a, torch.float64, "a") if a is not None else None
    if a is not None and (a.device != out.device or n > a.numel()):
        raise ValueError("a and out must be on the same GPU and n <= a.numel()")
    device = out.device.index if out.device.index is not None else torch.cuda.current_device()
    if stream is None:
        stream = torch.cuda.current_stream(device).cuda_stream
    err = C.create_string_buffer(512)
    rc = lib.gsr_norm2_noalloc(pa, n, _dev(out, torch.float64, "out"), device, stream or None, err, len(err))
    if rc != GSR_OK:
        raise GsrError(rc, err.value.decode())
    return out
