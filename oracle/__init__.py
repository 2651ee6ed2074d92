"""CPU oracle for the AVU-GSR LSQR hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes loader around ``oracle/gsr_oracle.c`` (plain C, FP64, single thread,
``gcc -O2 -ffp-contract=off``).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.
It imports nothing from ``paper_2308_00778_b200`` and that package never imports it.

The arithmetic lives entirely in the C file; this module only marshals numpy arrays.
See the header of ``gsr_oracle.c`` for the citations (PAPER.md lines) and for what pins
each function.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gsr_oracle.c")
_LIB = os.path.join(_HERE, "libgsr_oracle.so")

N_PAR = 24          # row width of the production layout (n_glob = 1); in general 23 + n_glob


def build(force: bool = False) -> str:
    """Compile the oracle (gcc, no FMA contraction).  Returns the path of the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-shared", "-fPIC",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Sys(C.Structure):
    _fields_ = [
        ("n_obs", C.c_int64), ("n_stars", C.c_int64), ("n_dof_att", C.c_int64),
        ("n_instr", C.c_int64), ("n_con", C.c_int64), ("n_glob", C.c_int64),
        ("V", C.c_void_p), ("ia", C.c_void_p), ("iatt", C.c_void_p), ("ic", C.c_void_p),
        ("con_rowptr", C.c_void_p), ("con_col", C.c_void_p), ("con_val", C.c_void_p),
        ("n_astro_par", C.c_int64), ("n_att_par", C.c_int64), ("n_instr_par", C.c_int64),
    ]


class _Res(C.Structure):
    _fields_ = [("istop", C.c_int32), ("itn", C.c_int64), ("anorm", C.c_double),
                ("acond", C.c_double), ("rnorm", C.c_double), ("arnorm", C.c_double),
                ("xnorm", C.c_double)]


_SRC_OMP = os.path.join(_HERE, "gsr_oracle_omp.c")
_LIB_OMP = os.path.join(_HERE, "libgsr_oracle_omp.so")


def build_omp(force: bool = False) -> str:
    """Compile the OpenMP-threaded restatement (bench.py's all-core cpu_baseline only; not the parity oracle)."""
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC_OMP):
        tmp = _LIB_OMP + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-shared", "-fPIC",
             "-o", tmp, _SRC_OMP, "-lm"])
        os.replace(tmp, _LIB_OMP)
    return _LIB_OMP


_lib = None
_lib_omp = None


def _load_omp():
    global _lib_omp
    if _lib_omp is None:
        lib = C.CDLL(build_omp())
        P = C.c_void_p
        lib.gsr_omp_threads.restype = C.c_int
        lib.gsr_omp_set_threads.argtypes = [C.c_int]
        lib.gsr_omp_aprod1.restype = None
        lib.gsr_omp_aprod1.argtypes = [P, P, P]
        lib.gsr_omp_aprod2.restype = None
        lib.gsr_omp_aprod2.argtypes = [P, P, P]
        lib.gsr_omp_lsqr.restype = C.c_int
        lib.gsr_omp_lsqr.argtypes = [P, P, C.c_int64, C.c_double, C.c_double, C.c_double, P, P, P, P]
        _lib_omp = lib
    return _lib_omp


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        P = C.c_void_p
        lib.gsr_oracle_ncols.restype = C.c_int64
        lib.gsr_oracle_ncols.argtypes = [P]
        lib.gsr_oracle_col.restype = C.c_int64
        lib.gsr_oracle_col.argtypes = [P, C.c_int64, C.c_int]
        lib.gsr_oracle_aprod1.restype = None
        lib.gsr_oracle_aprod1.argtypes = [P, P, P, P]
        lib.gsr_oracle_aprod2.restype = None
        lib.gsr_oracle_aprod2.argtypes = [P, P, P, P]
        lib.gsr_oracle_norm.restype = C.c_double
        lib.gsr_oracle_norm.argtypes = [P, C.c_int64]
        lib.gsr_oracle_precondition.restype = None
        lib.gsr_oracle_precondition.argtypes = [P, P]
        lib.gsr_oracle_lsqr.restype = C.c_int
        lib.gsr_oracle_lsqr.argtypes = [P, P, C.c_int64, C.c_double, C.c_double, C.c_double,
                                        P, P, P, P, P]
        lib.gsr_oracle_lsqr_cov.restype = C.c_int
        lib.gsr_oracle_lsqr_cov.argtypes = [P, P, C.c_int64, C.c_double, C.c_double, C.c_double,
                                            P, P, P, P, P, C.c_int64, P, P, P]
        _lib = lib
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data


@dataclass
class LsqrResult:
    x: np.ndarray
    se: np.ndarray
    istop: int
    itn: int
    anorm: float
    acond: float
    rnorm: float
    arnorm: float
    xnorm: float
    trace: np.ndarray | None = None  # [itn, 5]: rnorm, arnorm, anorm, acond, xnorm
    cov: np.ndarray | None = None    # covariances of the couples passed to lsqr(pairs=...)


class OracleSystem:
    """Holds (private copies of) the upload-format arrays of one system.

    values [m, n_par] f64 row-major with n_par = n_astro_par + n_att_par + n_instr_par + n_glob;
    matrixIndexAstro [m] i64 (= n_astro_par*star, non-decreasing); matrixIndexAtt [m] i64 (axis-0 start);
    instrCol [m, n_instr_par] i32; optional constraint rows as CSR with absolute columns.
    5 / 12 / 6 / 1 is the paper's production layout (24 per row); a section of width 0 has no
    columns and its index array is ignored (may be None).
    """

    def __init__(self, n_stars, n_dof_att, n_instr, values, matrixIndexAstro, matrixIndexAtt,
                 instrCol, con_rowptr=None, con_col=None, con_val=None, n_glob=1,
                 n_astro_par=5, n_att_par=12, n_instr_par=6):
        self.lib = _load()
        self.n_glob = int(n_glob)
        self.n_astro_par, self.n_att_par, self.n_instr_par = int(n_astro_par), int(n_att_par), int(n_instr_par)
        assert 0 <= self.n_astro_par <= 5 and self.n_att_par in (0, 12) and 0 <= self.n_instr_par <= 6 and self.n_glob >= 0
        self.n_par = self.n_astro_par + self.n_att_par + self.n_instr_par + self.n_glob
        assert self.n_par > 0
        self.V = np.array(values, dtype=np.float64, order="C", copy=True).reshape(-1, self.n_par)
        self.m = self.V.shape[0]
        zeros = np.zeros(self.m, dtype=np.int64)
        self.ia = np.array(matrixIndexAstro if self.n_astro_par else zeros, dtype=np.int64, copy=True).reshape(-1)
        self.iatt = np.array(matrixIndexAtt if self.n_att_par else zeros, dtype=np.int64, copy=True).reshape(-1)
        self.ic = (np.array(instrCol, dtype=np.int32, order="C", copy=True).reshape(-1, self.n_instr_par)
                   if self.n_instr_par else np.zeros((self.m, 0), dtype=np.int32))
        assert self.ia.shape[0] == self.m and self.iatt.shape[0] == self.m and self.ic.shape[0] == self.m
        self.n_stars, self.n_dof_att, self.n_instr = int(n_stars), int(n_dof_att), int(n_instr)
        if con_rowptr is not None:
            self.con_rowptr = np.array(con_rowptr, dtype=np.int64, copy=True)
            self.con_col = np.array(con_col, dtype=np.int64, copy=True)
            self.con_val = np.array(con_val, dtype=np.float64, copy=True)
            self.n_con = self.con_rowptr.shape[0] - 1
        else:
            self.con_rowptr = np.zeros(1, dtype=np.int64)
            self.con_col = np.zeros(0, dtype=np.int64)
            self.con_val = np.zeros(0, dtype=np.float64)
            self.n_con = 0
        self.p = None
        self._s = _Sys(self.m, self.n_stars, self.n_dof_att, self.n_instr, self.n_con, self.n_glob,
                       _ptr(self.V), _ptr(self.ia), _ptr(self.iatt), _ptr(self.ic),
                       _ptr(self.con_rowptr), _ptr(self.con_col), _ptr(self.con_val),
                       self.n_astro_par, self.n_att_par, self.n_instr_par)
        self._sp = C.addressof(self._s)
        self.n = int(self.lib.gsr_oracle_ncols(self._sp))
        self.m_tot = self.m + self.n_con

    def col(self, i: int, k: int) -> int:
        return int(self.lib.gsr_oracle_col(self._sp, i, k))

    def aprod1(self, x, y, want_abs=False):
        """y += A x (in place on a float64 copy of y); returns y or (y, abs bound)."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.array(y, dtype=np.float64, copy=True)
        assert x.shape == (self.n,) and y.shape == (self.m_tot,)
        ab = np.zeros(self.m_tot) if want_abs else None
        self.lib.gsr_oracle_aprod1(self._sp, _ptr(x), _ptr(y), _ptr(ab))
        return (y, ab) if want_abs else y

    def aprod2(self, y, x, want_abs=False):
        """x += A^T y; returns x or (x, abs bound)."""
        y = np.ascontiguousarray(y, dtype=np.float64)
        x = np.array(x, dtype=np.float64, copy=True)
        assert x.shape == (self.n,) and y.shape == (self.m_tot,)
        ab = np.zeros(self.n) if want_abs else None
        self.lib.gsr_oracle_aprod2(self._sp, _ptr(y), _ptr(x), _ptr(ab))
        return (x, ab) if want_abs else x

    def precondition(self):
        """Compute p, scale the stored A in place; returns p."""
        assert self.p is None, "already preconditioned"
        self.p = np.zeros(self.n)
        self.lib.gsr_oracle_precondition(self._sp, _ptr(self.p))
        return self.p

    def lsqr(self, b, itnlim, atol, btol, conlim=0.0, want_trace=False, pairs=None) -> LsqrResult:
        """LSQR on the system as stored; if preconditioned, returns x = p*z, se = p*se_z.
        pairs = (i[], j[]): also the covariances of those couples of unknowns (gsr_oracle_lsqr_cov)."""
        b = np.ascontiguousarray(b, dtype=np.float64)
        assert b.shape == (self.m_tot,)
        x = np.zeros(self.n)
        se = np.zeros(self.n)
        res = _Res()
        trace = np.zeros((max(int(itnlim), 1), 5)) if want_trace else None
        cov = None
        if pairs is None:
            rc = self.lib.gsr_oracle_lsqr(self._sp, _ptr(b), int(itnlim), float(atol), float(btol),
                                          float(conlim), _ptr(self.p), _ptr(x), _ptr(se),
                                          C.addressof(res), _ptr(trace))
        else:
            pi = np.ascontiguousarray(pairs[0], dtype=np.int64)
            pj = np.ascontiguousarray(pairs[1], dtype=np.int64)
            assert pi.shape == pj.shape and pi.ndim == 1
            assert pi.size == 0 or (min(pi.min(), pj.min()) >= 0 and max(pi.max(), pj.max()) < self.n)
            cov = np.zeros(pi.shape[0])
            rc = self.lib.gsr_oracle_lsqr_cov(self._sp, _ptr(b), int(itnlim), float(atol), float(btol),
                                              float(conlim), _ptr(self.p), _ptr(x), _ptr(se),
                                              C.addressof(res), _ptr(trace), pi.shape[0], _ptr(pi), _ptr(pj), _ptr(cov))
        if rc != 0:
            raise MemoryError("oracle lsqr allocation failed")
        return LsqrResult(x, se, int(res.istop), int(res.itn), res.anorm, res.acond, res.rnorm,
                          res.arnorm, res.xnorm, None if trace is None else trace[: res.itn], cov)


class OmpRunner:
    """The OpenMP-threaded restatement (gsr_oracle_omp.c) on an OracleSystem's arrays: the paper's section 3.1
    threading.  For bench.py's all-core cpu_baseline; checked against the oracle in the tests."""

    def __init__(self, S: OracleSystem, threads: int = 0):
        assert (S.n_astro_par, S.n_att_par, S.n_instr_par) == (5, 12, 6), "the threaded restatement covers the 5/12/6/n_glob layout"
        self.S = S
        self.lib = _load_omp()
        self.lib.gsr_omp_set_threads(int(threads) if threads > 0 else (os.cpu_count() or 1))
        self.threads = int(self.lib.gsr_omp_threads())

    def aprod1(self, x, y):
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.array(y, dtype=np.float64, copy=True)
        self.lib.gsr_omp_aprod1(self.S._sp, _ptr(x), _ptr(y))
        return y

    def aprod2(self, y, x):
        y = np.ascontiguousarray(y, dtype=np.float64)
        x = np.array(x, dtype=np.float64, copy=True)
        self.lib.gsr_omp_aprod2(self.S._sp, _ptr(y), _ptr(x))
        return x

    def lsqr(self, b, itnlim, atol, btol, conlim=0.0) -> LsqrResult:
        b = np.ascontiguousarray(b, dtype=np.float64)
        x = np.zeros(self.S.n)
        se = np.zeros(self.S.n)
        res = _Res()
        rc = self.lib.gsr_omp_lsqr(self.S._sp, _ptr(b), int(itnlim), float(atol), float(btol), float(conlim),
                                   _ptr(self.S.p), _ptr(x), _ptr(se), C.addressof(res))
        if rc != 0:
            raise MemoryError("omp lsqr allocation failed")
        return LsqrResult(x, se, int(res.istop), int(res.itn), res.anorm, res.acond, res.rnorm, res.arnorm, res.xnorm)


def norm(a) -> float:
    """Eq. 4 of the paper (max-scaled Euclidean norm)."""
    a = np.ascontiguousarray(a, dtype=np.float64).reshape(-1)
    return float(_load().gsr_oracle_norm(_ptr(a), a.shape[0]))
