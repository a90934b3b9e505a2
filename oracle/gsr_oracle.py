"""ctypes wrapper of the CPU oracle (oracle/gsr_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.  Arrays are numpy, caller
form (the paper's M_i / I_c / A_d): star_idx i32[m], att_start i32[m],
instr_col i32[m,6], values f64[m,24].
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
_LIB_OMP = os.path.join(_HERE, "libgsr_oracle_omp.so")


def build(force: bool = False, omp: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, reading A6).  omp=True: the timing-only
    OpenMP build of the same file (-DORC_OPENMP, the paper's CPU scheme)."""
    out = _LIB_OMP if omp else _LIB
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        tmp = out + f".tmp{os.getpid()}"
        extra = ["-fopenmp", "-DORC_OPENMP"] if omp else []
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared",
                               *extra, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, out)
    return out


class _Dims(C.Structure):
    _fields_ = [("n_rows", C.c_int64), ("n_stars", C.c_int64), ("n_dfa", C.c_int64),
                ("n_instr", C.c_int64)]


class _Result(C.Structure):
    _fields_ = [("istop", C.c_int32), ("istop_natural", C.c_int32), ("itn", C.c_int64),
                ("itn_natural", C.c_int64), ("rnorm", C.c_double), ("arnorm", C.c_double),
                ("anorm", C.c_double), ("acond", C.c_double), ("xnorm", C.c_double),
                ("bnorm", C.c_double)]


@dataclass
class LsqrResult:
    x: np.ndarray
    istop: int
    itn: int
    istop_natural: int
    itn_natural: int
    rnorm: float
    arnorm: float
    anorm: float
    acond: float
    xnorm: float
    bnorm: float
    hist: np.ndarray | None = None
    var: np.ndarray | None = None      # sum_k (w_j/rho_k)^2 of the iterated (scaled) system
    se: np.ndarray | None = None       # standard errors of x (multiplied by p when scaled)


_libs = {}


def lib(omp: bool = False):
    if omp not in _libs:
        L = C.CDLL(build(omp=omp))
        L.orc_validate.restype = C.c_int
        L.orc_lsqr.restype = C.c_int
        L.orc_lsqr_var.restype = C.c_int
        L.orc_threads.restype = C.c_int
        _libs[omp] = L
    return _libs[omp]


def omp_threads() -> int:
    """Threads the OpenMP timing build uses (OMP_NUM_THREADS or all cores)."""
    return int(lib(True).orc_threads())


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


class OracleSystem:
    """One system in caller form.  `values` is copied so precondition() can scale it."""

    def __init__(self, n_stars, n_dfa, n_instr, star_idx, att_start, instr_col, values, omp=False,
                 copy_values=True):
        self.omp = bool(omp)   # route every call through the OpenMP timing build
        self.star_idx = np.ascontiguousarray(star_idx, dtype=np.int32)
        self.att_start = np.ascontiguousarray(att_start, dtype=np.int32)
        self.instr_col = np.ascontiguousarray(instr_col, dtype=np.int32).reshape(-1, 6)
        self.values = (np.array(values, dtype=np.float64, order="C", copy=True) if copy_values
                       else np.ascontiguousarray(values, dtype=np.float64)).reshape(-1, 24)
        self.m = int(self.star_idx.shape[0])
        assert self.att_start.shape == (self.m,) and self.instr_col.shape == (self.m, 6)
        assert self.values.shape == (self.m, 24)
        self.n_stars, self.n_dfa, self.n_instr = int(n_stars), int(n_dfa), int(n_instr)
        self.n = 5 * self.n_stars + 3 * self.n_dfa + self.n_instr + 1
        self.dims = _Dims(self.m, self.n_stars, self.n_dfa, self.n_instr)
        self.p = None
        self.n_con, self.con_ptr, self.con_col, self.con_val = 0, None, None, None

    def _L(self):
        return lib(self.omp)

    def set_constraints(self, row_ptr, col, val):
        """n_con extra rows in CSR form appended below the observations.
        From now on m-vectors have m + n_con entries.  `val` is copied (precondition scales it)."""
        self.con_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
        self.con_col = np.ascontiguousarray(col, dtype=np.int32)
        self.con_val = np.array(val, dtype=np.float64, order="C", copy=True)
        self.n_con = int(self.con_ptr.shape[0]) - 1
        assert self.con_ptr[0] == 0 and self.con_ptr[-1] == self.con_col.shape[0] == self.con_val.shape[0]
        assert self.con_col.size == 0 or (self.con_col.min() >= 0 and self.con_col.max() < self.n)

    @property
    def m_total(self) -> int:
        return self.m + self.n_con

    def _con(self, on=True):
        if self.n_con and on:
            self._L().orc_set_constraints(C.c_int64(self.n_con), _p(self.con_ptr, C.c_int64),
                                      _p(self.con_col, C.c_int32), _p(self.con_val, C.c_double))
        else:
            self._L().orc_set_constraints(C.c_int64(0), None, None, None)

    def _idx(self):
        return (C.byref(self.dims), _p(self.star_idx, C.c_int32), _p(self.att_start, C.c_int32),
                _p(self.instr_col, C.c_int32))

    def validate(self) -> int:
        return int(self._L().orc_validate(*self._idx()))

    def expand_rows(self, row0=0, nrows=None):
        nrows = self.m - row0 if nrows is None else nrows
        cols = np.empty((nrows, 24), dtype=np.int64)
        vals = np.empty((nrows, 24), dtype=np.float64)
        self._L().orc_expand_rows(*self._idx(), _p(self.values, C.c_double), C.c_int64(row0),
                              C.c_int64(nrows), _p(cols, C.c_int64), _p(vals, C.c_double))
        return cols, vals

    def aprod1(self, x, y, want_scale=False):
        """y += A x (in place on a copy); returns y or (y, scale)."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.array(y, dtype=np.float64, copy=True)
        assert x.shape == (self.n,) and y.shape == (self.m_total,)
        sc = np.empty(self.m_total) if want_scale else None
        self._con()
        self._L().orc_aprod1(*self._idx(), _p(self.values, C.c_double), _p(x, C.c_double),
                         _p(y, C.c_double), _p(sc, C.c_double))
        self._con(False)
        return (y, sc) if want_scale else y

    def aprod2(self, y, x, want_scale=False):
        """x += A^T y (on a copy); returns x or (x, scale)."""
        y = np.ascontiguousarray(y, dtype=np.float64)
        x = np.array(x, dtype=np.float64, copy=True)
        assert x.shape == (self.n,) and y.shape == (self.m_total,)
        sc = np.empty(self.n) if want_scale else None
        self._con()
        self._L().orc_aprod2(*self._idx(), _p(self.values, C.c_double), _p(y, C.c_double),
                         _p(x, C.c_double), _p(sc, C.c_double))
        self._con(False)
        return (x, sc) if want_scale else x

    def colsumsq(self):
        q = np.empty(self.n)
        self._con()
        self._L().orc_colsumsq(*self._idx(), _p(self.values, C.c_double), _p(q, C.c_double))
        self._con(False)
        return q

    def precondition(self):
        """Scales self.values in place, keeps and returns p."""
        assert self.p is None, "already preconditioned"
        p = np.empty(self.n)
        self._con()
        self._L().orc_precondition(*self._idx(), _p(self.values, C.c_double), _p(p, C.c_double))
        self._con(False)
        self.p = p
        return p

    def lsqr(self, b, itnlim, atol=0.0, btol=0.0, conlim=0.0, force_itnlim=False,
             want_hist=False, want_se=False, damp=0.0) -> LsqrResult:
        """min ||A x - b||.  If preconditioned, iterates on A.diag(p), returns x = p (.) z."""
        b = np.ascontiguousarray(b, dtype=np.float64)
        assert b.shape == (self.m_total,)
        x = np.empty(self.n)
        res = _Result()
        hist = np.zeros((int(itnlim), 7)) if want_hist else None
        var = np.zeros(self.n) if want_se else None
        self._con()
        self._L().orc_set_damp(C.c_double(damp))
        rc = self._L().orc_lsqr_var(*self._idx(), _p(self.values, C.c_double), _p(b, C.c_double),
                                _p(x, C.c_double), C.c_int64(itnlim), C.c_double(atol),
                                C.c_double(btol), C.c_double(conlim),
                                C.c_int(1 if force_itnlim else 0), C.byref(res),
                                _p(hist, C.c_double), _p(var, C.c_double))
        self._con(False)
        self._L().orc_set_damp(C.c_double(0.0))
        assert rc == 0
        se = None
        if want_se:
            se = np.empty(self.n)
            self._L().orc_standard_errors(C.c_int64(self.m_total), C.c_int64(self.n), C.c_double(res.rnorm),
                                      _p(var, C.c_double), _p(self.p, C.c_double), _p(se, C.c_double))
        if self.p is not None:
            self._L().orc_unscale(C.c_int64(self.n), _p(self.p, C.c_double), _p(x, C.c_double))
        if hist is not None:
            hist = hist[:res.itn]
        return LsqrResult(x, res.istop, res.itn, res.istop_natural, res.itn_natural, res.rnorm,
                          res.arnorm, res.anorm, res.acond, res.xnorm, res.bnorm, hist, var, se)


def from_torch(cfg, star, att, instr, vals, omp=False) -> OracleSystem:
    """Build from the tensors of the shared input generator (host copies)."""
    return OracleSystem(cfg.n_stars, cfg.n_dfa, cfg.n_instr, star.cpu().numpy(), att.cpu().numpy(),
                        instr.cpu().numpy(), vals.cpu().numpy(), omp=omp)
