"""ctypes front end of oracle/cg_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this.  It shares nothing with the CUDA path.
See cg_oracle.c for the passages of PAPER.md each routine follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cg_oracle.c")
_LIB = os.path.join(_HERE, "libcg_oracle.so")
# -ffp-contract=off: no FMA contraction, so the oracle is one fixed function.
_CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-std=c99"]


def build(force: bool = False) -> str:
    """Compile cg_oracle.c with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", *_CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_SRC_OMP = os.path.join(_HERE, "cg_oracle_omp.c")
_LIB_OMP = os.path.join(_HERE, "libcg_oracle_omp.so")


def build_omp(force: bool = False) -> str:
    """Compile cg_oracle_omp.c (the all-cores baseline; not the parity reference)."""
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC_OMP):
        tmp = _LIB_OMP + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", *_CFLAGS, "-fopenmp", "-o", tmp, _SRC_OMP, "-lm"])
        os.replace(tmp, _LIB_OMP)
    return _LIB_OMP


_lib = None
_lib_omp = None
_c_i32p = ctypes.POINTER(ctypes.c_int32)
_c_f64p = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, f64 = ctypes.c_int64, ctypes.c_double
        csr = [i64, _c_i32p, _c_i32p, _c_f64p]
        for name in ("oracle_spmv", "oracle_spmv_ld", "oracle_absrow"):
            getattr(lib, name).argtypes = csr + [_c_f64p, _c_f64p]
            getattr(lib, name).restype = None
        for name in ("oracle_dot", "oracle_dot_ld"):
            getattr(lib, name).argtypes = [i64, _c_f64p, _c_f64p]
            getattr(lib, name).restype = f64
        lib.oracle_cg.argtypes = csr + [_c_f64p, _c_f64p, _c_f64p, f64, i64, _c_f64p,
                                        ctypes.POINTER(i64), _c_f64p, _c_f64p, _c_f64p,
                                        _c_f64p, _c_f64p, _c_f64p, i64]
        lib.oracle_cg.restype = ctypes.c_int
        _lib = lib
    return _lib


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_c_f64p)


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(_c_i32p)


def _csr(rowptr, colind, vals):
    rp, prp = _i32(rowptr)
    ci, pci = _i32(colind)
    va, pva = _f64(vals)
    n = len(rp) - 1
    return (rp, ci, va), (ctypes.c_int64(n), prp, pci, pva), n


def _spmv_like(fn, rowptr, colind, vals, x):
    keep, args, n = _csr(rowptr, colind, vals)
    xx, px = _f64(x)
    y = np.empty(n, dtype=np.float64)
    getattr(_load(), fn)(*args, px, y.ctypes.data_as(_c_f64p))
    return y


def spmv(rowptr, colind, vals, x):
    """y = A x ("DGEMV(sparse)"), sequential fp64."""
    return _spmv_like("oracle_spmv", rowptr, colind, vals, x)


def spmv_ld(rowptr, colind, vals, x):
    """Diagnostic: y = A x accumulated in long double."""
    return _spmv_like("oracle_spmv_ld", rowptr, colind, vals, x)


def absrow(rowptr, colind, vals, x):
    """Diagnostic: (|A||x|)_i, the denominator of the SpMV error metric."""
    return _spmv_like("oracle_absrow", rowptr, colind, vals, x)


def dot(a, b) -> float:
    aa, pa = _f64(a)
    bb, pb = _f64(b)
    assert aa.shape == bb.shape
    return float(_load().oracle_dot(ctypes.c_int64(aa.size), pa, pb))


def dot_ld(a, b) -> float:
    aa, pa = _f64(a)
    bb, pb = _f64(b)
    return float(_load().oracle_dot_ld(ctypes.c_int64(aa.size), pa, pb))


@dataclass
class CGResult:
    x: np.ndarray
    iters: int
    status: int            # 0 converged, 1 maxit, 2 breakdown
    resnorm: float
    hist: np.ndarray       # ||r_j||_2, j = 0..iters
    alpha: np.ndarray
    beta: np.ndarray
    P: Optional[np.ndarray] = None
    R: Optional[np.ndarray] = None
    X: Optional[np.ndarray] = None


def cg(rowptr, colind, vals, b, x0=None, rtol=1e-10, maxit=None, dinv=None,
       keep: int = 0) -> CGResult:
    """Unpreconditioned CG; Jacobi PCG when ``dinv`` is given.

    ``keep`` > 0 also returns the first ``keep`` search directions p_j, residuals
    r_j and iterates x_j (rows of P, R, X) for the orthogonality / A-norm pins.
    """
    keepalive, args, n = _csr(rowptr, colind, vals)
    if maxit is None:
        maxit = n
    bb, pb = _f64(b)
    x = np.zeros(n, dtype=np.float64) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    hist = np.zeros(maxit + 1, dtype=np.float64)
    alpha = np.zeros(max(maxit, 1), dtype=np.float64)
    beta = np.zeros(max(maxit, 1), dtype=np.float64)
    iters = ctypes.c_int64(0)
    res = ctypes.c_double(0.0)
    null = ctypes.cast(None, _c_f64p)
    if dinv is not None:
        dd, pd = _f64(dinv)
    else:
        pd = null
    P = R = X = None
    pP = pR = pX = null
    if keep > 0:
        P = np.zeros((keep, n)); R = np.zeros((keep, n)); X = np.zeros((keep, n))
        pP, pR, pX = (a.ctypes.data_as(_c_f64p) for a in (P, R, X))
    st = _load().oracle_cg(*args, pd, pb, x.ctypes.data_as(_c_f64p), ctypes.c_double(rtol),
                           ctypes.c_int64(maxit), hist.ctypes.data_as(_c_f64p),
                           ctypes.byref(iters), ctypes.byref(res),
                           alpha.ctypes.data_as(_c_f64p), beta.ctypes.data_as(_c_f64p),
                           pP, pR, pX, ctypes.c_int64(keep))
    if st < 0:
        raise ValueError("oracle_cg: invalid argument")
    k = int(iters.value)
    kk = min(keep, k + 1)
    return CGResult(x=x, iters=k, status=int(st), resnorm=float(res.value),
                    hist=hist[:k + 1].copy(), alpha=alpha[:k].copy(), beta=beta[:k].copy(),
                    P=None if P is None else P[:kk], R=None if R is None else R[:kk],
                    X=None if X is None else X[:kk])


def omp_threads() -> int:
    """Threads the OpenMP baseline uses (OMP_NUM_THREADS or all cores)."""
    global _lib_omp
    if _lib_omp is None:
        _lib_omp = ctypes.CDLL(build_omp())
    _lib_omp.oracle_omp_threads.restype = ctypes.c_int
    return int(_lib_omp.oracle_omp_threads())


def omp_set_threads(t: int) -> None:
    global _lib_omp
    if _lib_omp is None:
        _lib_omp = ctypes.CDLL(build_omp())
    _lib_omp.oracle_omp_set_threads.argtypes = [ctypes.c_int]
    _lib_omp.oracle_omp_set_threads(int(t))


def cg_omp(rowptr, colind, vals, b, x0=None, rtol=1e-10, maxit=None) -> CGResult:
    """The same CG with row-parallel OpenMP loops on all host cores (cg_oracle_omp.c): the
    all-cores CPU baseline of SURVEY.md 8(d), itself checked against `cg` in the tests."""
    global _lib_omp
    if _lib_omp is None:
        _lib_omp = ctypes.CDLL(build_omp())
    keepalive, args, n = _csr(rowptr, colind, vals)
    if maxit is None:
        maxit = n
    bb, pb = _f64(b)
    x = np.zeros(n, dtype=np.float64) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    hist = np.zeros(maxit + 1, dtype=np.float64)
    iters = ctypes.c_int64(0)
    res = ctypes.c_double(0.0)
    fn = _lib_omp.oracle_cg_omp
    fn.argtypes = [ctypes.c_int64, _c_i32p, _c_i32p, _c_f64p, _c_f64p, _c_f64p, ctypes.c_double,
                   ctypes.c_int64, _c_f64p, ctypes.POINTER(ctypes.c_int64), _c_f64p]
    fn.restype = ctypes.c_int
    st = fn(*args, pb, x.ctypes.data_as(_c_f64p), ctypes.c_double(rtol), ctypes.c_int64(maxit),
            hist.ctypes.data_as(_c_f64p), ctypes.byref(iters), ctypes.byref(res))
    if st < 0:
        raise ValueError("oracle_cg_omp: invalid argument")
    k = int(iters.value)
    return CGResult(x=x, iters=k, status=int(st), resnorm=float(res.value), hist=hist[:k + 1].copy(),
                    alpha=np.zeros(0), beta=np.zeros(0))
