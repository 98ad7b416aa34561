"""oracle/ -- TEST INFRASTRUCTURE ONLY (see oracle_spmv.c header).

ctypes binding over the plain-C CPU oracle.  Only tests/, the smoke check in
__graft_entry__ and bench.py's cpu_baseline / --impl reference leg may import
this package.  It imports nothing from paper_1309_1894_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_spmv.c")
_SRC_CG = os.path.join(_HERE, "oracle_cg.c")
_SRC_JAC = os.path.join(_HERE, "oracle_jacobi.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle_spmv.c -> liboracle.so (-O2, no FMA contraction, OpenMP)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_CG), os.path.getmtime(_SRC_JAC))):
        return _LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-std=c11", "-Wall", "-o", _LIB, _SRC, _SRC_CG, _SRC_JAC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB)
    i64, dbl, vp = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
    for name in ("oracle_spmv", "oracle_spmv_omp"):
        f = getattr(lib, name)
        f.argtypes = [i64, vp, vp, vp, dbl, vp, dbl, vp, vp]
    lib.oracle_spmv.restype = None
    lib.oracle_spmv_omp.restype = ctypes.c_int
    lib.oracle_spmv_ext.argtypes = [i64, vp, vp, vp, dbl, vp, dbl, vp]
    lib.oracle_spmv_ext.restype = None
    lib.oracle_long_double_bits.restype = ctypes.c_int
    lib.oracle_accept.argtypes = [i64, vp, vp, vp, dbl, vp, vp, vp]
    lib.oracle_accept.restype = None
    lib.oracle_cg.argtypes = [i64, vp, vp, vp, vp, vp, dbl, i64, vp, vp]
    lib.oracle_cg.restype = i64
    lib.oracle_jacobi.argtypes = [i64, vp, vp, vp, vp, vp, dbl, dbl, i64, vp, vp]
    lib.oracle_jacobi.restype = i64
    _lib = lib
    return lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _csr(row_ptr, col_idx, val):
    rp = np.ascontiguousarray(row_ptr, dtype=np.int32)
    ci = np.ascontiguousarray(col_idx, dtype=np.int32)
    va = np.ascontiguousarray(val, dtype=np.float64)
    assert rp.ndim == 1 and rp.size >= 1 and ci.size == va.size == int(rp[-1])
    return rp, ci, va


def spmv(row_ptr, col_idx, val, alpha, x, beta, y0=None, *, parallel=False):
    """Return (y, scale): y = alpha*A*x + beta*y0 and the per-row tolerance
    denominator.  y0 may be None only when beta == 0 (y is then not read)."""
    lib = _load()
    rp, ci, va = _csr(row_ptr, col_idx, val)
    rows = rp.size - 1
    x = np.ascontiguousarray(x, dtype=np.float64)
    if y0 is None:
        assert beta == 0.0, "y0 required when beta != 0"
        y = np.full(rows, np.nan)  # must never be read (reading A1)
    else:
        y = np.array(y0, dtype=np.float64, copy=True)
        assert y.size == rows
    scale = np.empty(rows, dtype=np.float64)
    fn = lib.oracle_spmv_omp if parallel else lib.oracle_spmv
    fn(rows, _p(rp), _p(ci), _p(va), float(alpha), _p(x), float(beta), _p(y), _p(scale))
    return y, scale


def spmv_inplace(rp, ci, va, alpha, x, beta, y, scale, *, parallel=False):
    """No-copy form for timing: arrays must already be contiguous and typed.
    Returns the thread count used."""
    lib = _load()
    rows = rp.size - 1
    if parallel:
        return lib.oracle_spmv_omp(rows, _p(rp), _p(ci), _p(va), float(alpha), _p(x),
                                   float(beta), _p(y), _p(scale) if scale is not None else None)
    lib.oracle_spmv(rows, _p(rp), _p(ci), _p(va), float(alpha), _p(x), float(beta),
                    _p(y), _p(scale) if scale is not None else None)
    return 1


def spmv_ext(row_ptr, col_idx, val, alpha, x, beta, y0=None):
    """Extended-precision accumulation (pin P9); not the oracle."""
    lib = _load()
    rp, ci, va = _csr(row_ptr, col_idx, val)
    rows = rp.size - 1
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.zeros(rows) if y0 is None else np.array(y0, dtype=np.float64, copy=True)
    lib.oracle_spmv_ext(rows, _p(rp), _p(ci), _p(va), float(alpha), _p(x), float(beta), _p(y))
    return y


def long_double_bits() -> int:
    return _load().oracle_long_double_bits()


def accept(y_test, y_ref, scale, tol=1e-12):
    """Acceptance rule: returns (ok, max_ratio, first_fail, n_fail)."""
    lib = _load()
    yt = np.ascontiguousarray(y_test, dtype=np.float64)
    yr = np.ascontiguousarray(y_ref, dtype=np.float64)
    sc = np.ascontiguousarray(scale, dtype=np.float64)
    assert yt.size == yr.size == sc.size
    mr = ctypes.c_double(0.0)
    ff = ctypes.c_int64(-1)
    nf = ctypes.c_int64(0)
    lib.oracle_accept(yt.size, _p(yt), _p(yr), _p(sc), float(tol),
                      ctypes.byref(mr), ctypes.byref(ff), ctypes.byref(nf))
    return nf.value == 0, mr.value, ff.value, nf.value


def cg(row_ptr, col_idx, val, b, x0=None, tol=1e-10, max_iters=1000):
    """Plain conjugate gradients (oracle_cg.c).  Returns (x, iters, rel_res, res_hist)."""
    lib = _load()
    rp, ci, va = _csr(row_ptr, col_idx, val)
    rows = rp.size - 1
    b = np.ascontiguousarray(b, dtype=np.float64)
    x = np.zeros(rows) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    hist = np.full(int(max_iters) + 1, np.nan)
    rel = ctypes.c_double(0.0)
    k = lib.oracle_cg(rows, _p(rp), _p(ci), _p(va), _p(b), _p(x), float(tol), int(max_iters),
                      ctypes.byref(rel), _p(hist))
    return x, int(k), rel.value, hist[:int(k) + 1]


def jacobi(row_ptr, col_idx, val, b, x0=None, omega=1.0, tol=1e-10, max_iters=1000):
    """Weighted Jacobi (oracle_jacobi.c).  Returns (x, iters, rel_res, res_hist); iters == -1: zero diagonal."""
    lib = _load()
    rp, ci, va = _csr(row_ptr, col_idx, val)
    rows = rp.size - 1
    b = np.ascontiguousarray(b, dtype=np.float64)
    x = np.zeros(rows) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    hist = np.full(int(max_iters) + 1, np.nan)
    rel = ctypes.c_double(0.0)
    k = lib.oracle_jacobi(rows, _p(rp), _p(ci), _p(va), _p(b), _p(x), float(omega), float(tol), int(max_iters),
                          ctypes.byref(rel), _p(hist))
    return x, int(k), rel.value, hist[:max(int(k), 0) + 1]
