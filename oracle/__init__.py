"""CPU oracle for the SP2 hot path — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes wrapper over ``oracle/sp2_oracle.c`` (plain C, compiled here with gcc).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.
It imports nothing from ``paper_2401_13772_b200`` and the CUDA path never imports it.

Every function cites the passage of /root/reference/PAPER.md (``P:<line>``) it follows; see the header of
``sp2_oracle.c`` for the algorithm, the readings of the paper, and the list of pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sp2_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
LOG_LEN = 128

_f64p = ctypes.POINTER(ctypes.c_double)
_i32p = ctypes.POINTER(ctypes.c_int32)
_i64p = ctypes.POINTER(ctypes.c_int64)


class OracleStats(ctypes.Structure):
    _fields_ = [
        ("status", ctypes.c_int32),
        ("n_products", ctypes.c_int32),
        ("m_star", ctypes.c_int32),
        ("overflow_row", ctypes.c_int32),
        ("emin", ctypes.c_double),
        ("emax", ctypes.c_double),
        ("branch", ctypes.c_uint8 * LOG_LEN),
        ("trace", ctypes.c_double * LOG_LEN),
        ("idem", ctypes.c_double * LOG_LEN),
        ("max_row_nnz", ctypes.c_int32 * LOG_LEN),
    ]


def build(force: bool = False) -> str:
    """Compile sp2_oracle.c -> liboracle.so (gcc, -O3, OpenMP over output rows, no FP contraction)."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        cmd = ["gcc", "-O3", "-mavx2", "-mfma", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", _LIB,
               _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_trace_dense.restype = ctypes.c_double
        lib.oracle_trace_ellpack.restype = ctypes.c_double
        lib.oracle_trace_ellblock.restype = ctypes.c_double
        for name in ("oracle_rescale_ellpack", "oracle_x2_ellpack", "oracle_update_ellpack", "oracle_rescale_ellblock",
                     "oracle_x2_ellblock", "oracle_update_ellblock"):
            getattr(lib, name).restype = ctypes.c_int64
        lib.oracle_x2_dense.restype = None
        lib.oracle_x2_dense_sampled.restype = None
        lib.oracle_rescale_dense.restype = None
        _lib = lib
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _c32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _stats_dict(st: OracleStats) -> dict:
    n = max(int(st.n_products), 0)
    m = max(int(st.m_star), 0)
    return {
        "status": int(st.status),
        "n_products": int(st.n_products),
        "m_star": int(st.m_star),
        "overflow_row": int(st.overflow_row),
        "emin": float(st.emin),
        "emax": float(st.emax),
        "branch": "".join(str(int(b)) for b in st.branch[:m]),
        "trace": np.array(st.trace[:n]),
        "idem": np.array(st.idem[:n]),
        "max_row_nnz": np.array(st.max_row_nnz[:n]),
    }


def omp_threads() -> int:
    return int(_L().oracle_omp_threads())


# ------------------------------------------------ dense -------------------------------------------------
def gershgorin_dense(H):
    """(e_min, e_max) by Gershgorin circles, P:452 / SURVEY 8(c) line 1."""
    H = _c64(H)
    lo, hi = ctypes.c_double(), ctypes.c_double()
    rc = _L().oracle_gershgorin_dense(_p(H, _f64p), ctypes.c_int64(H.shape[0]), ctypes.c_int64(H.shape[1]),
                                      ctypes.byref(lo), ctypes.byref(hi))
    assert rc == 0
    return lo.value, hi.value


def trace_dense(A):
    """tr A, Listing 2 P:201."""
    A = _c64(A)
    return float(_L().oracle_trace_dense(_p(A, _f64p), ctypes.c_int64(A.shape[0]), ctypes.c_int64(A.shape[1])))


def rescale_dense(H, emin, emax):
    """X_0 of Eq. 5."""
    H = _c64(H)
    X = np.empty_like(H)
    _L().oracle_rescale_dense(_p(H, _f64p), ctypes.c_int64(H.shape[0]), ctypes.c_int64(H.shape[1]),
                              ctypes.c_double(emin), ctypes.c_double(emax), _p(X, _f64p))
    return X


def x2_dense(X):
    """P = X X by the definition (triple loop)."""
    X = _c64(X)
    P = np.empty_like(X)
    _L().oracle_x2_dense(_p(X, _f64p), ctypes.c_int64(X.shape[0]), _p(P, _f64p))
    return P


def x2_dense_sampled(X, rows, cols):
    """Selected entries (X X)_ij, one compensated dot product each."""
    X = _c64(X)
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    cols = np.ascontiguousarray(cols, dtype=np.int64)
    out = np.empty(rows.size, dtype=np.float64)
    _L().oracle_x2_dense_sampled(_p(X, _f64p), ctypes.c_int64(X.shape[0]), ctypes.c_int64(X.shape[1]),
                                 ctypes.c_int64(rows.size), _p(rows, _i64p), _p(cols, _i64p), _p(out, _f64p))
    return out


def sp2_dense(H, n_occ, tol, max_products=100, bounds=None):
    """Dense SP2 (Eq. 5-7, Listing 2; SURVEY 8(c) lines 1-13).  bounds = (e_min, e_max) replaces the Gershgorin bounds
    (oracle/bounds.py).  Returns (D, stats dict)."""
    H = _c64(H)
    N = H.shape[0]
    D = np.zeros((N, N), dtype=np.float64)
    st = OracleStats()
    b = None if bounds is None else (ctypes.c_double * 2)(float(bounds[0]), float(bounds[1]))
    _L().oracle_sp2_dense_bounds(_p(H, _f64p), ctypes.c_int64(N), ctypes.c_int64(H.shape[1]), ctypes.c_int32(n_occ),
                                 ctypes.c_double(tol), ctypes.c_int32(max_products), b, _p(D, _f64p), ctypes.byref(st))
    return D, _stats_dict(st)


# ----------------------------------------------- ELLPACK-R ----------------------------------------------
def gershgorin_ellpack(value, index, nnz):
    value, index, nnz = _c64(value), _c32(index), _c32(nnz)
    N, M = value.shape
    lo, hi = ctypes.c_double(), ctypes.c_double()
    rc = _L().oracle_gershgorin_ellpack(ctypes.c_int64(N), ctypes.c_int32(M), _p(value, _f64p), _p(index, _i32p),
                                        _p(nnz, _i32p), ctypes.byref(lo), ctypes.byref(hi))
    assert rc == 0
    return lo.value, hi.value


def trace_ellpack(value, index, nnz):
    value, index, nnz = _c64(value), _c32(index), _c32(nnz)
    N, M = value.shape
    return float(_L().oracle_trace_ellpack(ctypes.c_int64(N), ctypes.c_int32(M), _p(value, _f64p), _p(index, _i32p),
                                           _p(nnz, _i32p)))


def rescale_ellpack(value, index, nnz, emin, emax):
    """Eq. 5 on ELLPACK-R; returns (value, index, nnz, overflow_row)."""
    value, index, nnz = _c64(value), _c32(index), _c32(nnz)
    N, M = value.shape
    xv, xi, xn = np.zeros_like(value), np.zeros_like(index), np.zeros_like(nnz)
    bad = _L().oracle_rescale_ellpack(ctypes.c_int64(N), ctypes.c_int32(M), _p(value, _f64p), _p(index, _i32p),
                                      _p(nnz, _i32p), ctypes.c_double(emin), ctypes.c_double(emax),
                                      _p(xv, _f64p), _p(xi, _i32p), _p(xn, _i32p))
    return xv, xi, xn, int(bad)


def x2_ellpack(value, index, nnz, tau):
    """P = thr_tau(X X), Gustavson row merge; returns (value, index, nnz, overflow_row, max_nnz)."""
    value, index, nnz = _c64(value), _c32(index), _c32(nnz)
    N, M = value.shape
    pv, pi, pn = np.zeros_like(value), np.zeros_like(index), np.zeros_like(nnz)
    mx = ctypes.c_int32()
    bad = _L().oracle_x2_ellpack(ctypes.c_int64(N), ctypes.c_int32(M), _p(value, _f64p), _p(index, _i32p),
                                 _p(nnz, _i32p), ctypes.c_double(tau), _p(pv, _f64p), _p(pi, _i32p), _p(pn, _i32p),
                                 ctypes.byref(mx))
    return pv, pi, pn, int(bad), int(mx.value)


def update_ellpack(X, P, tau):
    """X' = thr_tau(2X - P) on the union pattern; X, P are (value, index, nnz) triples."""
    xv, xi, xn = _c64(X[0]), _c32(X[1]), _c32(X[2])
    pv, pi, pn = _c64(P[0]), _c32(P[1]), _c32(P[2])
    N, M = xv.shape
    ov, oi, on = np.zeros_like(xv), np.zeros_like(xi), np.zeros_like(xn)
    mx = ctypes.c_int32()
    bad = _L().oracle_update_ellpack(ctypes.c_int64(N), ctypes.c_int32(M), _p(xv, _f64p), _p(xi, _i32p), _p(xn, _i32p),
                                     _p(pv, _f64p), _p(pi, _i32p), _p(pn, _i32p), ctypes.c_double(tau),
                                     _p(ov, _f64p), _p(oi, _i32p), _p(on, _i32p), ctypes.byref(mx))
    return ov, oi, on, int(bad), int(mx.value)


def sp2_ellpack(value, index, nnz, n_occ, tol, tau, max_products=100, bounds=None):
    """Sparse thresholded SP2 (SURVEY 8(c) sparse oracle); bounds as in sp2_dense.
    Returns ((value, index, nnz) of D, stats dict)."""
    value, index, nnz = _c64(value), _c32(index), _c32(nnz)
    N, M = value.shape
    dv, di, dn = np.zeros_like(value), np.zeros_like(index), np.zeros_like(nnz)
    st = OracleStats()
    b = None if bounds is None else (ctypes.c_double * 2)(float(bounds[0]), float(bounds[1]))
    _L().oracle_sp2_ellpack_bounds(ctypes.c_int64(N), ctypes.c_int32(M), _p(value, _f64p), _p(index, _i32p),
                                   _p(nnz, _i32p), ctypes.c_int32(n_occ), ctypes.c_double(tol), ctypes.c_double(tau),
                                   ctypes.c_int32(max_products), b, _p(dv, _f64p), _p(di, _i32p), _p(dn, _i32p),
                                   ctypes.byref(st))
    return (dv, di, dn), _stats_dict(st)


# ----------------------------------------------- ELLBLOCK -----------------------------------------------
# value[NB, MB, bs, bs] float64, index[NB, MB] int32 (block columns), nnz[NB] int32 (readings E1-E4 in sp2_oracle.c)
def _blk(value, index, nnz):
    value, index, nnz = _c64(value), _c32(index), _c32(nnz)
    NB, MB, bs, bs2 = value.shape
    assert bs == bs2 and index.shape == (NB, MB) and nnz.shape == (NB,)
    return value, index, nnz, NB, MB, bs


def gershgorin_ellblock(value, index, nnz):
    value, index, nnz, NB, MB, bs = _blk(value, index, nnz)
    lo, hi = ctypes.c_double(), ctypes.c_double()
    rc = _L().oracle_gershgorin_ellblock(ctypes.c_int64(NB), ctypes.c_int32(MB), ctypes.c_int32(bs), _p(value, _f64p),
                                         _p(index, _i32p), _p(nnz, _i32p), ctypes.byref(lo), ctypes.byref(hi))
    assert rc == 0
    return lo.value, hi.value


def trace_ellblock(value, index, nnz):
    value, index, nnz, NB, MB, bs = _blk(value, index, nnz)
    return float(_L().oracle_trace_ellblock(ctypes.c_int64(NB), ctypes.c_int32(MB), ctypes.c_int32(bs), _p(value, _f64p),
                                            _p(index, _i32p), _p(nnz, _i32p)))


def rescale_ellblock(value, index, nnz, emin, emax):
    """Eq. 5 on ELLBLOCK; returns (value, index, nnz, overflow block row)."""
    value, index, nnz, NB, MB, bs = _blk(value, index, nnz)
    xv, xi, xn = np.zeros_like(value), np.zeros_like(index), np.zeros_like(nnz)
    bad = _L().oracle_rescale_ellblock(ctypes.c_int64(NB), ctypes.c_int32(MB), ctypes.c_int32(bs), _p(value, _f64p),
                                       _p(index, _i32p), _p(nnz, _i32p), ctypes.c_double(emin), ctypes.c_double(emax),
                                       _p(xv, _f64p), _p(xi, _i32p), _p(xn, _i32p))
    return xv, xi, xn, int(bad)


def x2_ellblock(value, index, nnz, tau):
    """P = thr_tau(X X) on blocks (a block is kept iff its Frobenius norm >= tau or it is diagonal).
    Returns (value, index, nnz, overflow block row, max blocks per block row)."""
    value, index, nnz, NB, MB, bs = _blk(value, index, nnz)
    pv, pi, pn = np.zeros_like(value), np.zeros_like(index), np.zeros_like(nnz)
    mx = ctypes.c_int32()
    bad = _L().oracle_x2_ellblock(ctypes.c_int64(NB), ctypes.c_int32(MB), ctypes.c_int32(bs), _p(value, _f64p),
                                  _p(index, _i32p), _p(nnz, _i32p), ctypes.c_double(tau), _p(pv, _f64p), _p(pi, _i32p),
                                  _p(pn, _i32p), ctypes.byref(mx))
    return pv, pi, pn, int(bad), int(mx.value)


def update_ellblock(X, P, tau):
    """X' = thr_tau(2X - P) on the union of the block patterns."""
    xv, xi, xn, NB, MB, bs = _blk(*X)
    pv, pi, pn, _, _, _ = _blk(*P)
    ov, oi, on = np.zeros_like(xv), np.zeros_like(xi), np.zeros_like(xn)
    mx = ctypes.c_int32()
    bad = _L().oracle_update_ellblock(ctypes.c_int64(NB), ctypes.c_int32(MB), ctypes.c_int32(bs), _p(xv, _f64p),
                                      _p(xi, _i32p), _p(xn, _i32p), _p(pv, _f64p), _p(pi, _i32p), _p(pn, _i32p),
                                      ctypes.c_double(tau), _p(ov, _f64p), _p(oi, _i32p), _p(on, _i32p), ctypes.byref(mx))
    return ov, oi, on, int(bad), int(mx.value)


def sp2_ellblock(value, index, nnz, n_occ, tol, tau, max_products=100):
    """Thresholded SP2 on ELLBLOCK.  Returns ((value, index, nnz) of D, stats dict)."""
    value, index, nnz, NB, MB, bs = _blk(value, index, nnz)
    dv, di, dn = np.zeros_like(value), np.zeros_like(index), np.zeros_like(nnz)
    st = OracleStats()
    _L().oracle_sp2_ellblock(ctypes.c_int64(NB), ctypes.c_int32(MB), ctypes.c_int32(bs), _p(value, _f64p), _p(index, _i32p),
                             _p(nnz, _i32p), ctypes.c_int32(n_occ), ctypes.c_double(tol), ctypes.c_double(tau),
                             ctypes.c_int32(max_products), _p(dv, _f64p), _p(di, _i32p), _p(dn, _i32p), ctypes.byref(st))
    return (dv, di, dn), _stats_dict(st)
