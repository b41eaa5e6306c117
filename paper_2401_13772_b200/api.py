"""Thin ctypes binding of libbmlsp2.so (include/bml_sp2.h, include/bml_chebyshev.h, include/bml_graph.h) — argument marshalling only.

Every function has the name of the C entry point it calls and takes torch CUDA tensors for device memory; all
arithmetic of the method runs in the library's sm_100a kernels.  There is no CPU fallback: if the library is missing
or a tensor is not on a CUDA device this module raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass, field

import numpy as np
import torch

from . import build as _build

LOG_LEN = 128
ELL_MAX_M = 1024
ELL_ACC_SLOTS = 4096
BML_DENSE, BML_ELLPACK = 0, 1
FLAG_CHECK_SYMMETRY = 1


def FLAG_LANCZOS_BOUNDS(steps: int) -> int:
    """BML_SP2_FLAG_LANCZOS_BOUNDS(K): tighter spectral bounds from K Lanczos steps (8..64) instead of Gershgorin alone."""
    return (int(steps) & 0xFF) << 8

EXPORTS = [
    "bml_version", "bml_status_string", "bml_gershgorin_workspace_bytes", "bml_gershgorin", "bml_trace",
    "bml_sp2_workspace_bytes", "bml_sp2_dense", "bml_sp2_ellpack", "bml_x2_dense_workspace_bytes", "bml_x2_dense",
    "bml_x2_ellpack_workspace_bytes", "bml_x2_ellpack", "bml_sp2_read_stats", "bml_sp2_release_cached",
    "bml_lanczos_bounds_workspace_bytes", "bml_lanczos_bounds",
    # include/bml_sp2_testing.h (test / measurement hooks, not the product interface)
    "bml_probe_fp64_tensor_peak", "bml_dense_work_item", "bml_dense_mixed_tile_count", "bml_dense_mixed_tile_of_cta",
    # include/bml_chebyshev.h
    "bml_chebyshev_workspace_bytes", "bml_chebyshev_dense", "bml_symm_ab_workspace_bytes", "bml_symm_ab_dense",
    "bml_cheb_schedule", "bml_symm_work_item",
    # include/bml_graph.h
    "bml_graph_workspace_bytes", "bml_graph_chebyshev_ellpack", "bml_graph_core_halo", "bml_matrix2submatrix_ellpack",
    "bml_submatrix2matrix_ellpack", "bml_graph_sp2_workspace_bytes", "bml_graph_sp2_ellpack",
    "bml_dense_batch_work_item",
    # include/bml_ellblock.h
    "bml_gershgorin_ellblock_workspace_bytes", "bml_gershgorin_ellblock", "bml_trace_ellblock",
    "bml_sp2_ellblock_workspace_bytes", "bml_sp2_ellblock", "bml_x2_ellblock_workspace_bytes", "bml_x2_ellblock",
    # include/bml_no_alloc.h
    "bml_gershgorin_static", "bml_no_alloc_status_string",
]
GERSHGORIN_STATIC_MAX_N = 65536
GRAPH_MAX_PARTS = 256
CHEB_MAX_K, CHEB_MAX_M, CHEB_MAX_TERMS, SYMM_MAX_JOBS = 32, 32, 1024, 16


class bml_matrix_t(ctypes.Structure):
    _fields_ = [
        ("type", ctypes.c_int32),
        ("M", ctypes.c_int32),
        ("N", ctypes.c_int64),
        ("ld", ctypes.c_int64),
        ("value", ctypes.c_void_p),
        ("index", ctypes.c_void_p),
        ("nnz", ctypes.c_void_p),
    ]


class bml_sp2_params_t(ctypes.Structure):
    _fields_ = [
        ("n_occ", ctypes.c_int32),
        ("max_products", ctypes.c_int32),
        ("idem_tol", ctypes.c_double),
        ("drop_tol", ctypes.c_double),
        ("precision", ctypes.c_int32),
        ("flags", ctypes.c_uint32),
    ]


class bml_sp2_stats_t(ctypes.Structure):
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


class bml_cheb_params_t(ctypes.Structure):
    _fields_ = [
        ("mu", ctypes.c_double),
        ("beta", ctypes.c_double),
        ("k", ctypes.c_int32),
        ("m", ctypes.c_int32),
        ("flags", ctypes.c_uint32),
        ("pad", ctypes.c_uint32),
    ]


class bml_cheb_stats_t(ctypes.Structure):
    _fields_ = [
        ("status", ctypes.c_int32),
        ("n_products", ctypes.c_int32),
        ("n_launches", ctypes.c_int32),
        ("L", ctypes.c_int32),
        ("emin", ctypes.c_double),
        ("emax", ctypes.c_double),
        ("trace", ctypes.c_double),
        ("c", ctypes.c_double * CHEB_MAX_TERMS),
        ("d", ctypes.c_double * CHEB_MAX_TERMS),
    ]


class bml_graph_params_t(ctypes.Structure):
    _fields_ = [
        ("mu", ctypes.c_double),
        ("beta", ctypes.c_double),
        ("graph_tol", ctypes.c_double),
        ("drop_tol", ctypes.c_double),
        ("k", ctypes.c_int32),
        ("m", ctypes.c_int32),
        ("n_parts", ctypes.c_int32),
        ("part_capacity", ctypes.c_int32),
    ]


class bml_graph_stats_t(ctypes.Structure):
    _fields_ = [
        ("status", ctypes.c_int32),
        ("n_parts", ctypes.c_int32),
        ("overflow_row", ctypes.c_int32),
        ("max_part_size", ctypes.c_int32),
        ("n_products", ctypes.c_int32),
        ("pad", ctypes.c_int32),
        ("part_size", ctypes.c_int32 * GRAPH_MAX_PARTS),
        ("core_size", ctypes.c_int32 * GRAPH_MAX_PARTS),
    ]


class bml_ellblock_t(ctypes.Structure):
    _fields_ = [
        ("bs", ctypes.c_int32),
        ("MB", ctypes.c_int32),
        ("NB", ctypes.c_int64),
        ("value", ctypes.c_void_p),
        ("index", ctypes.c_void_p),
        ("nnz", ctypes.c_void_p),
    ]


class bml_graph_sp2_params_t(ctypes.Structure):
    _fields_ = [
        ("graph_tol", ctypes.c_double),
        ("drop_tol", ctypes.c_double),
        ("idem_tol", ctypes.c_double),
        ("n_occ", ctypes.c_int32),
        ("max_products", ctypes.c_int32),
        ("n_parts", ctypes.c_int32),
        ("part_capacity", ctypes.c_int32),
    ]


class bml_graph_sp2_stats_t(ctypes.Structure):
    _fields_ = [
        ("sp2", bml_sp2_stats_t),
        ("status", ctypes.c_int32),
        ("n_parts", ctypes.c_int32),
        ("overflow_row", ctypes.c_int32),
        ("max_part_size", ctypes.c_int32),
        ("part_size", ctypes.c_int32 * GRAPH_MAX_PARTS),
        ("core_size", ctypes.c_int32 * GRAPH_MAX_PARTS),
    ]


_lib = None


def lib_path() -> str:
    return _build.LIB_PATH


def load(build_if_missing: bool = True):
    """dlopen libbmlsp2.so (building it with nvcc first if it is absent or stale) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build() if build_if_missing else _build.LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2401_13772_b200.build` (there is no CPU fallback)")
    L = ctypes.CDLL(path)
    vp, sz, i32, i64, dbl = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    MP, PP, SP = ctypes.POINTER(bml_matrix_t), ctypes.POINTER(bml_sp2_params_t), ctypes.POINTER(bml_sp2_stats_t)
    L.bml_version.restype = ctypes.c_char_p
    L.bml_status_string.restype = ctypes.c_char_p
    L.bml_status_string.argtypes = [ctypes.c_int]
    L.bml_gershgorin_workspace_bytes.restype = sz
    L.bml_gershgorin_workspace_bytes.argtypes = [i64]
    L.bml_gershgorin.restype = ctypes.c_int
    L.bml_gershgorin.argtypes = [MP, vp, vp, sz, vp]
    L.bml_trace.restype = ctypes.c_int
    L.bml_trace.argtypes = [MP, vp, vp]
    L.bml_gershgorin_static.restype = ctypes.c_int
    L.bml_gershgorin_static.argtypes = [MP, vp, vp]
    L.bml_no_alloc_status_string.restype = ctypes.c_char_p
    L.bml_no_alloc_status_string.argtypes = [ctypes.c_int]
    L.bml_lanczos_bounds_workspace_bytes.restype = sz
    L.bml_lanczos_bounds_workspace_bytes.argtypes = [i64]
    L.bml_lanczos_bounds.restype = ctypes.c_int
    L.bml_lanczos_bounds.argtypes = [MP, i32, ctypes.c_uint64, vp, vp, sz, vp]
    L.bml_sp2_workspace_bytes.restype = sz
    L.bml_sp2_workspace_bytes.argtypes = [MP, PP]
    for name in ("bml_sp2_dense", "bml_sp2_ellpack"):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [MP, PP, MP, vp, sz, SP, vp]
    L.bml_sp2_read_stats.restype = ctypes.c_int
    L.bml_sp2_read_stats.argtypes = [vp, SP, vp]
    L.bml_sp2_release_cached.restype = None
    L.bml_sp2_release_cached.argtypes = []
    L.bml_x2_dense_workspace_bytes.restype = sz
    L.bml_x2_dense_workspace_bytes.argtypes = [i64, i32]
    L.bml_x2_dense.restype = ctypes.c_int
    L.bml_x2_dense.argtypes = [MP, MP, i32, i32, vp, vp, sz, vp]
    L.bml_x2_ellpack_workspace_bytes.restype = sz
    L.bml_x2_ellpack_workspace_bytes.argtypes = [i64, ctypes.c_int32]
    L.bml_x2_ellpack.restype = ctypes.c_int
    L.bml_x2_ellpack.argtypes = [MP, MP, i32, dbl, vp, vp, vp, sz, vp]
    L.bml_probe_fp64_tensor_peak.restype = ctypes.c_int
    L.bml_probe_fp64_tensor_peak.argtypes = [i32, ctypes.POINTER(dbl), ctypes.POINTER(dbl), vp]
    L.bml_dense_work_item.restype = ctypes.c_int
    L.bml_dense_work_item.argtypes = [i64, i32, i32, i32, ctypes.POINTER(ctypes.c_int32)]
    L.bml_dense_mixed_tile_count.restype = ctypes.c_int
    L.bml_dense_mixed_tile_count.argtypes = [i64]
    L.bml_dense_mixed_tile_of_cta.restype = ctypes.c_int
    L.bml_dense_mixed_tile_of_cta.argtypes = [i64, i32, ctypes.POINTER(ctypes.c_int32)]
    i32p, dblp = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(dbl)
    L.bml_chebyshev_workspace_bytes.restype = sz
    L.bml_chebyshev_workspace_bytes.argtypes = [i64, i32, i32]
    L.bml_chebyshev_dense.restype = ctypes.c_int
    L.bml_chebyshev_dense.argtypes = [MP, ctypes.POINTER(bml_cheb_params_t), MP, vp, sz,
                                      ctypes.POINTER(bml_cheb_stats_t), vp]
    L.bml_symm_ab_workspace_bytes.restype = sz
    L.bml_symm_ab_workspace_bytes.argtypes = []
    L.bml_symm_ab_dense.restype = ctypes.c_int
    L.bml_symm_ab_dense.argtypes = [vp, i64, i64, i64, i32, i32, i32p, i32p, i32p, i32p, dblp, dblp, dblp, vp, sz, vp]
    L.bml_cheb_schedule.restype = ctypes.c_int
    L.bml_cheb_schedule.argtypes = [i32, i32p, i32p, i32p]
    L.bml_symm_work_item.restype = ctypes.c_int
    L.bml_symm_work_item.argtypes = [i64, i32, i32, i32, i32, i32p]
    L.bml_graph_workspace_bytes.restype = sz
    L.bml_graph_workspace_bytes.argtypes = [i64, i32, i32, i32, i32]
    L.bml_graph_chebyshev_ellpack.restype = ctypes.c_int
    L.bml_graph_chebyshev_ellpack.argtypes = [MP, vp, vp, ctypes.POINTER(bml_graph_params_t), MP, vp, sz,
                                              ctypes.POINTER(bml_graph_stats_t), vp]
    L.bml_graph_sp2_workspace_bytes.restype = sz
    L.bml_graph_sp2_workspace_bytes.argtypes = [i64, i32, i32]
    L.bml_graph_sp2_ellpack.restype = ctypes.c_int
    L.bml_graph_sp2_ellpack.argtypes = [MP, vp, vp, ctypes.POINTER(bml_graph_sp2_params_t), MP, vp, sz,
                                        ctypes.POINTER(bml_graph_sp2_stats_t), vp]
    L.bml_dense_batch_work_item.restype = ctypes.c_int
    L.bml_dense_batch_work_item.argtypes = [i32, i32p, i32, i32, i32, i32p]
    EP = ctypes.POINTER(bml_ellblock_t)
    L.bml_gershgorin_ellblock_workspace_bytes.restype = sz
    L.bml_gershgorin_ellblock_workspace_bytes.argtypes = [i64, i32]
    L.bml_gershgorin_ellblock.restype = ctypes.c_int
    L.bml_gershgorin_ellblock.argtypes = [EP, vp, vp, sz, vp]
    L.bml_trace_ellblock.restype = ctypes.c_int
    L.bml_trace_ellblock.argtypes = [EP, vp, vp]
    for name in ("bml_sp2_ellblock_workspace_bytes", "bml_x2_ellblock_workspace_bytes"):
        getattr(L, name).restype = sz
        getattr(L, name).argtypes = [i64, i32, i32]
    L.bml_sp2_ellblock.restype = ctypes.c_int
    L.bml_sp2_ellblock.argtypes = [EP, PP, EP, vp, sz, SP, vp]
    L.bml_x2_ellblock.restype = ctypes.c_int
    L.bml_x2_ellblock.argtypes = [EP, EP, i32, dbl, vp, vp, vp, sz, vp]
    L.bml_graph_core_halo.restype = ctypes.c_int
    L.bml_graph_core_halo.argtypes = [MP, vp, vp, i32, dbl, vp, vp, vp, vp, sz, vp]
    L.bml_matrix2submatrix_ellpack.restype = ctypes.c_int
    L.bml_matrix2submatrix_ellpack.argtypes = [MP, vp, i32, vp, i64, vp]
    L.bml_submatrix2matrix_ellpack.restype = ctypes.c_int
    L.bml_submatrix2matrix_ellpack.argtypes = [vp, i64, vp, vp, i32, dbl, MP, vp, vp]
    _lib = L
    return L


def bml_version() -> str:
    return load().bml_version().decode()


def bml_status_string(status: int) -> str:
    return load().bml_status_string(int(status)).decode()


# ------------------------------------------------------------------------------------------------------------
# marshalling helpers
# ------------------------------------------------------------------------------------------------------------
def _require_cuda(t: torch.Tensor, dtype, what: str):
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise RuntimeError(f"{what}: expected a CUDA tensor (libbmlsp2 has no CPU path)")
    if t.dtype != dtype:
        raise TypeError(f"{what}: expected {dtype}, got {t.dtype}")


def _stream() -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def dense_desc(A: torch.Tensor) -> bml_matrix_t:
    """Descriptor of a row-major 2-D float64 CUDA tensor (rows may be strided: ld = A.stride(0))."""
    _require_cuda(A, torch.float64, "dense matrix")
    if A.dim() != 2 or A.shape[0] != A.shape[1] or A.stride(1) != 1:
        raise ValueError("dense matrix must be square, row-major with unit column stride")
    return bml_matrix_t(BML_DENSE, 0, A.shape[0], A.stride(0), A.data_ptr(), None, None)


def ellpack_desc(value: torch.Tensor, index: torch.Tensor, nnz: torch.Tensor) -> bml_matrix_t:
    _require_cuda(value, torch.float64, "ellpack value")
    _require_cuda(index, torch.int32, "ellpack index")
    _require_cuda(nnz, torch.int32, "ellpack nnz")
    if value.dim() != 2 or index.shape != value.shape or nnz.shape != (value.shape[0],):
        raise ValueError("ellpack: value[N,M], index[N,M], nnz[N] expected")
    if not (value.is_contiguous() and index.is_contiguous() and nnz.is_contiguous()):
        raise ValueError("ellpack arrays must be contiguous")
    N, M = value.shape
    return bml_matrix_t(BML_ELLPACK, M, N, 0, value.data_ptr(), index.data_ptr(), nnz.data_ptr())


def _workspace(nbytes: int, device) -> torch.Tensor:
    # torch's caching allocator returns 512-byte aligned blocks; over-allocate and slice to a 1024-byte boundary
    raw = torch.empty(int(nbytes) + 1024, dtype=torch.uint8, device=device)
    off = (-raw.data_ptr()) % 1024
    return raw[off:off + int(nbytes)]


@dataclass
class Sp2Result:
    status: int
    n_products: int
    m_star: int
    overflow_row: int
    emin: float
    emax: float
    branch: str
    trace: np.ndarray
    idem: np.ndarray
    max_row_nnz: np.ndarray
    message: str = field(default="")


def _result(st: bml_sp2_stats_t, rc: int) -> Sp2Result:
    n = max(int(st.n_products), 0)
    m = max(int(st.m_star), 0)
    nb = m
    return Sp2Result(
        status=int(rc), n_products=n, m_star=int(st.m_star), overflow_row=int(st.overflow_row),
        emin=float(st.emin), emax=float(st.emax),
        branch="".join(str(int(b)) for b in st.branch[:nb]),
        trace=np.array(st.trace[:n]), idem=np.array(st.idem[:n]), max_row_nnz=np.array(st.max_row_nnz[:n]),
        message=bml_status_string(rc),
    )


# ------------------------------------------------------------------------------------------------------------
# entry points (same names as the C ABI)
# ------------------------------------------------------------------------------------------------------------
def bml_gershgorin(H, out: torch.Tensor | None = None) -> torch.Tensor:
    """H: dense tensor or (value, index, nnz).  Returns a CUDA float64 tensor [e_min, e_max] (asynchronous)."""
    L = load()
    desc = dense_desc(H) if isinstance(H, torch.Tensor) else ellpack_desc(*H)
    dev = H.device if isinstance(H, torch.Tensor) else H[0].device
    if out is None:
        out = torch.empty(2, dtype=torch.float64, device=dev)
    nbytes = L.bml_gershgorin_workspace_bytes(desc.N)
    ws = torch.empty(max(nbytes, 8), dtype=torch.uint8, device=dev)
    rc = L.bml_gershgorin(ctypes.byref(desc), out.data_ptr(), ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_gershgorin: {bml_status_string(rc)}")
    return out


def bml_gershgorin_static(H, out: torch.Tensor) -> torch.Tensor:
    """include/bml_no_alloc.h: bml_gershgorin with the library's static scratch; allocates nothing, so `out` (CUDA float64
    [2]) is the caller's.  N <= GERSHGORIN_STATIC_MAX_N; calls that overlap on the GPU race on the scratch."""
    L = load()
    desc = dense_desc(H) if isinstance(H, torch.Tensor) else ellpack_desc(*H)
    _require_cuda(out, torch.float64, "bounds")
    if out.numel() < 2 or not out.is_contiguous():
        raise ValueError("bounds: contiguous float64[2] expected")
    rc = L.bml_gershgorin_static(ctypes.byref(desc), out.data_ptr(), _stream())
    if rc != 0:
        raise RuntimeError(f"bml_gershgorin_static: {L.bml_no_alloc_status_string(rc).decode()}")
    return out


def bml_lanczos_bounds(H, steps: int, seed: int = 0) -> torch.Tensor:
    """Tighter spectral bounds (bml_sp2.h): CUDA float64 tensor [e_min, e_max] (asynchronous)."""
    L = load()
    desc = dense_desc(H) if isinstance(H, torch.Tensor) else ellpack_desc(*H)
    dev = H.device if isinstance(H, torch.Tensor) else H[0].device
    out = torch.empty(2, dtype=torch.float64, device=dev)
    nbytes = L.bml_lanczos_bounds_workspace_bytes(desc.N)
    ws = torch.empty(max(nbytes, 8), dtype=torch.uint8, device=dev)
    rc = L.bml_lanczos_bounds(ctypes.byref(desc), int(steps), int(seed), out.data_ptr(), ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_lanczos_bounds: {bml_status_string(rc)}")
    return out


def bml_trace(A, out: torch.Tensor | None = None) -> torch.Tensor:
    L = load()
    desc = dense_desc(A) if isinstance(A, torch.Tensor) else ellpack_desc(*A)
    dev = A.device if isinstance(A, torch.Tensor) else A[0].device
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=dev)
    rc = L.bml_trace(ctypes.byref(desc), out.data_ptr(), _stream())
    if rc != 0:
        raise RuntimeError(f"bml_trace: {bml_status_string(rc)}")
    return out


class DenseSolver:
    """Pre-allocated buffers for repeated bml_sp2_dense calls on one problem size (bench.py's timed loop)."""

    def __init__(self, N: int, device="cuda", precision: int = 0):
        L = load()
        self.N, self.precision = int(N), int(precision)
        self.device = torch.device(device)
        self.D = torch.empty((N, N), dtype=torch.float64, device=self.device)
        d = bml_matrix_t(BML_DENSE, 0, N, N, None, None, None)
        p = bml_sp2_params_t(1, 1, 1.0, 0.0, precision, 0)
        self.ws_bytes = L.bml_sp2_workspace_bytes(ctypes.byref(d), ctypes.byref(p))
        self.ws = _workspace(self.ws_bytes, self.device)

    def solve(self, H: torch.Tensor, n_occ: int, idem_tol: float, max_products: int = 100, flags: int = 0,
              asynchronous: bool = False):
        """asynchronous=True passes stats = NULL: nothing is synchronised, the result is read later by read_stats()."""
        L = load()
        h, d = dense_desc(H), dense_desc(self.D)
        p = bml_sp2_params_t(int(n_occ), int(max_products), float(idem_tol), 0.0, self.precision, int(flags))
        st = bml_sp2_stats_t()
        rc = L.bml_sp2_dense(ctypes.byref(h), ctypes.byref(p), ctypes.byref(d), self.ws.data_ptr(), self.ws_bytes,
                             None if asynchronous else ctypes.byref(st), _stream())
        if asynchronous:
            if rc != 0:
                raise RuntimeError(f"bml_sp2_dense: {bml_status_string(rc)}")
            return self.D, None
        return self.D, _result(st, rc)

    def read_stats(self) -> "Sp2Result":
        return bml_sp2_read_stats(self.ws)


def bml_sp2_dense(H: torch.Tensor, n_occ: int, idem_tol: float, max_products: int = 100, precision: int = 0,
                  flags: int = 0):
    """Dense SP2.  Returns (D CUDA tensor, Sp2Result)."""
    _require_cuda(H, torch.float64, "H")
    return DenseSolver(H.shape[0], H.device, precision).solve(H, n_occ, idem_tol, max_products, flags)


class EllpackSolver:
    def __init__(self, N: int, M: int, device="cuda"):
        L = load()
        self.N, self.M = int(N), int(M)
        self.device = torch.device(device)
        self.dv = torch.zeros((N, M), dtype=torch.float64, device=self.device)
        self.di = torch.zeros((N, M), dtype=torch.int32, device=self.device)
        self.dn = torch.zeros((N,), dtype=torch.int32, device=self.device)
        d = bml_matrix_t(BML_ELLPACK, M, N, 0, None, None, None)
        self.ws_bytes = L.bml_sp2_workspace_bytes(ctypes.byref(d), None)
        self.ws = _workspace(self.ws_bytes, self.device)

    def solve(self, value, index, nnz, n_occ: int, idem_tol: float, drop_tol: float, max_products: int = 100,
              flags: int = 0, asynchronous: bool = False):
        L = load()
        h = ellpack_desc(value, index, nnz)
        d = ellpack_desc(self.dv, self.di, self.dn)
        p = bml_sp2_params_t(int(n_occ), int(max_products), float(idem_tol), float(drop_tol), 0, int(flags))
        st = bml_sp2_stats_t()
        rc = L.bml_sp2_ellpack(ctypes.byref(h), ctypes.byref(p), ctypes.byref(d), self.ws.data_ptr(), self.ws_bytes,
                               None if asynchronous else ctypes.byref(st), _stream())
        if asynchronous:
            if rc != 0:
                raise RuntimeError(f"bml_sp2_ellpack: {bml_status_string(rc)}")
            return (self.dv, self.di, self.dn), None
        return (self.dv, self.di, self.dn), _result(st, rc)

    def read_stats(self) -> "Sp2Result":
        return bml_sp2_read_stats(self.ws)


def bml_sp2_ellpack(value, index, nnz, n_occ: int, idem_tol: float, drop_tol: float, max_products: int = 100,
                    flags: int = 0):
    """Sparse thresholded SP2 on ELLPACK-R.  Returns ((value, index, nnz) CUDA tensors of D, Sp2Result)."""
    _require_cuda(value, torch.float64, "value")
    return EllpackSolver(value.shape[0], value.shape[1], value.device).solve(value, index, nnz, n_occ, idem_tol,
                                                                           drop_tol, max_products, flags)


def bml_sp2_read_stats(ws: torch.Tensor) -> Sp2Result:
    """Result of the last bml_sp2_* call on workspace `ws` (for calls made with stats = NULL); synchronises."""
    st = bml_sp2_stats_t()
    rc = load().bml_sp2_read_stats(ws.data_ptr(), ctypes.byref(st), _stream())
    return _result(st, rc)


def bml_sp2_release_cached() -> None:
    load().bml_sp2_release_cached()


def padded_ld(N: int) -> int:
    return (int(N) + 15) // 16 * 16


def bml_x2_dense(X: torch.Tensor, branch: int, precision: int = 0, Xnext: torch.Tensor | None = None, ws=None):
    """One fused product on a padded iterate (ld multiple of 16).  Returns (Xnext, sums[4] CUDA tensor)."""
    L = load()
    x = dense_desc(X)
    if Xnext is None:
        Xnext = torch.empty_strided(X.shape, X.stride(), dtype=X.dtype, device=X.device)
    xn = dense_desc(Xnext)
    sums = torch.empty(4, dtype=torch.float64, device=X.device)
    nbytes = L.bml_x2_dense_workspace_bytes(x.N, precision)
    if ws is None:
        ws = _workspace(nbytes, X.device)
    rc = L.bml_x2_dense(ctypes.byref(x), ctypes.byref(xn), int(branch), int(precision), sums.data_ptr(),
                        ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_x2_dense: {bml_status_string(rc)}")
    return Xnext, sums


def padded_dense(A: np.ndarray | torch.Tensor, device="cuda") -> torch.Tensor:
    """Copy a square matrix into a zero-padded CUDA buffer with ld = padded_ld(N), 128-byte aligned; returns the
    N x N view (stride ld)."""
    A = torch.as_tensor(A, dtype=torch.float64)
    N = A.shape[0]
    ld = padded_ld(N)
    raw = torch.zeros(N * ld + 16, dtype=torch.float64, device=device)
    off = ((-raw.data_ptr()) % 128) // 8
    buf = raw[off:off + N * ld].view(N, ld)
    buf[:, :N].copy_(A)
    return buf[:, :N]


def bml_x2_ellpack(X, branch: int, drop_tol: float, out=None, ws=None):
    """One fused thresholded product on ELLPACK-R rows in ascending column order.
    Returns ((value, index, nnz), sums[4], info[4]) — all CUDA tensors."""
    L = load()
    value, index, nnz = X
    x = ellpack_desc(value, index, nnz)
    if out is None:
        out = (torch.zeros_like(value), torch.zeros_like(index), torch.zeros_like(nnz))
    o = ellpack_desc(*out)
    sums = torch.empty(4, dtype=torch.float64, device=value.device)
    info = torch.empty(4, dtype=torch.int32, device=value.device)
    nbytes = L.bml_x2_ellpack_workspace_bytes(x.N, x.M)
    if ws is None:
        ws = _workspace(nbytes, value.device)
    rc = L.bml_x2_ellpack(ctypes.byref(x), ctypes.byref(o), int(branch), float(drop_tol), sums.data_ptr(),
                          info.data_ptr(), ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_x2_ellpack: {bml_status_string(rc)}")
    return out, sums, info


def bml_dense_work_items(N: int, n_ctas: int, cta: int):
    """Work list of one CTA of the persistent FP64 kernel: [(tile, I, J, kt_begin, kt_end), ...] (host arithmetic)."""
    L = load()
    out = (ctypes.c_int32 * 5)()
    items, it = [], 0
    while True:
        rc = L.bml_dense_work_item(int(N), int(n_ctas), int(cta), it, out)
        if rc == 1:
            return items
        if rc != 0:
            raise RuntimeError(f"bml_dense_work_item: {bml_status_string(rc)}")
        items.append(tuple(out))
        it += 1


def bml_dense_mixed_tiles(N: int):
    """CTA -> tile map of the mixed kernel: list of (I, J) or None for the empty slots (host arithmetic)."""
    L = load()
    out = (ctypes.c_int32 * 2)()
    res = []
    for cta in range(L.bml_dense_mixed_tile_count(int(N))):
        rc = L.bml_dense_mixed_tile_of_cta(int(N), cta, out)
        if rc < 0:
            raise RuntimeError(f"bml_dense_mixed_tile_of_cta: {bml_status_string(rc)}")
        res.append(None if rc == 1 else (out[0], out[1]))
    return res


def bml_probe_fp64_tensor_peak(iters: int = 20000) -> float:
    """FP64 tensor-pipe (DMMA) issue peak in TFLOP/s at the clocks of this run."""
    L = load()
    flops, ms = ctypes.c_double(), ctypes.c_double()
    rc = L.bml_probe_fp64_tensor_peak(int(iters), ctypes.byref(flops), ctypes.byref(ms), _stream())
    if rc != 0:
        raise RuntimeError(f"bml_probe_fp64_tensor_peak: {bml_status_string(rc)}")
    return flops.value / (ms.value * 1e-3) / 1e12


# ------------------------------------------------------------------------------------------------------------
# include/bml_chebyshev.h
# ------------------------------------------------------------------------------------------------------------
@dataclass
class ChebResult:
    status: int
    n_products: int
    n_launches: int
    L: int
    emin: float
    emax: float
    trace: float
    c: np.ndarray          # c_0 .. c_L
    d: np.ndarray          # d[i, j], shape (k, m)
    message: str = field(default="")


class ChebyshevSolver:
    """Pre-allocated workspace for repeated bml_chebyshev_dense calls on one (N, k, m)."""

    def __init__(self, N: int, k: int, m: int, device="cuda"):
        L = load()
        self.N, self.k, self.m = int(N), int(k), int(m)
        self.device = torch.device(device)
        self.D = torch.empty((N, N), dtype=torch.float64, device=self.device)
        self.ws_bytes = L.bml_chebyshev_workspace_bytes(self.N, self.k, self.m)
        if self.ws_bytes == 0:
            raise RuntimeError("bml_chebyshev_workspace_bytes: " + bml_status_string(-1))
        self.ws = _workspace(self.ws_bytes, self.device)

    def solve(self, H: torch.Tensor, mu: float, beta: float, flags: int = 0):
        L = load()
        h, d = dense_desc(H), dense_desc(self.D)
        p = bml_cheb_params_t(float(mu), float(beta), self.k, self.m, int(flags), 0)
        st = bml_cheb_stats_t()
        rc = L.bml_chebyshev_dense(ctypes.byref(h), ctypes.byref(p), ctypes.byref(d), self.ws.data_ptr(),
                                   self.ws_bytes, ctypes.byref(st), _stream())
        n = self.k * self.m
        res = ChebResult(status=int(rc), n_products=int(st.n_products), n_launches=int(st.n_launches), L=int(st.L),
                         emin=float(st.emin), emax=float(st.emax), trace=float(st.trace), c=np.array(st.c[:n]),
                         d=np.array(st.d[:n]).reshape(self.m, self.k).T.copy(), message=bml_status_string(rc))
        return self.D, res


def bml_chebyshev_dense(H: torch.Tensor, mu: float, beta: float, k: int, m: int, flags: int = 0):
    """D ~ f_mu(H) by the resummed Chebyshev expansion (Eq. 10-14).  Returns (D CUDA tensor, ChebResult)."""
    _require_cuda(H, torch.float64, "H")
    if not (2 <= int(k) <= CHEB_MAX_K and 1 <= int(m) <= CHEB_MAX_M and int(k) * int(m) <= CHEB_MAX_TERMS):
        D = torch.empty_like(H)
        h, d = dense_desc(H), dense_desc(D)
        p = bml_cheb_params_t(float(mu), float(beta), int(k), int(m), int(flags), 0)
        st = bml_cheb_stats_t()
        rc = load().bml_chebyshev_dense(ctypes.byref(h), ctypes.byref(p), ctypes.byref(d), None, 0, ctypes.byref(st),
                                        _stream())
        return D, ChebResult(int(rc), 0, 0, 0, 0.0, 0.0, 0.0, np.zeros(0), np.zeros((0, 0)), bml_status_string(rc))
    return ChebyshevSolver(H.shape[0], k, m, H.device).solve(H, mu, beta, flags)


def matrix_slab(mats, device="cuda"):
    """Copy square matrices into one zero-padded CUDA slab (slot s at s * slot_elems, ld = padded_ld(N), 128-byte
    aligned).  Returns (slab tensor [n, slot_elems], N, ld, slot_elems)."""
    mats = [torch.as_tensor(np.asarray(a), dtype=torch.float64) for a in mats]
    N = mats[0].shape[0]
    ld = padded_ld(N)
    slot_elems = (N * ld + 127) // 128 * 128
    raw = torch.zeros(len(mats) * slot_elems + 16, dtype=torch.float64, device=device)
    off = ((-raw.data_ptr()) % 128) // 8
    slab = raw[off:off + len(mats) * slot_elems].view(len(mats), slot_elems)
    for s, a in enumerate(mats):
        slab[s, :N * ld].view(N, ld)[:, :N].copy_(a)
    return slab, N, ld, slot_elems


def slab_matrix(slab: torch.Tensor, s: int, N: int, ld: int) -> torch.Tensor:
    return slab[s, :N * ld].view(N, ld)[:, :N]


def bml_symm_ab_dense(slab: torch.Tensor, N: int, ld: int, jobs, ws=None):
    """One grouped launch on a slab from matrix_slab().  jobs: [(a, b, c or -1, out, alpha, beta, gamma), ...]:
    slot[out] <- alpha slot[a] slot[b] + beta slot[c] + gamma I.  Asynchronous; results are written into the slab."""
    L = load()
    _require_cuda(slab, torch.float64, "slab")
    n = len(jobs)
    i32a, dbla = ctypes.c_int32 * max(n, 1), ctypes.c_double * max(n, 1)
    cols = list(zip(*jobs)) if n else [[]] * 7
    a, b, c, o = (i32a(*[int(v) for v in col]) for col in cols[:4])
    al, be, ga = (dbla(*[float(v) for v in col]) for col in cols[4:])
    nbytes = L.bml_symm_ab_workspace_bytes()
    if ws is None:
        ws = _workspace(nbytes, slab.device)
    rc = L.bml_symm_ab_dense(slab.data_ptr(), int(N), int(ld), int(slab.stride(0)), int(slab.shape[0]), n, a, b, c, o,
                             al, be, ga, ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_symm_ab_dense: {bml_status_string(rc)}")
    return slab


def bml_cheb_schedule(k: int):
    """[(i, level, a, b)] for i = 2..k with T_i = 2 T_a T_b - T_{a-b} (host arithmetic)."""
    L = load()
    n = max(int(k) - 1, 1)
    lv, a, b = (ctypes.c_int32 * n)(), (ctypes.c_int32 * n)(), (ctypes.c_int32 * n)()
    rc = L.bml_cheb_schedule(int(k), lv, a, b)
    if rc < 0:
        raise RuntimeError(f"bml_cheb_schedule: {bml_status_string(rc)}")
    return [(i, lv[i - 2], a[i - 2], b[i - 2]) for i in range(2, int(k) + 1)]


def bml_symm_work_items(N: int, n_jobs: int, n_ctas: int, cta: int):
    """Work list of one CTA of a grouped launch: [(job, I, J, kt_begin, kt_end, tile_edge), ...] (host arithmetic)."""
    L = load()
    out = (ctypes.c_int32 * 6)()
    items, it = [], 0
    while True:
        rc = L.bml_symm_work_item(int(N), int(n_jobs), int(n_ctas), int(cta), it, out)
        if rc == 1:
            return items
        if rc != 0:
            raise RuntimeError(f"bml_symm_work_item: {bml_status_string(rc)}")
        items.append(tuple(out))
        it += 1


# ------------------------------------------------------------------------------------------------------------
# include/bml_graph.h
# ------------------------------------------------------------------------------------------------------------
@dataclass
class GraphResult:
    status: int
    n_parts: int
    overflow_row: int
    max_part_size: int
    n_products: int
    part_size: list
    core_size: list
    message: str = field(default="")


class GraphSolver:
    """Pre-allocated output and workspace for repeated bml_graph_chebyshev_ellpack calls."""

    def __init__(self, N: int, M_out: int, n_parts: int, part_capacity: int, k: int, m: int, device="cuda"):
        L = load()
        self.N, self.M_out, self.n_parts, self.cap, self.k, self.m = int(N), int(M_out), int(n_parts), int(part_capacity), int(k), int(m)
        self.device = torch.device(device)
        self.dv = torch.zeros((N, M_out), dtype=torch.float64, device=self.device)
        self.di = torch.zeros((N, M_out), dtype=torch.int32, device=self.device)
        self.dn = torch.zeros((N,), dtype=torch.int32, device=self.device)
        self.ws_bytes = L.bml_graph_workspace_bytes(self.N, self.n_parts, self.cap, self.k, self.m)
        if self.ws_bytes == 0:
            raise RuntimeError("bml_graph_workspace_bytes: " + bml_status_string(-1))
        self.ws = _workspace(self.ws_bytes, self.device)

    def solve(self, H, core_offsets: torch.Tensor, core_nodes: torch.Tensor, graph_tol: float, mu: float, beta: float,
              drop_tol: float):
        L = load()
        h = ellpack_desc(*H)
        d = ellpack_desc(self.dv, self.di, self.dn)
        _require_cuda(core_offsets, torch.int32, "core_offsets")
        _require_cuda(core_nodes, torch.int32, "core_nodes")
        p = bml_graph_params_t(float(mu), float(beta), float(graph_tol), float(drop_tol), self.k, self.m, self.n_parts,
                               self.cap)
        st = bml_graph_stats_t()
        rc = L.bml_graph_chebyshev_ellpack(ctypes.byref(h), core_offsets.data_ptr(), core_nodes.data_ptr(), ctypes.byref(p),
                                           ctypes.byref(d), self.ws.data_ptr(), self.ws_bytes, ctypes.byref(st), _stream())
        P = self.n_parts
        res = GraphResult(int(rc), int(st.n_parts), int(st.overflow_row), int(st.max_part_size), int(st.n_products),
                          list(st.part_size[:P]), list(st.core_size[:P]), bml_status_string(rc))
        return (self.dv, self.di, self.dn), res


def bml_graph_chebyshev_ellpack(H, core_offsets, core_nodes, graph_tol, mu, beta, k, m, drop_tol, M_out, part_capacity):
    """Graph-based D (Listing 11 with the Chebyshev local solver).  Returns ((value, index, nnz) of D, GraphResult)."""
    N = H[0].shape[0]
    solver = GraphSolver(N, M_out, core_offsets.numel() - 1, part_capacity, k, m, H[0].device)
    return solver.solve(H, core_offsets, core_nodes, graph_tol, mu, beta, drop_tol)


@dataclass
class GraphSp2Result:
    status: int
    sp2: Sp2Result
    n_parts: int
    overflow_row: int
    max_part_size: int
    part_size: list
    core_size: list
    message: str = field(default="")


class GraphSp2Solver:
    """Pre-allocated output and workspace for repeated bml_graph_sp2_ellpack calls (SP2 as the local solver)."""

    def __init__(self, N: int, M_out: int, n_parts: int, part_capacity: int, device="cuda"):
        L = load()
        self.N, self.M_out, self.n_parts, self.cap = int(N), int(M_out), int(n_parts), int(part_capacity)
        self.device = torch.device(device)
        self.dv = torch.zeros((N, M_out), dtype=torch.float64, device=self.device)
        self.di = torch.zeros((N, M_out), dtype=torch.int32, device=self.device)
        self.dn = torch.zeros((N,), dtype=torch.int32, device=self.device)
        self.ws_bytes = L.bml_graph_sp2_workspace_bytes(self.N, self.n_parts, self.cap)
        if self.ws_bytes == 0:
            raise RuntimeError("bml_graph_sp2_workspace_bytes: " + bml_status_string(-1))
        self.ws = _workspace(self.ws_bytes, self.device)

    def solve(self, H, core_offsets: torch.Tensor, core_nodes: torch.Tensor, graph_tol: float, n_occ: int,
              idem_tol: float, drop_tol: float, max_products: int = 100):
        L = load()
        h = ellpack_desc(*H)
        d = ellpack_desc(self.dv, self.di, self.dn)
        _require_cuda(core_offsets, torch.int32, "core_offsets")
        _require_cuda(core_nodes, torch.int32, "core_nodes")
        p = bml_graph_sp2_params_t(float(graph_tol), float(drop_tol), float(idem_tol), int(n_occ), int(max_products),
                                   self.n_parts, self.cap)
        st = bml_graph_sp2_stats_t()
        rc = L.bml_graph_sp2_ellpack(ctypes.byref(h), core_offsets.data_ptr(), core_nodes.data_ptr(), ctypes.byref(p),
                                     ctypes.byref(d), self.ws.data_ptr(), self.ws_bytes, ctypes.byref(st), _stream())
        P = self.n_parts
        res = GraphSp2Result(int(rc), _result(st.sp2, rc), int(st.n_parts), int(st.overflow_row), int(st.max_part_size),
                             list(st.part_size[:P]), list(st.core_size[:P]), bml_status_string(rc))
        return (self.dv, self.di, self.dn), res


def bml_graph_sp2_ellpack(H, core_offsets, core_nodes, graph_tol, n_occ, idem_tol, drop_tol, M_out, part_capacity,
                          max_products: int = 100):
    """Graph-based D with SP2 as the local solver (one shared polynomial).  Returns ((value, index, nnz), GraphSp2Result)."""
    N = H[0].shape[0]
    solver = GraphSp2Solver(N, M_out, core_offsets.numel() - 1, part_capacity, H[0].device)
    return solver.solve(H, core_offsets, core_nodes, graph_tol, n_occ, idem_tol, drop_tol, max_products)


# ------------------------------------------------------------------------------------------------------------
# ELLBLOCK (include/bml_ellblock.h): value[NB, MB, bs, bs] float64, index[NB, MB] int32, nnz[NB] int32
# ------------------------------------------------------------------------------------------------------------
def ellblock_desc(value: torch.Tensor, index: torch.Tensor, nnz: torch.Tensor) -> bml_ellblock_t:
    _require_cuda(value, torch.float64, "ellblock value")
    _require_cuda(index, torch.int32, "ellblock index")
    _require_cuda(nnz, torch.int32, "ellblock nnz")
    if value.dim() != 4 or value.shape[2] != value.shape[3] or index.shape != value.shape[:2] or nnz.shape != (value.shape[0],):
        raise ValueError("ellblock: value[NB,MB,bs,bs], index[NB,MB], nnz[NB] expected")
    if not (value.is_contiguous() and index.is_contiguous() and nnz.is_contiguous()):
        raise ValueError("ellblock arrays must be contiguous")
    NB, MB, bs, _ = value.shape
    return bml_ellblock_t(bs, MB, NB, value.data_ptr(), index.data_ptr(), nnz.data_ptr())


def bml_gershgorin_ellblock(H) -> torch.Tensor:
    L = load()
    d = ellblock_desc(*H)
    out = torch.empty(2, dtype=torch.float64, device=H[0].device)
    nbytes = L.bml_gershgorin_ellblock_workspace_bytes(d.NB, d.bs)
    ws = torch.empty(max(nbytes, 8), dtype=torch.uint8, device=H[0].device)
    rc = L.bml_gershgorin_ellblock(ctypes.byref(d), out.data_ptr(), ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_gershgorin_ellblock: {bml_status_string(rc)}")
    return out


def bml_trace_ellblock(A) -> torch.Tensor:
    d = ellblock_desc(*A)
    out = torch.empty(1, dtype=torch.float64, device=A[0].device)
    rc = load().bml_trace_ellblock(ctypes.byref(d), out.data_ptr(), _stream())
    if rc != 0:
        raise RuntimeError(f"bml_trace_ellblock: {bml_status_string(rc)}")
    return out


class EllblockSolver:
    def __init__(self, NB: int, MB: int, bs: int, device="cuda"):
        L = load()
        self.NB, self.MB, self.bs = int(NB), int(MB), int(bs)
        self.device = torch.device(device)
        self.dv = torch.zeros((NB, MB, bs, bs), dtype=torch.float64, device=self.device)
        self.di = torch.zeros((NB, MB), dtype=torch.int32, device=self.device)
        self.dn = torch.zeros((NB,), dtype=torch.int32, device=self.device)
        self.ws_bytes = L.bml_sp2_ellblock_workspace_bytes(self.NB, self.MB, self.bs)
        if self.ws_bytes == 0:
            raise RuntimeError("bml_sp2_ellblock_workspace_bytes: " + bml_status_string(-1))
        self.ws = _workspace(self.ws_bytes, self.device)

    def solve(self, value, index, nnz, n_occ: int, idem_tol: float, drop_tol: float, max_products: int = 100):
        L = load()
        h = ellblock_desc(value, index, nnz)
        d = ellblock_desc(self.dv, self.di, self.dn)
        p = bml_sp2_params_t(int(n_occ), int(max_products), float(idem_tol), float(drop_tol), 0, 0)
        st = bml_sp2_stats_t()
        rc = L.bml_sp2_ellblock(ctypes.byref(h), ctypes.byref(p), ctypes.byref(d), self.ws.data_ptr(), self.ws_bytes,
                                ctypes.byref(st), _stream())
        return (self.dv, self.di, self.dn), _result(st, rc)


def bml_sp2_ellblock(value, index, nnz, n_occ: int, idem_tol: float, drop_tol: float, max_products: int = 100):
    """Thresholded SP2 on ELLBLOCK.  Returns ((value, index, nnz) CUDA tensors of D, Sp2Result)."""
    _require_cuda(value, torch.float64, "value")
    NB, MB, bs, _ = value.shape
    return EllblockSolver(NB, MB, bs, value.device).solve(value, index, nnz, n_occ, idem_tol, drop_tol, max_products)


def bml_x2_ellblock(X, branch: int, drop_tol: float, out=None, ws=None):
    """One fused block product on an ELLBLOCK iterate (block rows ascending, X symmetric).
    Returns ((value, index, nnz), sums[4], info[4]) -- all CUDA tensors."""
    L = load()
    value, index, nnz = X
    x = ellblock_desc(value, index, nnz)
    if out is None:
        out = (torch.zeros_like(value), torch.zeros_like(index), torch.zeros_like(nnz))
    o = ellblock_desc(*out)
    sums = torch.empty(4, dtype=torch.float64, device=value.device)
    info = torch.empty(4, dtype=torch.int32, device=value.device)
    nbytes = L.bml_x2_ellblock_workspace_bytes(x.NB, x.MB, x.bs)
    if nbytes == 0:
        raise RuntimeError("bml_x2_ellblock_workspace_bytes: " + bml_status_string(-1))
    if ws is None:
        ws = _workspace(nbytes, value.device)
    rc = L.bml_x2_ellblock(ctypes.byref(x), ctypes.byref(o), int(branch), float(drop_tol), sums.data_ptr(), info.data_ptr(),
                           ws.data_ptr(), nbytes, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_x2_ellblock: {bml_status_string(rc)}")
    return out, sums, info


def bml_dense_batch_work_items(sizes, n_ctas: int, cta: int):
    """Work list of one CTA of the batched symmetric-square kernel: [(part, tile, kt_begin, kt_end, KT), ...]."""
    L = load()
    n = (ctypes.c_int32 * len(sizes))(*[int(x) for x in sizes])
    out = (ctypes.c_int32 * 5)()
    items, it = [], 0
    while True:
        rc = L.bml_dense_batch_work_item(len(sizes), n, int(n_ctas), int(cta), it, out)
        if rc == 1:
            return items
        if rc != 0:
            raise RuntimeError(f"bml_dense_batch_work_item: {bml_status_string(rc)}")
        items.append(tuple(out))
        it += 1


def bml_graph_core_halo(H, core_offsets: torch.Tensor, core_nodes: torch.Tensor, graph_tol: float):
    """Returns (part_nodes[P, N] int32, is_core[P, N] uint8, sizes[P, 2] int32) CUDA tensors (asynchronous)."""
    L = load()
    h = ellpack_desc(*H)
    P, N = core_offsets.numel() - 1, h.N
    dev = H[0].device
    nodes = torch.zeros((P, N), dtype=torch.int32, device=dev)
    is_core = torch.zeros((P, N), dtype=torch.uint8, device=dev)
    sizes = torch.zeros((P, 2), dtype=torch.int32, device=dev)
    ws = torch.empty(P * N, dtype=torch.uint8, device=dev)
    rc = L.bml_graph_core_halo(ctypes.byref(h), core_offsets.data_ptr(), core_nodes.data_ptr(), P, float(graph_tol),
                               nodes.data_ptr(), is_core.data_ptr(), sizes.data_ptr(), ws.data_ptr(), P * N, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_graph_core_halo: {bml_status_string(rc)}")
    return nodes, is_core, sizes


def bml_matrix2submatrix_ellpack(H, nodes: torch.Tensor) -> torch.Tensor:
    """Dense h = H[nodes, nodes] (nodes: ascending int32 CUDA tensor)."""
    L = load()
    h = ellpack_desc(*H)
    s = int(nodes.numel())
    out = torch.empty((s, s), dtype=torch.float64, device=nodes.device)
    rc = L.bml_matrix2submatrix_ellpack(ctypes.byref(h), nodes.data_ptr(), s, out.data_ptr(), s, _stream())
    if rc != 0:
        raise RuntimeError(f"bml_matrix2submatrix_ellpack: {bml_status_string(rc)}")
    return out


def bml_submatrix2matrix_ellpack(d: torch.Tensor, nodes: torch.Tensor, is_core: torch.Tensor, drop_tol: float, D):
    """Scatter the core rows of dense d into the ELLPACK-R triple D.  Returns the overflow row tensor (INT32_MAX = none)."""
    L = load()
    _require_cuda(d, torch.float64, "d")
    dd = ellpack_desc(*D)
    ov = torch.full((1,), 2**31 - 1, dtype=torch.int32, device=d.device)
    rc = L.bml_submatrix2matrix_ellpack(d.data_ptr(), d.stride(0), nodes.data_ptr(), is_core.data_ptr(), int(nodes.numel()),
                                        float(drop_tol), ctypes.byref(dd), ov.data_ptr(), _stream())
    if rc != 0:
        raise RuntimeError(f"bml_submatrix2matrix_ellpack: {bml_status_string(rc)}")
    return ov
