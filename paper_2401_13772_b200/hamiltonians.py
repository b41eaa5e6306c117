"""Seeded synthetic Hamiltonians (inputs only — none of the SP2 method's arithmetic lives here).

These stand in for the paper's PROGRESS bio-benchmark (Table I) and the
"soft matter synthetic Hamiltonians" of its Fig. 5, neither of which is available.
The recipes are BASELINE.json's five `configs`, made concrete by SURVEY.md Appendix A:

* RNG: ``numpy.random.default_rng(seed)`` (PCG64), seed 0; on-site noise drawn first, config-1's
  dense Gaussian noise second.
* Site index of an ``Lx x Ly x Lz`` lattice: ``i = (x*Ly + y)*Lz + z``; periodic in all directions.
* On-site ``H_ii = delta*(+1 if (x+y+z) even else -1) + U[-a, a]``; hopping ``f(r)`` on the Euclidean
  minimum-image distance ``r``.

This module is used by the tests, bench.py and the smoke test to feed the SAME matrices to the CUDA path
and to the CPU oracle.  It imports neither of them.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np


# ----------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------
def stencil_offsets(rmax: float):
    """All integer displacements (dx,dy,dz) != 0 with Euclidean length <= rmax, with their length."""
    R = int(math.floor(rmax))
    out = []
    for dx in range(-R, R + 1):
        for dy in range(-R, R + 1):
            for dz in range(-R, R + 1):
                r2 = dx * dx + dy * dy + dz * dz
                if 0 < r2 <= rmax * rmax + 1e-12:
                    out.append((dx, dy, dz, math.sqrt(r2)))
    return out


def _site_coords(L):
    Lx, Ly, Lz = L
    x, y, z = np.meshgrid(np.arange(Lx), np.arange(Ly), np.arange(Lz), indexing="ij")
    return x.ravel(), y.ravel(), z.ravel()


def _onsite(L, delta, noise, rng):
    x, y, z = _site_coords(L)
    sign = np.where((x + y + z) % 2 == 0, 1.0, -1.0)
    return delta * sign + rng.uniform(-noise, noise, size=sign.size)


def lattice_dense(L, delta, noise, rmax, hop, seed=0):
    """Dense symmetric H on a periodic Lx x Ly x Lz lattice; ``hop(r)`` is the hopping at distance r."""
    Lx, Ly, Lz = L
    N = Lx * Ly * Lz
    rng = np.random.default_rng(seed)
    H = np.zeros((N, N), dtype=np.float64)
    idx = np.arange(N)
    H[idx, idx] = _onsite(L, delta, noise, rng)
    x, y, z = _site_coords(L)
    for dx, dy, dz, r in stencil_offsets(rmax):
        j = (((x + dx) % Lx) * Ly + (y + dy) % Ly) * Lz + (z + dz) % Lz
        H[idx, j] += hop(r)  # j is a permutation of idx for one displacement: no duplicate targets per call
    return H


def _images_coincide(L, rmax):
    """True when two different displacements can reach the same site (tiny boxes): use add.at then."""
    return any(2 * math.floor(rmax) >= l for l in L)


def lattice_ellpack(L, delta, noise, rmax, hop, M, seed=0):
    """ELLPACK-R (Listing 1) H: value[N*M], index[N*M] (int32), nnz[N]; rows in ascending column order.

    Unused slots hold value 0.0 / index 0.  Requires a box large enough that periodic images
    of the stencil do not coincide (2*floor(rmax) < min(L)).
    """
    Lx, Ly, Lz = L
    N = Lx * Ly * Lz
    assert not _images_coincide(L, rmax), "box too small for a unique minimum image"
    rng = np.random.default_rng(seed)
    offs = stencil_offsets(rmax)
    n_row = len(offs) + 1
    assert n_row <= M
    x, y, z = _site_coords(L)
    cols = np.empty((N, n_row), dtype=np.int64)
    vals = np.empty((N, n_row), dtype=np.float64)
    cols[:, 0] = np.arange(N)
    vals[:, 0] = _onsite(L, delta, noise, rng)
    for q, (dx, dy, dz, r) in enumerate(offs, start=1):
        cols[:, q] = (((x + dx) % Lx) * Ly + (y + dy) % Ly) * Lz + (z + dz) % Lz
        vals[:, q] = hop(r)
    order = np.argsort(cols, axis=1, kind="stable")
    cols = np.take_along_axis(cols, order, axis=1)
    vals = np.take_along_axis(vals, order, axis=1)
    value = np.zeros((N, M), dtype=np.float64)
    index = np.zeros((N, M), dtype=np.int32)
    value[:, :n_row] = vals
    index[:, :n_row] = cols.astype(np.int32)
    nnz = np.full(N, n_row, dtype=np.int32)
    return value, index, nnz


def ring_dense(N, delta, noise, sigma, seed=0):
    """Config 1: 1D ring, alternating on-site +/-delta + U[-noise,noise], NN hopping -1, plus symmetric
    Gaussian noise of std sigma on every independent entry i<=j."""
    rng = np.random.default_rng(seed)
    i = np.arange(N)
    H = np.zeros((N, N), dtype=np.float64)
    H[i, i] = np.where(i % 2 == 0, delta, -delta) + rng.uniform(-noise, noise, size=N)
    H[i, (i + 1) % N] += -1.0
    H[(i + 1) % N, i] += -1.0
    if sigma > 0:
        G = rng.normal(0.0, sigma, size=(N, N))
        H = H + (np.triu(G) + np.triu(G, 1).T)
    return H


def ellpack_from_dense(A, M, tol=0.0):
    """Pack a dense matrix into ELLPACK-R keeping |a| > tol and the diagonal (ascending columns)."""
    N = A.shape[0]
    value = np.zeros((N, M), dtype=np.float64)
    index = np.zeros((N, M), dtype=np.int32)
    nnz = np.zeros(N, dtype=np.int32)
    for i in range(N):
        keep = np.abs(A[i]) > tol
        keep[i] = True
        c = np.nonzero(keep)[0]
        assert c.size <= M, f"row {i} needs {c.size} > M={M}"
        nnz[i] = c.size
        index[i, : c.size] = c
        value[i, : c.size] = A[i, c]
    return value, index, nnz


def ellpack_to_dense(value, index, nnz, N=None):
    """Scatter an ELLPACK-R matrix into a dense array (test convenience)."""
    n = value.shape[0] if N is None else N
    M = value.shape[1]
    D = np.zeros((n, n), dtype=np.float64)
    mask = np.arange(M)[None, :] < np.asarray(nnz)[:, None]
    rows = np.broadcast_to(np.arange(n)[:, None], (n, M))[mask]
    D[rows, np.asarray(index)[mask]] = np.asarray(value)[mask]
    return D


# ----------------------------------------------------------------------------------------------
# the BASELINE.json configs
# ----------------------------------------------------------------------------------------------
def ellblock_from_dense(A, bs, MB, tol=0.0):
    """Pack a dense matrix into ELLBLOCK: value[NB, MB, bs, bs], index[NB, MB] int32 block columns
    (ascending), nnz[NB]; a block is stored iff one of its entries has |a| > tol, or it is a diagonal block.
    N must be a multiple of bs.  Layout only: no method arithmetic."""
    N = A.shape[0]
    assert N % bs == 0
    NB = N // bs
    blocks = np.ascontiguousarray(A.reshape(NB, bs, NB, bs).transpose(0, 2, 1, 3))
    keep = (np.abs(blocks) > tol).any(axis=(2, 3)) | np.eye(NB, dtype=bool)
    value = np.zeros((NB, MB, bs, bs), dtype=np.float64)
    index = np.zeros((NB, MB), dtype=np.int32)
    nnz = np.zeros(NB, dtype=np.int32)
    for I in range(NB):
        cols = np.nonzero(keep[I])[0]
        assert cols.size <= MB, "block row does not fit MB slots"
        nnz[I] = cols.size
        index[I, : cols.size] = cols
        value[I, : cols.size] = blocks[I, cols]
    return value, index, nnz


def ellblock_to_dense(value, index, nnz):
    NB, MB, bs, _ = value.shape
    A = np.zeros((NB, bs, NB, bs), dtype=np.float64)
    for I in range(NB):
        for p in range(int(nnz[I])):
            A[I, :, int(index[I, p]), :] = value[I, p]
    return A.reshape(NB * bs, NB * bs)


def ellblock_from_ellpack(value, index, nnz, bs, MB):
    """The same matrix in ELLBLOCK: every block that holds a stored scalar entry (and every diagonal block) is stored.
    Layout only (vectorised: the N = 65536 workloads have 8 million entries)."""
    N, M = value.shape
    assert N % bs == 0
    NB = N // bs
    rows = np.repeat(np.arange(N, dtype=np.int64), M).reshape(N, M)
    live = np.arange(M)[None, :] < np.asarray(nnz)[:, None]
    i, j, v = rows[live], np.asarray(index, dtype=np.int64)[live], np.asarray(value)[live]
    key = np.concatenate([(i // bs) * NB + (j // bs), np.arange(NB, dtype=np.int64) * (NB + 1)])     # + diagonal blocks
    ukey = np.unique(key)                                       # sorted: block rows ascending, block columns ascending
    bI, bJ = ukey // NB, ukey % NB
    counts = np.bincount(bI, minlength=NB)
    assert counts.max() <= MB, "block row does not fit MB slots"
    start = np.concatenate([[0], np.cumsum(counts)[:-1]])
    slot = np.arange(ukey.size) - start[bI]                     # position of every block inside its block row
    bv = np.zeros((NB, MB, bs, bs), dtype=np.float64)
    bi = np.zeros((NB, MB), dtype=np.int32)
    bi[bI, slot] = bJ.astype(np.int32)
    pos = slot[np.searchsorted(ukey, (i // bs) * NB + (j // bs))]
    bv[i // bs, pos, i % bs, j % bs] = v
    return bv, bi, counts.astype(np.int32)


@dataclasses.dataclass
class Workload:
    name: str
    kind: str  # "dense" | "ellpack"
    N: int
    n_occ: int
    idem_tol: float
    drop_tol: float = 0.0
    precision: int = 0  # 0 = FP64, 1 = mixed (FP16 x 2 split), 2 = mixed (BF16 x 3 split)
    M: int = 0
    lattice: tuple | None = None
    note: str = ""
    # Chebyshev workloads (kind "cheby"): chemical potential, inverse temperature, Eq. 10 factors L + 1 = k m
    mu: float = 0.0
    beta: float = 0.0
    k: int = 0
    m: int = 0
    # graph workloads (kind "graph"): number of core parts (regular index segments), Eq. 15 threshold, D row capacity
    n_parts: int = 0
    graph_tol: float = 0.0
    M_out: int = 0
    # ELLBLOCK workloads (kind "ellblock"): block edge and block slots per block row
    bs: int = 0
    MB: int = 0


WORKLOADS = {
    # BASELINE.json configs[0]
    "dense_n256": Workload("dense_n256", "dense", 256, 128, 1e-10, note="1D ring + dense Gaussian noise"),
    # configs[1]
    "dense_n2048": Workload("dense_n2048", "dense", 2048, 1024, 1e-10, lattice=(16, 16, 8), note="16x16x8, NN hopping"),
    # configs[2]
    "dense_n8192": Workload("dense_n8192", "dense", 8192, 4096, 1e-10, lattice=(32, 16, 16),
                            note="32x16x16, -exp(-r/1.5), r<=6"),
    # configs[3]
    "mixed_n16384": Workload("mixed_n16384", "dense", 16384, 8192, 1e-6, precision=1, lattice=(32, 32, 16),
                             note="32x32x16, -exp(-r/1.5), r<=6, mixed precision"),
    # configs[3] with the three-plane BF16 split instead of the default two-plane FP16 split
    "mixed_bf16x3_n16384": Workload("mixed_bf16x3_n16384", "dense", 16384, 8192, 1e-6, precision=2, lattice=(32, 32, 16),
                                    note="32x32x16, -exp(-r/1.5), r<=6, mixed precision (BF16 x 3 planes)"),
    # configs[4], literally as written (overflows M=512 at product 0 — SURVEY §8(d))
    "ellpack_n65536_literal": Workload("ellpack_n65536_literal", "ellpack", 65536, 32768, 1e-8, 1e-6, M=512,
                                       lattice=(64, 32, 32), note="64x32x32, -exp(-r/1.0), r<=3, delta=1.5"),
    # configs[4] labelled fallback 5': delta=12, hopping -exp(-r/0.5); same N, stencil, M, tau
    "ellpack_n65536": Workload("ellpack_n65536", "ellpack", 65536, 32768, 1e-8, 1e-6, M=512,
                               lattice=(64, 32, 32), note="5' fallback: 64x32x32, -exp(-r/0.5), r<=3, delta=12"),
}


# Chebyshev expansion workloads (PAPER.md IV.B, Fig. 3 P:247 sizes N = 500, 1000, 2000, 4000).
# The paper's inputs for Fig. 3 are not given; stand-in: a gapless ("metallic") periodic lattice -- uniform on-site
# level + U[-0.2, 0.2], nearest-neighbour hopping -1 -- at k_B T = 1/6 hopping units, mu = 0 (about half filling),
# expansion order L = 255 = 16 x 16 - 1 (truncation error 1.2e-10 relative at N = 500), i.e. the vanishing-gap / finite-temperature case SP2 cannot treat.
for _name, _L3 in (("cheby_n500", (10, 10, 5)), ("cheby_n1000", (10, 10, 10)), ("cheby_n2000", (20, 10, 10)),
                   ("cheby_n4000", (20, 20, 10)), ("cheby_n8000", (20, 20, 20))):
    _N = _L3[0] * _L3[1] * _L3[2]
    WORKLOADS[_name] = Workload(_name, "cheby", _N, _N // 2, 0.0, lattice=_L3, mu=0.0, beta=6.0, k=16, m=16,
                                note="%dx%dx%d gapless lattice, NN hopping -1, kT=1/6, L=255" % _L3)


# Graph-based solver workloads (PAPER.md VIII.B, Table II: N = 12,972, 4 parts, core
# 3149-3314, core+halo 5657-5810 -- the benchmark system itself is not available).  Stand-in: the 5' model of the sparse
# SP2 path (on-site +-12 + U[-0.2, 0.2], hopping -exp(-r/0.5), r <= 3, 123 entries per row) on a 32x20x20 box, N = 12,800,
# 4 contiguous index segments = x-slabs of 8 layers (core 3200), graph threshold 0.002 = every stored hopping, i.e. a
# halo of 3 layers on each side (core+halo 5600); mu = 0, beta = 2 (the 22.7-wide gap makes f_mu a step to 1e-10), L = 255,
# D kept at |v| >= 1e-6 in rows of 512 slots.  The small variant is what the oracle finishes in seconds.
WORKLOADS["graph_n12800"] = Workload("graph_n12800", "graph", 12800, 6400, 0.0, 1e-6, M=128, lattice=(32, 20, 20), mu=0.0,
                                     beta=2.0, k=16, m=16, n_parts=4, graph_tol=0.002, M_out=512,
                                     note="32x20x20, -exp(-r/0.5), r<=3, delta=12; 4 x-slab parts, halo 3 layers")
WORKLOADS["graph_n1536"] = Workload("graph_n1536", "graph", 1536, 768, 0.0, 1e-6, M=128, lattice=(24, 8, 8), mu=0.0,
                                    beta=2.0, k=16, m=16, n_parts=3, graph_tol=0.002, M_out=512,
                                    note="24x8x8, same model; 3 x-slab parts, halo 3 layers")


# The same two systems with SP2 as the local solver (bml_graph_sp2_ellpack, reading G3': one SP2 polynomial for all
# parts): half filling, idempotency tolerance 1e-10 on the norms summed over the parts.
WORKLOADS["graph_sp2_n12800"] = Workload("graph_sp2_n12800", "graph_sp2", 12800, 6400, 1e-10, 1e-6, M=128, lattice=(32, 20, 20),
                                         n_parts=4, graph_tol=0.002, M_out=512,
                                         note="32x20x20, -exp(-r/0.5), r<=3, delta=12; 4 x-slab parts, halo 3 layers; SP2 local solver")
WORKLOADS["graph_sp2_n1536"] = Workload("graph_sp2_n1536", "graph_sp2", 1536, 768, 1e-10, 1e-6, M=128, lattice=(24, 8, 8),
                                        n_parts=3, graph_tol=0.002, M_out=512,
                                        note="24x8x8, same model; 3 x-slab parts, halo 3 layers; SP2 local solver")


# ELLBLOCK: the 5' sparse workload of the scalar ELLPACK path stored in 8 x 8 blocks
# (z runs fastest in the site index, so a block is 8 consecutive z sites of one lattice column); same N, N_occ, tol, tau --
# tau now acts on the Frobenius norm of a block (reading E2), so the block path keeps a superset of the scalar path's
# entries.  256 block slots per block row (the iterates reach ~190).  The small variant is what the oracle finishes in seconds.
WORKLOADS["ellblock_n65536"] = Workload("ellblock_n65536", "ellblock", 65536, 32768, 1e-8, 1e-6, M=512, lattice=(64, 32, 32),
                                        bs=8, MB=256, note="5' model (64x32x32, -exp(-r/0.5), r<=3, delta=12) in 8x8 blocks")
WORKLOADS["ellblock_n8192"] = Workload("ellblock_n8192", "ellblock", 8192, 4096, 1e-8, 1e-6, M=512, lattice=(16, 16, 32),
                                       bs=8, MB=256, note="same model on 16x16x32, 8x8 blocks")


def make_ellblock(name: str, seed: int = 0):
    w = WORKLOADS[name]
    ell = lattice_ellpack(w.lattice, 12.0, 0.2, 3.0, lambda r: -math.exp(-r / 0.5), w.M, seed)
    return ellblock_from_ellpack(*ell, w.bs, w.MB)


def regular_core_partition(N: int, n_parts: int):
    """Core partition into contiguous index segments (an INPUT of the graph path): (offsets[n_parts+1], nodes[N])."""
    offs = np.array([(p * N) // n_parts for p in range(n_parts + 1)], dtype=np.int32)
    return offs, np.arange(N, dtype=np.int32)


def make_dense(name: str, seed: int = 0) -> np.ndarray:
    w = WORKLOADS[name]
    if w.kind == "cheby":
        return lattice_dense(w.lattice, 0.0, 0.2, 1.0, lambda r: -1.0, seed)
    if name == "dense_n256":
        return ring_dense(256, 1.5, 0.1, 1e-3, seed)
    if name == "dense_n2048":
        return lattice_dense(w.lattice, 1.5, 0.2, 1.0, lambda r: -1.0, seed)
    if name in ("dense_n8192", "mixed_n16384", "mixed_bf16x3_n16384"):
        return lattice_dense(w.lattice, 1.5, 0.2, 6.0, lambda r: -math.exp(-r / 1.5), seed)
    raise KeyError(name)


def make_ellpack(name: str, seed: int = 0):
    w = WORKLOADS[name]
    if w.kind in ("graph", "graph_sp2"):
        return lattice_ellpack(w.lattice, 12.0, 0.2, 3.0, lambda r: -math.exp(-r / 0.5), w.M, seed)
    if name == "ellpack_n65536_literal":
        return lattice_ellpack(w.lattice, 1.5, 0.2, 3.0, lambda r: -math.exp(-r / 1.0), w.M, seed)
    if name == "ellpack_n65536":
        return lattice_ellpack(w.lattice, 12.0, 0.2, 3.0, lambda r: -math.exp(-r / 0.5), w.M, seed)
    raise KeyError(name)


def small_long_range(L=(8, 8, 6), seed=0, rmax=3.0, decay=1.5, delta=1.5, noise=0.2):
    """Reduced-size stand-in of the config-3/4 model for parity tests the oracle finishes in seconds."""
    return lattice_dense(L, delta, noise, rmax, lambda r: -math.exp(-r / decay), seed)


def small_sparse_model(L=(12, 10, 8), seed=0, M=512, delta=12.0, decay=0.5, rmax=3.0):
    """Reduced-size stand-in of the 5' ELLPACK model."""
    return lattice_ellpack(L, delta, 0.2, rmax, lambda r: -math.exp(-r / decay), M, seed)


def planted_gap(N, n_occ, gap=1.0, width=1.0, seed=0):
    """Random dense symmetric H = Q diag(eps) Q^T with n_occ levels in [-gap/2-width, -gap/2] and the rest in
    [gap/2, gap/2+width]; Q from QR of a Gaussian matrix.  Returns (H, eps sorted ascending)."""
    rng = np.random.default_rng(seed)
    lo = -gap / 2 - width * rng.uniform(0, 1, size=n_occ)
    hi = gap / 2 + width * rng.uniform(0, 1, size=N - n_occ)
    eps = np.sort(np.concatenate([lo, hi]))
    Q, _ = np.linalg.qr(rng.normal(size=(N, N)))
    H = (Q * eps) @ Q.T
    H = np.triu(H) + np.triu(H, 1).T  # bitwise symmetric
    return H, eps
