"""CPU oracle for the graph-based density-matrix path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain numpy, FP64, pure-Python loops over rows.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this module; it imports nothing from ``paper_2401_13772_b200``.

What the path computes (section VIII.B, Listing 11):

    A_ij = 1 if |G_ij| >= tau and i != j else 0                                   Eq. 15
    core partition  Pi_c = {pi_1^c .. pi_m^c}: every node in exactly one part
    core-halo part  pi_k^ch = pi_k^c  U  { o : A_lo = 1 for some l in pi_k^c }
    h^k = H[i in pi_k^ch, j in pi_k^ch]            (bml_matrix2submatrix)          P:496, Listing 11
    d^k = f(h^k)                                   (the local solver)
    D[l, :] <- d^k[l, :] for the CORE nodes l of part k   (bml_submatrix2matrix)   P:498, Listing 11

Readings of the paper (items G1-G6):
  G1. The auxiliary matrix G "can be the Hamiltonian itself": G = H.
  G2. The order of the nodes inside a part is not given ("a one-to-one mapping"): ascending global index.
  G3. The local solver is any DM solver ("for example a regular diagonalization").  Here: the Fermi operator
      f_mu at a known chemical potential by the Chebyshev expansion of section IV.B (oracle/chebyshev.py), each part
      on its OWN Gershgorin interval.
  G4. What is mapped back: the rows of the core nodes, over all columns of the part ("extract the submatrices
      corresponding to the core partition and map them back"; the halo rows are discarded, they belong to
      other cores).  D is therefore assembled row by row and is symmetric only up to the method's own error.
  G5. D is stored in ELLPACK-R with the SP2 path's drop rule: keep |v| >= drop_tol or the diagonal; a row that needs
      more than M slots is the overflow failure of P:47-49 (status -3).
  G6. The core partition is an INPUT (partitioning "stays external": METIS etc.); ``regular_partition`` is the
      paper's "simply divide the matrix index list into relatively regular segments".

H is given in ELLPACK-R as (value[N, M], index[N, M], nnz[N]) like everywhere else in this repository.
"""
from __future__ import annotations

import numpy as np

from . import chebyshev as och


def regular_partition(N, n_parts):
    """Core partition into n_parts contiguous index segments of nearly equal length (reading G6).
    Returns (core_offsets[n_parts + 1], core_nodes[N])."""
    offs = np.array([(p * N) // n_parts for p in range(n_parts + 1)], dtype=np.int32)
    return offs, np.arange(N, dtype=np.int32)


def core_halo(value, index, nnz, core, tau):
    """Sorted node list of pi^ch for one core part and the mask of its core nodes (Eq. 15 + P:494, readings G1, G2)."""
    N = value.shape[0]
    mark = np.zeros(N, dtype=np.int8)
    for l in core:
        for p in range(int(nnz[l])):
            o = int(index[l, p])
            if o != l and abs(value[l, p]) >= tau:
                mark[o] = 1
    for l in core:
        mark[l] = 2
    nodes = np.nonzero(mark)[0].astype(np.int32)
    return nodes, mark[nodes] == 2


def matrix2submatrix(value, index, nnz, nodes):
    """Dense h[a, b] = H[nodes[a], nodes[b]] (bml_matrix2submatrix): every stored entry, no threshold."""
    s = nodes.size
    pos = {int(j): b for b, j in enumerate(nodes)}
    h = np.zeros((s, s))
    for a, i in enumerate(nodes):
        for p in range(int(nnz[i])):
            b = pos.get(int(index[i, p]))
            if b is not None:
                h[a, b] = value[i, p]
    return h


def submatrix2matrix(d, nodes, is_core, drop_tol, dv, di, dn):
    """Write the core rows of d into the ELLPACK-R matrix (dv, di, dn) (bml_submatrix2matrix, readings G4, G5).
    Returns the lowest overflowing row or -1."""
    M = dv.shape[1]
    bad = -1
    for a, i in enumerate(nodes):
        if not is_core[a]:
            continue
        keep = (np.abs(d[a]) >= drop_tol) | (nodes == i)
        cols = nodes[keep]
        if cols.size > M:
            bad = int(i) if bad < 0 else min(bad, int(i))
            continue
        dn[i] = cols.size
        di[i, : cols.size] = cols
        dv[i, : cols.size] = d[a, keep]
    return bad


def graph_fermi(value, index, nnz, core_offsets, core_nodes, graph_tol, mu, beta, k, m, drop_tol, M_out=None,
                local="chebyshev"):
    """Listing 11 with the local solver of reading G3.  D has M_out slots per row (default: as H).
    Returns ((dv, di, dn), info).
    local = "chebyshev": sum_n c_n T_n(h~) by the plain series (the parity target of the GPU path);
    local = "exact": U f(Lambda) U^T by LAPACK (used by the pins to separate the graph error from the expansion's)."""
    N = value.shape[0]
    M = value.shape[1] if M_out is None else int(M_out)
    dv, di, dn = np.zeros((N, M)), np.zeros((N, M), dtype=np.int32), np.zeros(N, dtype=np.int32)
    sizes, bad = [], -1
    for p in range(len(core_offsets) - 1):
        core = core_nodes[core_offsets[p]: core_offsets[p + 1]]
        nodes, is_core = core_halo(value, index, nnz, core, graph_tol)
        h = matrix2submatrix(value, index, nnz, nodes)
        if local == "exact":
            d = och.fermi_exact(h, mu, beta)
        else:
            d, _ = och.chebyshev_serial(h, mu, beta, k * m - 1)
        b = submatrix2matrix(d, nodes, is_core, drop_tol, dv, di, dn)
        if b >= 0:
            bad = b if bad < 0 else min(bad, b)
        sizes.append(int(nodes.size))
    return (dv, di, dn), {"part_sizes": sizes, "overflow_row": bad, "status": -3 if bad >= 0 else 0}
