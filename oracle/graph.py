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
  G3'. SP2 as the local solver (``graph_sp2``; "prg_build_DM" of Listing 11 is any DM solver, and SP2 is the
      paper's, section IV.A).  The graph theory behind the method needs the SAME matrix function on every part (P:456:
      "the same functions applied to only certain graph-restricted domains"), and SP2's function is fixed by its
      spectral bounds and its branch sequence.  Reading: ONE SP2 polynomial for all parts --
        * one Eq. 5 map: e_min, e_max = Gershgorin bounds of the whole H (they enclose the spectrum of every
          principal sub-matrix h^k by interlacing), X_0^k = (e_max I - h^k) / (e_max - e_min);
        * one branch bit per product, b_m = [t_m - N_occ <= 0] with the occupation counted where the result is read:
          t_m = sum_k sum_{a core of k} (X_m^k)_aa  (every orbital is a core node of exactly one part);
        * one stop test, e_m = sqrt(sum_k ||(X_m^k)^2 - X_m^k||_F^2) / sqrt(sum_k ||X_m^k||_F^2), rules S1-S3 of
          the SP2 path with the same constants; D rows = core rows of X_{m*}^k.
      A partition whose single part is the whole matrix reproduces the dense SP2 oracle exactly; on disconnected
      parts (no halo) it reproduces it up to the order of the trace / norm sums.
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


def graph_sp2(value, index, nnz, core_offsets, core_nodes, graph_tol, n_occ, idem_tol, drop_tol, max_products=100,
              M_out=None):
    """Listing 11 with SP2 (Eq. 5-7, Listing 2) as the local solver, reading G3': one Eq. 5 map, one branch sequence
    and one stop test shared by all parts.  Step by step in the order of Listing 2: trace, product, test, branch.
    Returns ((dv, di, dn), info) with info = status, m_star, n_products, branch string, trace[], idem[], emin, emax,
    part_sizes, core_sizes, overflow_row.  Status as in the SP2 path: 0 S1, 1 S2, 2 S3, -2 degenerate bounds, -3 overflow
    of a row of D.  The products are the plain triple loop of the dense SP2 oracle (sp2_oracle.c oracle_x2_dense)."""
    import math

    import oracle as osp2                      # the C SP2 oracle: Gershgorin, Eq. 5 rescale, triple-loop product

    N = value.shape[0]
    M = value.shape[1] if M_out is None else int(M_out)
    dv, di, dn = np.zeros((N, M)), np.zeros((N, M), dtype=np.int32), np.zeros(N, dtype=np.int32)
    emin, emax = osp2.gershgorin_ellpack(value, index, nnz)                       # one map for every part (Eq. 5)
    info = {"emin": emin, "emax": emax, "overflow_row": -1, "branch": "", "trace": [], "idem": [], "m_star": 0,
            "n_products": 0, "part_sizes": [], "core_sizes": []}
    if not emax - emin > 0:
        info["status"] = -2
        return (dv, di, dn), info
    parts = []
    for p in range(len(core_offsets) - 1):
        core = core_nodes[core_offsets[p]: core_offsets[p + 1]]
        nodes, is_core = core_halo(value, index, nnz, core, graph_tol)
        h = matrix2submatrix(value, index, nnz, nodes)
        parts.append([nodes, is_core, osp2.rescale_dense(h, emin, emax)])         # X_0^k
        info["part_sizes"].append(int(nodes.size))
        info["core_sizes"].append(int(is_core.sum()))
    status, m = 2, 0
    while True:
        t = math.fsum(float(X[a, a]) for _, is_core, X in parts for a in np.nonzero(is_core)[0])   # core trace
        P = [osp2.x2_dense(X) for _, _, X in parts]                                               # products
        e2 = math.fsum(float(v) for (_, _, X), Pk in zip(parts, P) for v in ((Pk - X) ** 2).ravel())
        x2 = math.fsum(float(v) for _, _, X in parts for v in (X ** 2).ravel())
        info["trace"].append(t)
        info["idem"].append(math.sqrt(e2) / math.sqrt(x2))
        e = info["idem"]
        if e[m] < idem_tol:                                       # S1
            status = 0
            break
        if m >= 2 and e[m] < 1e-2 and e[m] >= e[m - 2]:           # S2
            status = 1
            break
        if m + 1 == max_products:                                 # S3
            status = 2
            break
        b = t - float(n_occ) <= 0.0                               # Eq. 6-7, "<=" of Listing 2
        info["branch"] += "1" if b else "0"
        for part, Pk in zip(parts, P):
            part[2] = 2.0 * part[2] - Pk if b else Pk
        m += 1
    info["m_star"], info["n_products"] = m, m + 1
    bad = -1
    for nodes, is_core, X in parts:
        r = submatrix2matrix(X, nodes, is_core, drop_tol, dv, di, dn)
        if r >= 0:
            bad = r if bad < 0 else min(bad, r)
    info["overflow_row"] = bad
    info["status"] = -3 if bad >= 0 else status
    return (dv, di, dn), info
