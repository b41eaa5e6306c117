"""Pins of the graph-based density-matrix oracle (oracle/graph.py; PAPER.md VIII.B, Eq. 15, Listing 11) against what
the definitions fix.  CPU only.  Each pin names the mistake it is meant to catch."""
import math

import numpy as np
import pytest

from oracle import chebyshev as och
from oracle import graph as og
from paper_2401_13772_b200 import hamiltonians as hm


def model(L=(8, 6, 6), rmax=2.0, decay=1.0, delta=1.5, M=64, seed=0):
    return hm.lattice_ellpack(L, delta, 0.2, rmax, lambda r: -math.exp(-r / decay), M, seed)


def dense_of(ell):
    return hm.ellpack_to_dense(*ell)


def test_regular_partition_is_an_exact_cover():
    for N, P in [(10, 3), (64, 8), (1000, 7), (5, 5)]:
        offs, nodes = og.regular_partition(N, P)
        assert offs[0] == 0 and offs[-1] == N and np.all(np.diff(offs) >= N // P) and np.all(np.diff(offs) <= N // P + 1)
        assert np.array_equal(np.sort(nodes), np.arange(N))


@pytest.mark.parametrize("tau", [0.0, 0.1, 0.2, 0.5])
def test_core_halo_is_core_plus_first_neighbours_of_eq15(tau):
    """pi^ch against the definition written with a dense boolean adjacency matrix (Eq. 15): catches a threshold applied
    with the wrong sign, the diagonal counted as an edge, or a halo built from rows of halo nodes (two hops)."""
    H = model()
    Hd = dense_of(H)
    N = Hd.shape[0]
    A = (np.abs(Hd) >= tau) & ~np.eye(N, dtype=bool) & (Hd != 0)
    offs, nodes = og.regular_partition(N, 4)
    for p in range(4):
        core = nodes[offs[p]: offs[p + 1]]
        got, is_core = og.core_halo(*H, core, tau)
        expect = np.zeros(N, dtype=bool)
        expect[core] = True
        expect |= A[core].any(axis=0)
        assert np.array_equal(got, np.nonzero(expect)[0])
        assert np.array_equal(got[is_core], np.sort(core))
        assert np.all(np.diff(got) > 0)


def test_matrix2submatrix_is_fancy_indexing():
    H = model()
    Hd = dense_of(H)
    rng = np.random.default_rng(1)
    nodes = np.sort(rng.choice(Hd.shape[0], 77, replace=False)).astype(np.int32)
    assert np.array_equal(og.matrix2submatrix(*H, nodes), Hd[np.ix_(nodes, nodes)])


def test_submatrix2matrix_writes_core_rows_only_with_the_drop_rule():
    nodes = np.array([2, 5, 7, 9], dtype=np.int32)
    is_core = np.array([False, True, True, False])
    d = np.array([[9.0, 9, 9, 9], [1e-3, 0.5, 1e-9, -2e-3], [1e-9, 1e-9, 1e-12, 1e-9], [9.0, 9, 9, 9]])
    dv, di, dn = np.zeros((12, 3)), np.zeros((12, 3), dtype=np.int32), np.zeros(12, dtype=np.int32)
    bad = og.submatrix2matrix(d, nodes, is_core, 1e-6, dv, di, dn)
    assert bad == -1
    assert dn.tolist() == [0, 0, 0, 0, 0, 3, 0, 1, 0, 0, 0, 0]
    assert di[5].tolist() == [2, 5, 9] and dv[5].tolist() == [1e-3, 0.5, -2e-3]
    assert di[7, 0] == 7 and dv[7, 0] == 1e-12          # the diagonal is kept whatever its size
    dv2, di2, dn2 = np.zeros((12, 2)), np.zeros((12, 2), dtype=np.int32), np.zeros(12, dtype=np.int32)
    assert og.submatrix2matrix(d, nodes, is_core, 1e-6, dv2, di2, dn2) == 5     # row 5 needs 3 > M = 2 slots


def test_halo_covering_everything_reproduces_the_global_expansion():
    """graph_tol = 0 on a full matrix: every part's core+halo is the whole system, h^k = H, so
    the core rows of every part are rows of the global sum_n c_n T_n(H~) bit for bit (catches a wrong row/column map
    in gather or scatter)."""
    rng = np.random.default_rng(8)
    G = rng.normal(size=(30, 30))
    Hd = (G + G.T) / 2
    H = hm.ellpack_from_dense(Hd, 30)
    N = 30
    offs, nodes = og.regular_partition(N, 3)
    first, _ = og.core_halo(*H, nodes[offs[0]: offs[1]], 0.0)
    assert first.size == N, "the test needs a halo that covers the box"
    (dv, di, dn), info = og.graph_fermi(*H, offs, nodes, 0.0, 0.0, 2.0, 8, 8, 0.0)
    D_ref, _ = och.chebyshev_serial(Hd, 0.0, 2.0, 63)
    assert info["part_sizes"] == [N, N, N] and info["status"] == 0
    assert np.array_equal(hm.ellpack_to_dense(dv, di, dn), D_ref)


def test_disconnected_parts_are_exact():
    """Block-diagonal H whose blocks are the parts: halo = core and D = blockdiag f(h_k) = f(H) (LAPACK) -- the
    graph-based theory's statement for a disconnected graph."""
    rng = np.random.default_rng(3)
    blocks = []
    for s in (20, 25, 19):
        G = rng.normal(size=(s, s))
        blocks.append((G + G.T) / 2)
    N = sum(b.shape[0] for b in blocks)
    Hd = np.zeros((N, N))
    o = 0
    for b in blocks:
        Hd[o:o + b.shape[0], o:o + b.shape[0]] = b
        o += b.shape[0]
    H = hm.ellpack_from_dense(Hd, 32)
    offs = np.array([0, 20, 45, 64], dtype=np.int32)
    (dv, di, dn), info = og.graph_fermi(*H, offs, np.arange(N, dtype=np.int32), 0.0, 0.2, 1.5, 8, 8, 0.0, local="exact")
    assert info["part_sizes"] == [20, 25, 19]
    assert np.allclose(hm.ellpack_to_dense(dv, di, dn), och.fermi_exact(Hd, 0.2, 1.5), atol=1e-13)


def test_error_falls_as_the_graph_threshold_falls():
    """Fig. 8's trend: a smaller adjacency threshold means larger halos and a smaller error against the dense Fermi
    operator; with the exact local solver the error is the graph approximation alone."""
    H = model(L=(24, 7, 7), rmax=3.0, decay=1.0, M=128)
    Hd = dense_of(H)
    N = Hd.shape[0]
    offs, nodes = og.regular_partition(N, 3)
    De = och.fermi_exact(Hd, 0.0, 3.0)
    errs, sizes = [], []
    for tau in (0.5, 0.2, 0.1, 0.04):          # neighbours up to r = 0 (none beyond e^-1 = 0.37), 1.41, 2.24, 3
        (dv, di, dn), info = og.graph_fermi(*H, offs, nodes, tau, 0.0, 3.0, 8, 8, 0.0, M_out=700, local="exact")
        assert info["status"] == 0
        errs.append(np.linalg.norm(hm.ellpack_to_dense(dv, di, dn) - De) / np.linalg.norm(De))
        sizes.append(max(info["part_sizes"]))
    assert sizes == sorted(sizes) and sizes[0] < sizes[-1]
    assert all(a > b for a, b in zip(errs, errs[1:])), errs
    assert errs[-1] < 0.2 * errs[0]


def test_chebyshev_local_solver_matches_the_exact_one_within_truncation():
    H = model(L=(8, 6, 6), rmax=2.0, M=64)
    N = H[0].shape[0]
    offs, nodes = og.regular_partition(N, 4)
    a, ia = og.graph_fermi(*H, offs, nodes, 0.1, 0.0, 1.0, 8, 8, 0.0, M_out=288, local="chebyshev")
    b, ib = og.graph_fermi(*H, offs, nodes, 0.1, 0.0, 1.0, 8, 8, 0.0, M_out=288, local="exact")
    assert ia["status"] == 0 and ib["status"] == 0
    assert np.allclose(hm.ellpack_to_dense(*a), hm.ellpack_to_dense(*b), atol=1e-8)
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[1], b[1])        # drop_tol = 0: same pattern


# ---------------------------------------------------------------------------------------------------------------
# graph_sp2: SP2 as the local solver (reading G3'; Listing 11 with prg_build_DM = SP2, one polynomial for all parts)
# ---------------------------------------------------------------------------------------------------------------
def gapped_model(L=(8, 6, 5), M=64, seed=0):
    """The 5'-like insulator (on-site +-12, hopping -exp(-r / 0.5), r <= 2): wide gap, D decays fast."""
    return hm.lattice_ellpack(L, 12.0, 0.2, 2.0, lambda r: -math.exp(-r / 0.5), M, seed)


def test_graph_sp2_single_part_is_the_dense_sp2_oracle():
    """One part that is the whole matrix (halo = nothing to add): graph_sp2 must walk exactly the dense SP2 oracle's
    iterates -- same bounds, same branch string, same product count, D equal entry by entry.  Catches a wrong Eq. 5 map
    (per-part bounds), a trace over the wrong node set, a branch / stop test out of Listing 2's order."""
    import oracle

    H = gapped_model()
    Hd = dense_of(H)
    N = Hd.shape[0]
    D_ref, st = oracle.sp2_dense(Hd, N // 2, 1e-10)
    offs, nodes = og.regular_partition(N, 1)
    (dv, di, dn), info = og.graph_sp2(*H, offs, nodes, 0.0, N // 2, 1e-10, 0.0, M_out=N)
    assert info["status"] == st["status"] == 0
    assert (info["emin"], info["emax"]) == (st["emin"], st["emax"])
    assert info["branch"] == st["branch"] and info["n_products"] == st["n_products"]
    np.testing.assert_allclose(info["trace"], st["trace"], rtol=0, atol=1e-11)
    np.testing.assert_allclose(info["idem"], st["idem"], rtol=1e-9, atol=1e-16)
    assert np.array_equal(hm.ellpack_to_dense(dv, di, dn), D_ref)


def test_graph_sp2_disconnected_parts_equal_the_global_solve():
    """H block diagonal with the blocks as parts (no halo at any threshold): the global X_m stays block diagonal, the
    traces and squared norms add up over the blocks, so the shared branch sequence is the global one and every block
    of D is the global D's block.  Catches per-part branch decisions and per-part occupation counts."""
    import oracle

    rng = np.random.default_rng(5)
    sizes = [7, 12, 9]
    N = sum(sizes)
    Hd = np.zeros((N, N))
    o = 0
    for s, shift in zip(sizes, (-0.8, 0.1, 0.9)):          # different fillings per block: the split of N_occ is not N/2 each
        A = rng.normal(size=(s, s))
        Hd[o:o + s, o:o + s] = (A + A.T) / 2 + shift * np.eye(s)
        o += s
    eps = np.linalg.eigvalsh(Hd)
    n_occ = 13
    assert eps[n_occ] - eps[n_occ - 1] > 0.05              # a gap at the chosen filling
    H = hm.ellpack_from_dense(Hd, N)
    offs = np.array([0, 7, 19, 28], dtype=np.int32)
    nodes = np.arange(N, dtype=np.int32)
    D_ref, st = oracle.sp2_dense(Hd, n_occ, 1e-10)
    (dv, di, dn), info = og.graph_sp2(*H, offs, nodes, 0.0, n_occ, 1e-10, 0.0, M_out=N)
    assert info["part_sizes"] == sizes and info["core_sizes"] == sizes
    assert info["status"] == st["status"] == 0 and info["branch"] == st["branch"]
    D = hm.ellpack_to_dense(dv, di, dn)
    assert np.abs(D - D_ref).max() <= 1e-13
    # the occupations of the blocks are what the global Fermi level gives them, not N_occ / parts
    occ = [np.trace(D[a:b, a:b]) for a, b in zip(offs[:-1], offs[1:])]
    want = [int((np.linalg.eigvalsh(Hd[a:b, a:b]) < (eps[n_occ - 1] + eps[n_occ]) / 2).sum()) for a, b in zip(offs[:-1], offs[1:])]
    assert np.allclose(occ, want, atol=1e-8) and len(set(want)) > 1


def test_graph_sp2_approaches_the_dense_projector_as_the_halo_grows():
    """With real halos the result is the graph approximation of the dense projector (LAPACK, Eq. 2 with the step
    function): the error must fall as graph_tol falls (Fig. 8's trend), tr D must stay near N_occ, and core rows only
    are written.  Catches halo rows leaking into D and a scatter that uses part-local column numbers."""
    H = gapped_model((12, 6, 5))
    Hd = dense_of(H)
    N = Hd.shape[0]
    w, U = np.linalg.eigh(Hd)
    n_occ = N // 2
    D_exact = U[:, :n_occ] @ U[:, :n_occ].T
    offs, nodes = og.regular_partition(N, 4)
    errs = []
    for tol in (0.2, 0.02, 0.002):                          # hopping -exp(-r/0.5): 0.135 (r=1), 0.059, 0.031, 0.018 (r=2)
        (dv, di, dn), info = og.graph_sp2(*H, offs, nodes, tol, n_occ, 1e-9, 0.0, M_out=N)
        assert info["status"] in (0, 1)
        D = hm.ellpack_to_dense(dv, di, dn)
        errs.append(np.linalg.norm(D - D_exact) / np.linalg.norm(D_exact))
        assert abs(np.trace(D) - n_occ) < 50 * errs[-1] * n_occ ** 0.5 + 1e-8
        assert np.all(dn >= 1)
    assert errs[0] > errs[1] > errs[2] and errs[2] < 2e-3
    assert info["part_sizes"][0] > info["core_sizes"][0]


def test_graph_sp2_overflow_and_degenerate_bounds():
    H = gapped_model()
    N = H[0].shape[0]
    offs, nodes = og.regular_partition(N, 2)
    (_, _, dn), info = og.graph_sp2(*H, offs, nodes, 0.02, N // 2, 1e-9, 0.0, M_out=8)      # rows of D need > 8 slots
    assert info["status"] == -3 and info["overflow_row"] == 0
    I = hm.ellpack_from_dense(2.0 * np.eye(6), 4)
    assert og.graph_sp2(*I, np.array([0, 6], dtype=np.int32), np.arange(6, dtype=np.int32), 0.0, 3, 1e-9, 0.0)[1]["status"] == -2
