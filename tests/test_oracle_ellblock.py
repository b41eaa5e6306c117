"""Pins of the ELLBLOCK oracle (oracle/sp2_oracle.c section ELLBLOCK; "ELLBLOCK is a generalization of
ELLPACK-R where each element is a block"; readings E1-E4) against what the definitions fix.  CPU only.

* bs = 1 IS the scalar ELLPACK-R format: every routine must reproduce the (already pinned) scalar ELLPACK oracle bit
  for bit -- product, update, rescale with an inserted diagonal, the whole thresholded SP2 solve.
* tau = 0 with every block stored is the dense matrix in block storage: the product must equal the dense product, the
  solve the dense SP2 solve (Jacobi-pinned in test_oracle_pins.py).
* the block threshold (Frobenius norm of the BLOCK >= tau, diagonal blocks always kept) on hand-built blocks.
* block products against numpy's matmul on random blocks (catches a transposed operand inside the block loop, a
  wrong k range, row-major / column-major confusion in the block layout)."""
import math

import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm


def sparse_model(L=(8, 6, 5), M=64, seed=0):
    return hm.lattice_ellpack(L, 12.0, 0.2, 2.0, lambda r: -math.exp(-r / 0.5), M, seed)


def as_bs1(ell):
    v, i, n = ell
    return v[:, :, None, None].copy(), i.copy(), n.copy()


def test_bs1_is_the_scalar_ellpack_oracle_bit_for_bit(oracle_mod):
    H = sparse_model()
    lo, hi = oracle_mod.gershgorin_ellpack(*H)
    assert oracle_mod.gershgorin_ellblock(*as_bs1(H)) == (lo, hi)
    X = oracle_mod.rescale_ellpack(*H, lo, hi)
    Xb = oracle_mod.rescale_ellblock(*as_bs1(H), lo, hi)
    assert X[3] == Xb[3] == -1
    for a, b in zip(X[:3], Xb[:3]):
        assert np.array_equal(a, b.reshape(a.shape))
    assert oracle_mod.trace_ellblock(*Xb[:3]) == oracle_mod.trace_ellpack(*X[:3])
    for tau in (0.0, 1e-6, 1e-3):
        P = oracle_mod.x2_ellpack(*X[:3], tau)
        Pb = oracle_mod.x2_ellblock(*Xb[:3], tau)
        assert P[3:] == Pb[3:]
        for a, b in zip(P[:3], Pb[:3]):
            assert np.array_equal(a, b.reshape(a.shape))
        U = oracle_mod.update_ellpack(X[:3], P[:3], tau)
        Ub = oracle_mod.update_ellblock(Xb[:3], Pb[:3], tau)
        assert U[3:] == Ub[3:]
        for a, b in zip(U[:3], Ub[:3]):
            assert np.array_equal(a, b.reshape(a.shape))


@pytest.mark.parametrize("tau,tol", [(1e-6, 1e-8), (0.0, 1e-10), (1e-4, 1e-8)])
def test_bs1_full_solve_is_the_scalar_ellpack_solve(oracle_mod, tau, tol):
    H = sparse_model((8, 6, 5), M=240)
    N = H[0].shape[0]
    D, st = oracle_mod.sp2_ellpack(*H, N // 2, tol, tau)
    Db, stb = oracle_mod.sp2_ellblock(*as_bs1(H), N // 2, tol, tau)
    for key in ("status", "n_products", "m_star", "branch", "emin", "emax", "overflow_row"):
        assert st[key] == stb[key], key
    assert np.array_equal(st["trace"], stb["trace"]) and np.array_equal(st["max_row_nnz"], stb["max_row_nnz"])
    np.testing.assert_allclose(stb["idem"], st["idem"], rtol=1e-12)        # norms are summed row-wise vs block-row-wise
    for a, b in zip(D, Db):
        assert np.array_equal(a, b.reshape(a.shape))


def test_missing_diagonal_block_is_inserted_in_order(oracle_mod):
    bs, MB = 2, 3
    A = np.zeros((6, 6))
    A[0:2, 0:2] = [[1.0, 0.5], [0.5, -1.0]]
    A[0:2, 4:6] = A[4:6, 0:2] = [[0.25, 0.0], [0.0, 0.25]]
    A[4:6, 4:6] = [[2.0, 0.0], [0.0, -2.0]]
    A[2:4, 0:2] = [[0.125, 0.0], [0.0, 0.0]]
    A[0:2, 2:4] = A[2:4, 0:2].T
    v, i, n = hm.ellblock_from_dense(A, bs, MB)
    # remove the (all-zero) diagonal block of block row 1: it holds only block column 0 then
    assert i[1, : n[1]].tolist() == [0, 1]
    v[1, 1] = 0.0; i[1, 1] = 0; n[1] = 1
    xv, xi, xn, bad = oracle_mod.rescale_ellblock(v, i, n, -3.0, 5.0)
    assert bad == -1 and xn.tolist() == [3, 2, 2] and xi[1, :2].tolist() == [0, 1]
    s = 1.0 / 8.0
    assert xv[1, 1].tolist() == [[s * 5.0, -0.0], [-0.0, s * 5.0]]            # inserted: X_ii = s (e_max - 0)
    assert xv[1, 0].tolist() == [[-s * 0.125, -0.0], [-0.0, -0.0]]
    assert xv[0, 0].tolist() == [[s * 4.0, -s * 0.5], [-s * 0.5, s * 6.0]]
    # a full block row without its diagonal block cannot take it: reported
    v2, i2, n2 = v[:, :1].copy(), i[:, :1].copy(), np.ones(3, dtype=np.int32)
    i2[:, 0] = [2, 0, 0]
    assert oracle_mod.rescale_ellblock(v2, i2, n2, -3.0, 5.0)[3] == 0


@pytest.mark.parametrize("bs", [2, 4, 8, 16])
def test_tau0_all_blocks_stored_is_the_dense_product_and_solve(oracle_mod, bs):
    rng = np.random.default_rng(bs)
    N = 48
    H, eps = hm.planted_gap(N, 20, gap=1.0, width=1.0, seed=bs)
    NB = N // bs
    Hb = hm.ellblock_from_dense(H, bs, NB, tol=-1.0)                      # tol < 0: every block stored
    assert int(Hb[2].min()) == NB
    lo, hi = oracle_mod.gershgorin_dense(H)
    assert oracle_mod.gershgorin_ellblock(*Hb) == (lo, hi)
    X = oracle_mod.rescale_dense(H, lo, hi)
    Xb = oracle_mod.rescale_ellblock(*Hb, lo, hi)
    assert np.array_equal(hm.ellblock_to_dense(*Xb[:3]), X)
    P = hm.ellblock_to_dense(*oracle_mod.x2_ellblock(*Xb[:3], 0.0)[:3])
    assert np.abs(P - X @ X).max() <= 1e-15 * N                           # numpy matmul: the independent routine
    assert np.abs(P - oracle_mod.x2_dense(X)).max() <= 1e-15 * N
    D, st = oracle_mod.sp2_dense(H, 20, 1e-10)
    Db, stb = oracle_mod.sp2_ellblock(*Hb, 20, 1e-10, 0.0)
    assert (st["status"], st["branch"], st["n_products"]) == (stb["status"], stb["branch"], stb["n_products"])
    assert np.abs(hm.ellblock_to_dense(*Db) - D).max() <= 1e-12
    v = np.linalg.eigh(H)[1][:, :20]
    assert np.linalg.norm(hm.ellblock_to_dense(*Db) - v @ v.T) / math.sqrt(20) <= 1e-9       # the projector itself


def test_block_products_against_numpy_on_a_block_sparse_pattern(oracle_mod):
    """Random block-sparse symmetric X (blocks missing): every stored block of X X against the dense numpy product;
    blocks whose chain is empty must not appear at all."""
    bs, NB, MB = 4, 9, 9
    rng = np.random.default_rng(2)
    A = np.zeros((NB * bs, NB * bs))
    for I in range(NB):
        for J in range(I, NB):
            if I == J or rng.random() < 0.25:
                B = rng.normal(size=(bs, bs))
                A[I * bs:(I + 1) * bs, J * bs:(J + 1) * bs] = B
                A[J * bs:(J + 1) * bs, I * bs:(I + 1) * bs] = B.T
        A[I * bs:(I + 1) * bs, I * bs:(I + 1) * bs] = (A[I * bs:(I + 1) * bs, I * bs:(I + 1) * bs] + A[I * bs:(I + 1) * bs, I * bs:(I + 1) * bs].T) / 2
    Xb = hm.ellblock_from_dense(A, bs, MB)
    pv, pi, pn, bad, mx = oracle_mod.x2_ellblock(*Xb, 0.0)
    assert bad == -1
    ref = A @ A
    pat = (np.abs(A.reshape(NB, bs, NB, bs)).sum(axis=(1, 3)) > 0).astype(int)
    reach = (pat @ pat) > 0                                                 # block (I, J) has a non-empty chain
    for I in range(NB):
        assert pi[I, : pn[I]].tolist() == np.nonzero(reach[I])[0].tolist()
        for p in range(pn[I]):
            J = pi[I, p]
            assert np.abs(pv[I, p] - ref[I * bs:(I + 1) * bs, J * bs:(J + 1) * bs]).max() <= 1e-13
    assert mx == int(reach.sum(axis=1).max())


def test_block_threshold_rule_hand_cases(oracle_mod):
    """Reading E2: a block is kept iff its Frobenius norm >= tau or it is diagonal.  X = diag of 2 x 2 blocks, so
    X X is block diagonal plus what the one off-diagonal coupling produces; norms are chosen by hand."""
    bs, MB = 2, 2
    A = np.zeros((4, 4))
    A[0:2, 0:2] = [[0.5, 0.0], [0.0, 0.5]]
    A[2:4, 2:4] = [[1e-3, 0.0], [0.0, 1e-3]]              # tiny diagonal block: kept whatever tau is
    A[0:2, 2:4] = [[0.3, 0.4], [0.0, 0.0]]                # Frobenius norm 0.5
    A[2:4, 0:2] = A[0:2, 2:4].T
    Xb = hm.ellblock_from_dense(A, bs, MB)
    P = A @ A
    off = np.linalg.norm(P[0:2, 2:4])                     # 0.5 * 0.501 = 0.2505
    for tau, kept in ((off, True), (np.nextafter(off, 1.0), False), (0.0, True)):
        pv, pi, pn, bad, mx = oracle_mod.x2_ellblock(*Xb, tau)
        assert pi[0, : pn[0]].tolist() == ([0, 1] if kept else [0])
        assert pi[1, : pn[1]].tolist() == ([0, 1] if kept else [1])        # the tiny diagonal block survives
        assert np.abs(pv[1, pn[1] - 1] - P[2:4, 2:4]).max() <= 1e-18
    # a single large entry keeps a block whose other entries are far below tau (norm, not entry-wise)
    pv, pi, pn, _, _ = oracle_mod.x2_ellblock(*Xb, 0.2)
    assert pn.tolist() == [2, 2] and abs(pv[0, 1, 1, 1]) < 0.2
    # overflow of the block slots: lowest block row reported
    H = sparse_model((8, 6, 5), M=64)
    Hb = hm.ellblock_from_ellpack(*H, 5, 24)
    lo, hi = oracle_mod.gershgorin_ellblock(*Hb)
    Xb2 = oracle_mod.rescale_ellblock(*Hb, lo, hi)[:3]
    bad = oracle_mod.x2_ellblock(*Xb2, 0.0)[3]
    assert bad == 0


@pytest.mark.parametrize("bs", [4, 8])
def test_thresholded_block_solve_reaches_the_projector(oracle_mod, bs):
    """The thresholded block solve on the sparse insulator: stops on S1 or its noise floor, tr D = N_occ, D close to
    the LAPACK projector at the level of the truncation, and at least as accurate as the scalar path at the same tau
    (block thresholding keeps a superset of the scalar path's entries)."""
    H = sparse_model((8, 5, 8), M=64)
    N = H[0].shape[0]
    Hd = hm.ellpack_to_dense(*H)
    Hb = hm.ellblock_from_ellpack(*H, bs, N // bs)          # as many slots as block columns: no overflow possible
    assert np.array_equal(hm.ellblock_to_dense(*Hb), Hd)
    Db, st = oracle_mod.sp2_ellblock(*Hb, N // 2, 1e-8, 1e-6)
    assert st["status"] in (0, 1)
    D = hm.ellblock_to_dense(*Db)
    v = np.linalg.eigh(Hd)[1][:, : N // 2]
    err = np.linalg.norm(D - v @ v.T) / np.linalg.norm(v @ v.T)
    Ds, _ = oracle_mod.sp2_ellpack(*H, N // 2, 1e-8, 1e-6)
    err_s = np.linalg.norm(hm.ellpack_to_dense(*Ds) - v @ v.T) / np.linalg.norm(v @ v.T)
    assert err <= 1e-5 and err <= 1.5 * err_s
    assert abs(np.trace(D) - N // 2) <= 1e-4
    assert np.array_equal(D, D.T)
