"""GPU parity of the ELLBLOCK path (include/bml_ellblock.h; readings E1-E4) against the ELLBLOCK oracle
(oracle/sp2_oracle.c), through the C ABI.

The block products run on the FP64 tensor cores (DMMA m8n8k4), whose accumulation order inside a k-step is the
hardware's: values are compared to round-off (|err| <= 1e-13 of the largest entry per product, 1e-10 relFro for D: the
FP64 tolerance of north_star), index work (block columns, counts) bit for bit, and a keep / drop decision that differs
from the oracle's is accepted only if the block's norm sits within round-off of the threshold."""
import math

import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu
TOL_P = 1e-13
TOL_D = 1e-10


@pytest.fixture(scope="module")
def api():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2401_13772_b200 import api as a

    a.load()
    return a


def sparse_model(L=(8, 6, 8), M=64, seed=0):
    return hm.lattice_ellpack(L, 12.0, 0.2, 2.0, lambda r: -math.exp(-r / 0.5), M, seed)


def gpu(blk):
    import torch

    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in blk)


def cpu(blk):
    return tuple(a.cpu().numpy() for a in blk)


def compare_blocks(got, ref, tau, scale_tol):
    """Block patterns equal except for blocks whose norm is within round-off of tau; stored values to scale_tol."""
    gv, gi, gn = got
    rv, ri, rn = ref
    G, R = hm.ellblock_to_dense(gv, gi, gn), hm.ellblock_to_dense(rv, ri, rn)
    scale = max(np.abs(R).max(), 1e-300)
    NB, MB, bs, _ = gv.shape
    pat_g = np.zeros((NB, NB), dtype=bool)
    pat_r = np.zeros((NB, NB), dtype=bool)
    for I in range(NB):
        assert np.all(np.diff(gi[I, : gn[I]]) > 0), "block columns must ascend"
        pat_g[I, gi[I, : gn[I]]] = True
        pat_r[I, ri[I, : rn[I]]] = True
    differ = pat_g != pat_r
    for I, J in zip(*np.nonzero(differ)):
        blk = (G if pat_g[I, J] else R)[I * bs:(I + 1) * bs, J * bs:(J + 1) * bs]
        assert abs(np.linalg.norm(blk) - tau) <= 1e-12 * max(tau, scale), (I, J)
    mask = np.kron(~differ, np.ones((bs, bs), dtype=bool))
    assert np.abs(G - R)[mask].max() <= scale_tol * scale
    return int(differ.sum())


@pytest.mark.parametrize("bs", [4, 8, 16])
def test_gershgorin_and_trace_ellblock(api, oracle_mod, bs):
    H = hm.ellblock_from_ellpack(*sparse_model(), bs, 40)
    lo, hi = oracle_mod.gershgorin_ellblock(*H)
    b = api.bml_gershgorin_ellblock(gpu(H)).cpu().numpy()
    assert (b[0], b[1]) == (lo, hi)
    assert abs(api.bml_trace_ellblock(gpu(H)).item() - oracle_mod.trace_ellblock(*H)) < 1e-10


@pytest.mark.parametrize("bs,MB", [(4, 96), (8, 48), (16, 24)])
@pytest.mark.parametrize("tau", [0.0, 1e-6, 1e-3])
@pytest.mark.parametrize("branch", [0, 1])
def test_x2_ellblock_one_product(api, oracle_mod, bs, MB, tau, branch):
    H = hm.ellblock_from_ellpack(*sparse_model(), bs, MB)
    lo, hi = oracle_mod.gershgorin_ellblock(*H)
    X = oracle_mod.rescale_ellblock(*H, lo, hi)[:3]
    pv, pi, pn, bad, mx = oracle_mod.x2_ellblock(*X, tau)
    assert bad < 0
    if branch:
        ev, ei, en, bad, mxu = oracle_mod.update_ellblock(X, (pv, pi, pn), tau)
        assert bad < 0
        mx = max(mx, mxu)
    else:
        ev, ei, en = pv, pi, pn
    out, sums, info = api.bml_x2_ellblock(gpu(X), branch, tau)
    n_diff = compare_blocks(cpu(out), (ev, ei, en), tau, TOL_P)
    info = info.cpu().numpy()
    assert info[0] == np.iinfo(np.int32).max and info[1] == np.iinfo(np.int32).max
    if n_diff == 0:
        assert info[2] == mx
    Xd, Pd, Ed = (hm.ellblock_to_dense(*A) for A in (X, (pv, pi, pn), (ev, ei, en)))
    ref = np.array([np.trace(Pd), np.linalg.norm(Pd - Xd) ** 2, np.linalg.norm(Xd) ** 2, np.trace(Ed)])
    assert np.allclose(sums.cpu().numpy(), ref, rtol=1e-11, atol=1e-14)
    # the result is symmetric bit for bit (both triangles come from one computed block)
    G = hm.ellblock_to_dense(*cpu(out))
    assert np.array_equal(G, G.T)


@pytest.mark.parametrize("bs", [4, 8, 16])
def test_x2_ellblock_second_iterate_denser_rows(api, oracle_mod, bs):
    H = hm.ellblock_from_ellpack(*sparse_model((8, 8, 16)), bs, 1024 // bs)
    lo, hi = oracle_mod.gershgorin_ellblock(*H)
    X = oracle_mod.rescale_ellblock(*H, lo, hi)[:3]
    P = oracle_mod.x2_ellblock(*X, 1e-6)[:3]
    X1 = oracle_mod.update_ellblock(X, P, 1e-6)[:3]
    ref = oracle_mod.x2_ellblock(*X1, 1e-6)
    assert ref[3] < 0
    out, _, info = api.bml_x2_ellblock(gpu(X1), 0, 1e-6)
    compare_blocks(cpu(out), ref[:3], 1e-6, TOL_P)


def _check_solve(api, oracle_mod, H, n_occ, tol, tau, max_products=100):
    D_ref, st = oracle_mod.sp2_ellblock(*H, n_occ, tol, tau, max_products)
    D, res = api.bml_sp2_ellblock(*gpu(H), n_occ, tol, tau, max_products)
    assert res.status == st["status"], res.message
    assert res.n_products == st["n_products"] and res.m_star == st["m_star"] and res.branch == st["branch"]
    assert (res.emin, res.emax) == (st["emin"], st["emax"])
    assert np.allclose(res.trace, st["trace"], rtol=0, atol=1e-9)
    if res.status >= 0:
        assert np.allclose(res.idem, st["idem"], rtol=1e-6, atol=1e-14)
        n_diff = compare_blocks(cpu(D), D_ref, tau, TOL_D)
        if n_diff == 0:
            assert np.array_equal(res.max_row_nnz, st["max_row_nnz"])
    else:
        assert res.overflow_row == st["overflow_row"]
    return res, st


@pytest.mark.parametrize("bs,tau,tol", [(4, 1e-6, 1e-8), (8, 1e-6, 1e-8), (16, 1e-6, 1e-8), (8, 0.0, 1e-10), (8, 1e-4, 1e-8)])
def test_sp2_ellblock_full_solve_parity(api, oracle_mod, bs, tau, tol):
    Hs = sparse_model((8, 8, 16))
    N = Hs[0].shape[0]
    H = hm.ellblock_from_ellpack(*Hs, bs, N // bs)
    res, _ = _check_solve(api, oracle_mod, H, N // 2, tol, tau)
    assert res.status in (0, 1)


def test_sp2_ellblock_unsorted_rows_and_missing_diagonal_block(api, oracle_mod):
    bs = 8
    Hs = sparse_model((8, 8, 16))
    N = Hs[0].shape[0]
    v, i, n = hm.ellblock_from_ellpack(*Hs, bs, N // bs)
    rng = np.random.default_rng(1)
    for I in range(v.shape[0]):
        perm = rng.permutation(n[I])
        v[I, : n[I]] = v[I, perm]
        i[I, : n[I]] = i[I, perm]
    # block row 3 loses its diagonal block (H_33 := 0, not stored)
    p = int(np.nonzero(i[3, : n[3]] == 3)[0][0])
    v[3, p] = v[3, n[3] - 1]; i[3, p] = i[3, n[3] - 1]
    v[3, n[3] - 1] = 0.0; i[3, n[3] - 1] = 0; n[3] -= 1
    _check_solve(api, oracle_mod, (v, i, n), N // 2, 1e-8, 1e-6)


def test_sp2_ellblock_overflow_and_degenerate(api, oracle_mod):
    Hs = sparse_model((8, 8, 16))
    N = Hs[0].shape[0]
    H = hm.ellblock_from_ellpack(*Hs, 8, 40)                          # 40 block slots: the first product overflows
    res, st = _check_solve(api, oracle_mod, H, N // 2, 1e-8, 0.0)
    assert res.status == -3
    I = hm.ellblock_from_dense(2.0 * np.eye(32), 8, 4)
    _, r = api.bml_sp2_ellblock(*gpu(I), 16, 1e-10, 0.0)
    assert r.status == -2


def test_ellblock_runs_are_bit_reproducible(api):
    import torch

    Hs = sparse_model((8, 8, 16))
    N = Hs[0].shape[0]
    H = gpu(hm.ellblock_from_ellpack(*Hs, 8, N // 8))
    solver = api.EllblockSolver(N // 8, N // 8, 8)
    (dv, di, dn), r0 = solver.solve(*H, N // 2, 1e-8, 1e-6)
    first = (dv.clone(), di.clone(), dn.clone())
    for _ in range(5):
        (dv, di, dn), r = solver.solve(*H, N // 2, 1e-8, 1e-6)
        assert torch.equal(dv, first[0]) and torch.equal(di, first[1]) and torch.equal(dn, first[2])
        assert r.branch == r0.branch
