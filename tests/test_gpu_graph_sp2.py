"""GPU parity of the graph-based construction with SP2 as the local solver (bml_graph_sp2_ellpack; PAPER.md VIII.B
Listing 11 with prg_build_DM = SP2 of IV.A; reading G3': one SP2 polynomial for all parts) against oracle/graph.py
graph_sp2, through the C ABI.

Bit-exact: bounds, branch string, product count, status, part sizes, the pattern of D at drop_tol = 0.
Floating point: traces to 1e-9, e_m to 1e-6 relative, values of D to 1e-10 of the largest entry (the FP64 tolerance
of north_star); with a positive drop_tol the keep decision |v| >= drop_tol is the GPU's own and is checked to be valid
where it differs from the oracle's (the value must then sit within round-off of the threshold)."""
import math

import numpy as np
import pytest

from oracle import graph as og
from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu
TOL_D = 1e-10


@pytest.fixture(scope="module")
def api():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2401_13772_b200 import api as a

    a.load()
    return a


def gapped_model(L=(8, 6, 5), M=64, seed=0, rmax=2.0):
    return hm.lattice_ellpack(L, 12.0, 0.2, rmax, lambda r: -math.exp(-r / 0.5), M, seed)


def gpu(ell):
    import torch

    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in ell)


def tgpu(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check(api, H, offs, nodes, graph_tol, n_occ, tol, drop_tol, M_out, cap=None, max_products=100):
    N = H[0].shape[0]
    (rv, ri, rn), info = og.graph_sp2(*H, offs, nodes, graph_tol, n_occ, tol, drop_tol, max_products, M_out=M_out)
    cap = cap or max(info["part_sizes"])
    (dv, di, dn), res = api.bml_graph_sp2_ellpack(gpu(H), tgpu(offs), tgpu(nodes), graph_tol, n_occ, tol, drop_tol, M_out,
                                                  cap, max_products)
    assert res.status == info["status"], (res.message, info["status"])
    assert res.part_size == info["part_sizes"] and res.core_size == info["core_sizes"]
    if info["status"] == -3:
        assert res.overflow_row == info["overflow_row"]
        return res, info
    s = res.sp2
    assert (s.emin, s.emax) == (info["emin"], info["emax"])
    assert s.branch == info["branch"] and s.n_products == info["n_products"] and s.m_star == info["m_star"]
    np.testing.assert_allclose(s.trace, info["trace"], rtol=0, atol=1e-9)
    np.testing.assert_allclose(s.idem, info["idem"], rtol=1e-6, atol=1e-15)
    dv, di, dn = dv.cpu().numpy(), di.cpu().numpy(), dn.cpu().numpy()
    scale = np.abs(rv).max()
    if drop_tol == 0.0:
        assert np.array_equal(dn, rn) and np.array_equal(di, ri)
        assert np.abs(dv - rv).max() <= TOL_D * scale
    else:
        D, R = hm.ellpack_to_dense(dv, di, dn, N), hm.ellpack_to_dense(rv, ri, rn, N)
        differ = (D != 0) != (R != 0)
        assert np.abs(D - R)[~differ].max() <= TOL_D * scale
        # where the patterns differ the entry was within round-off of the threshold on one side
        assert np.all(np.abs(np.abs(np.where(D != 0, D, R)[differ]) - drop_tol) <= TOL_D * scale)
    return res, info


def test_single_part_equals_dense_sp2(api, oracle_mod):
    """One part covering everything: the batched kernel must walk the dense SP2 iterates (oracle sp2_dense)."""
    H = gapped_model()
    N = H[0].shape[0]
    offs, nodes = og.regular_partition(N, 1)
    res, info = check(api, H, offs, nodes, 0.0, N // 2, 1e-10, 0.0, N)
    _, st = oracle_mod.sp2_dense(hm.ellpack_to_dense(*H), N // 2, 1e-10)
    assert res.sp2.branch == st["branch"] and res.status == 0


@pytest.mark.parametrize("graph_tol", [0.2, 0.02, 0.002])
def test_unequal_parts_match_the_oracle(api, graph_tol):
    """Four parts of unequal core sizes (an irregular cut of the index list); halos of one, two, all stored hops."""
    H = gapped_model((12, 6, 5))
    N = H[0].shape[0]
    offs = np.array([0, 50, 170, 171, N], dtype=np.int32)          # cores of 50, 120, 1 and 189 orbitals
    nodes = np.arange(N, dtype=np.int32)
    res, info = check(api, H, offs, nodes, graph_tol, N // 2, 1e-9, 0.0, N)
    assert len(set(res.part_size)) > 1 and res.status in (0, 1)


def test_permuted_cores_and_drop_tolerance(api):
    """A core partition that is a random permutation of the nodes (parts interleave in index space) and a positive
    drop tolerance on D."""
    H = gapped_model((12, 6, 5))
    N = H[0].shape[0]
    offs, _ = og.regular_partition(N, 5)
    nodes = np.random.default_rng(3).permutation(N).astype(np.int32)
    check(api, H, offs, nodes, 0.05, N // 2, 1e-9, 1e-6, 256)


def test_parts_that_span_several_tiles(api):
    """Parts of several hundred orbitals (several 128 x 128 tiles each, ragged edges), so that tiles are cut by the
    stream-K range boundaries and handed over between CTAs."""
    H = gapped_model((16, 8, 8), M=64)
    N = H[0].shape[0]                                               # 1024
    offs = np.array([0, 300, 301, 700, N], dtype=np.int32)
    nodes = np.arange(N, dtype=np.int32)
    res, info = check(api, H, offs, nodes, 0.02, N // 2, 1e-10, 0.0, N)
    assert max(res.part_size) > 384 and res.status == 0


def test_statuses(api):
    import torch

    H = gapped_model()
    N = H[0].shape[0]
    offs, nodes = og.regular_partition(N, 2)
    check(api, H, offs, nodes, 0.02, N // 2, 1e-9, 0.0, 8)                        # rows of D overflow 8 slots: -3
    res, info = check(api, H, offs, nodes, 0.02, N // 2, 1e-9, 0.0, N, max_products=3)
    assert res.status == 2 and res.sp2.n_products == 3                             # S3
    # part capacity too small: -7, sizes still reported
    (_, _, _), r = api.bml_graph_sp2_ellpack(gpu(H), tgpu(offs), tgpu(nodes), 0.02, N // 2, 1e-9, 0.0, N, 16)
    assert r.status == -7 and r.max_part_size > 16
    # degenerate bounds: -2
    I = hm.ellpack_from_dense(2.0 * np.eye(6), 4)
    (_, _, _), r = api.bml_graph_sp2_ellpack(gpu(I), tgpu(np.array([0, 6], dtype=np.int32)),
                                             tgpu(np.arange(6, dtype=np.int32)), 0.0, 3, 1e-9, 0.0, 6, 6)
    assert r.status == -2


def test_runs_are_bit_reproducible(api):
    import torch

    H = gapped_model((16, 8, 8), M=64)
    N = H[0].shape[0]
    offs = np.array([0, 300, 301, 700, N], dtype=np.int32)
    nodes = np.arange(N, dtype=np.int32)
    solver = api.GraphSp2Solver(N, N, 4, 700)
    Hg, og_, ng = gpu(H), tgpu(offs), tgpu(nodes)
    (dv, _, _), r0 = solver.solve(Hg, og_, ng, 0.02, N // 2, 1e-10, 0.0)
    first = dv.clone()
    for _ in range(10):
        (dv, _, _), r = solver.solve(Hg, og_, ng, 0.02, N // 2, 1e-10, 0.0)
        assert torch.equal(dv, first) and r.sp2.branch == r0.sp2.branch
