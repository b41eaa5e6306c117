"""GPU parity of the graph-based density-matrix path (include/bml_graph.h; PAPER.md VIII.B, Eq. 15, Listing 11)
against oracle/graph.py, through the C ABI.

Index work (node lists, core flags, patterns, row lengths) is compared bit for bit; gathered sub-matrices bit for bit
(a copy); values of D within the Chebyshev path's tolerance relative to the largest entry, with the
drop decision |v| >= drop_tol taken on the GPU's value and checked to be valid where it differs from the oracle's."""
import math

import numpy as np
import pytest

from oracle import chebyshev as och
from oracle import graph as og
from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2401_13772_b200 import api as a

    a.load()
    return a


def model(L=(8, 6, 6), rmax=2.0, decay=1.0, delta=1.5, M=64, seed=0):
    return hm.lattice_ellpack(L, delta, 0.2, rmax, lambda r: -math.exp(-r / decay), M, seed)


def gpu(ell):
    import torch

    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in ell)


def tgpu(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def shuffled_rows(H, seed=0):
    """The same matrix with the entries of every row in a random order (input rows may be unsorted)."""
    v, i, n = (a.copy() for a in H)
    rng = np.random.default_rng(seed)
    for r in range(v.shape[0]):
        perm = rng.permutation(int(n[r]))
        v[r, : n[r]] = v[r, perm]
        i[r, : n[r]] = i[r, perm]
    return v, i, n


@pytest.mark.parametrize("tau", [0.0, 0.1, 0.2, 0.5])
@pytest.mark.parametrize("P", [1, 3, 8])
def test_core_halo_lists_are_bit_exact(api, tau, P):
    H = shuffled_rows(model(L=(9, 7, 6), rmax=2.0))
    N = H[0].shape[0]
    offs, nodes = og.regular_partition(N, P)
    # an irregular partition too: a random permutation of the nodes cut at the same offsets
    for core_nodes in (nodes, np.random.default_rng(P).permutation(N).astype(np.int32)):
        got_nodes, got_core, sizes = api.bml_graph_core_halo(gpu(H), tgpu(offs), tgpu(core_nodes), tau)
        got_nodes, got_core, sizes = got_nodes.cpu().numpy(), got_core.cpu().numpy(), sizes.cpu().numpy()
        for p in range(P):
            ref_nodes, ref_core = og.core_halo(*H, core_nodes[offs[p]: offs[p + 1]], tau)
            s = ref_nodes.size
            assert sizes[p, 0] == s and sizes[p, 1] == offs[p + 1] - offs[p]
            assert np.array_equal(got_nodes[p, :s], ref_nodes)
            assert np.array_equal(got_core[p, :s].astype(bool), ref_core)


def test_matrix2submatrix_is_a_bit_exact_gather(api):
    H = shuffled_rows(model(L=(9, 7, 6), rmax=2.0), seed=1)
    N = H[0].shape[0]
    rng = np.random.default_rng(2)
    for s in (1, 2, 31, 200, N):
        nodes = np.sort(rng.choice(N, s, replace=False)).astype(np.int32)
        got = api.bml_matrix2submatrix_ellpack(gpu(H), tgpu(nodes)).cpu().numpy()
        assert np.array_equal(got, og.matrix2submatrix(*H, nodes))


@pytest.mark.parametrize("M_out,drop", [(64, 1e-3), (300, 0.0), (8, 1e-3)])
def test_submatrix2matrix_is_a_bit_exact_scatter(api, M_out, drop):
    import torch

    rng = np.random.default_rng(5)
    N, s = 400, 300
    nodes = np.sort(rng.choice(N, s, replace=False)).astype(np.int32)
    is_core = rng.random(s) < 0.4
    d = rng.normal(size=(s, s)) * 10.0 ** rng.uniform(-6, 0, size=(s, s))
    dv, di, dn = np.zeros((N, M_out)), np.zeros((N, M_out), dtype=np.int32), np.zeros(N, dtype=np.int32)
    bad = og.submatrix2matrix(d, nodes, is_core, drop, dv, di, dn)
    D = (torch.full((N, M_out), 7.0, dtype=torch.float64, device="cuda"),
         torch.full((N, M_out), 7, dtype=torch.int32, device="cuda"), torch.zeros(N, dtype=torch.int32, device="cuda"))
    ov = api.bml_submatrix2matrix_ellpack(tgpu(d), tgpu(nodes), tgpu(is_core.astype(np.uint8)), drop, D)
    ov = int(ov.item())
    assert (ov == 2**31 - 1 and bad == -1) or ov == bad
    gv, gi, gn = (a.cpu().numpy() for a in D)
    for a, i in enumerate(nodes):
        if is_core[a] and dn[i] > 0:
            assert gn[i] == dn[i] and np.array_equal(gi[i], di[i]) and np.array_equal(gv[i], dv[i])
    untouched = np.ones(N, dtype=bool)
    untouched[nodes[is_core]] = False
    assert (gv[untouched] == 7.0).all() and (gn[untouched] == 0).all()


def check_graph_solve(api, H, P, tau, mu, beta, k, m, drop, M_out, core_nodes=None):
    N = H[0].shape[0]
    offs, nodes = og.regular_partition(N, P)
    if core_nodes is not None:
        nodes = core_nodes
    (rv, ri, rn), info = og.graph_fermi(*H, offs, nodes, tau, mu, beta, k, m, drop, M_out=M_out)
    cap = max(info["part_sizes"])
    (gv, gi, gn), res = api.bml_graph_chebyshev_ellpack(gpu(H), tgpu(offs), tgpu(nodes), tau, mu, beta, k, m, drop, M_out,
                                                       cap)
    assert res.status == info["status"]
    assert res.part_size == info["part_sizes"] and res.core_size == list(np.diff(offs))
    assert res.n_products == P * (k + m - 2)
    if info["status"] != 0:
        assert res.overflow_row == info["overflow_row"]
        return res
    gv, gi, gn = gv.cpu().numpy(), gi.cpu().numpy(), gn.cpu().numpy()
    Dg, Dr = hm.ellpack_to_dense(gv, gi, gn), hm.ellpack_to_dense(rv, ri, rn)
    scale = np.abs(Dr).max()
    assert np.abs(Dg - Dr).max() <= 1e-11 * scale + (drop if drop > 0 else 0.0) * 1.000001
    if drop == 0.0:
        assert np.array_equal(gn, rn) and np.array_equal(gi, ri)
    else:
        # a drop decision may differ only for entries within round-off of the threshold
        diff = (Dg != 0) != (Dr != 0)
        assert (np.abs(np.abs(np.where(Dg != 0, Dg, Dr)[diff]) - drop) <= 1e-11 * scale).all()
    for r in range(N):
        assert (np.diff(gi[r, : gn[r]]) > 0).all() and (gv[r, gn[r]:] == 0).all() and (gi[r, gn[r]:] == 0).all()
    return res


@pytest.mark.parametrize("P,tau", [(1, 0.0), (2, 0.2), (4, 0.1), (4, 0.5), (7, 0.04)])
def test_graph_chebyshev_against_the_oracle(api, P, tau):
    H = shuffled_rows(model(L=(16, 6, 6), rmax=2.0), seed=3)
    check_graph_solve(api, H, P, tau, 0.0, 1.0, 8, 8, 0.0, 600)


def test_graph_chebyshev_with_drop_threshold_and_irregular_partition(api):
    H = model(L=(16, 6, 6), rmax=2.0)
    N = H[0].shape[0]
    core_nodes = np.random.default_rng(0).permutation(N).astype(np.int32)
    check_graph_solve(api, H, 5, 0.1, 0.1, 1.5, 8, 8, 1e-5, 600)
    check_graph_solve(api, H, 5, 0.1, 0.1, 1.5, 8, 8, 1e-5, 600, core_nodes=core_nodes)


def test_graph_overflow_and_capacity_statuses(api):
    H = model(L=(16, 6, 6), rmax=2.0)
    N = H[0].shape[0]
    res = check_graph_solve(api, H, 4, 0.1, 0.0, 1.0, 8, 8, 0.0, 40)          # rows are as long as a part: > 40
    assert res.status == -3 and res.overflow_row >= 0
    offs, nodes = og.regular_partition(N, 4)
    (_, _, _), res = api.bml_graph_chebyshev_ellpack(gpu(H), tgpu(offs), tgpu(nodes), 0.1, 0.0, 1.0, 8, 8, 0.0, 600, 100)
    assert res.status == -7 and res.max_part_size > 100


def test_graph_approaches_the_dense_expansion_as_the_halo_grows(api):
    """End to end on the GPU only: graph-based D against bml_chebyshev_dense of the whole matrix (itself oracle-checked):
    the difference is the graph approximation and falls with graph_tol (Fig. 8's trend)."""
    import torch

    H = model(L=(24, 7, 7), rmax=3.0, M=128)
    N = H[0].shape[0]
    Hd = hm.ellpack_to_dense(*H)
    D_full, r = api.bml_chebyshev_dense(tgpu(Hd), 0.0, 3.0, 16, 16)
    assert r.status == 0
    D_full = D_full.cpu().numpy()
    offs, nodes = og.regular_partition(N, 3)
    errs = []
    for tau in (0.5, 0.2, 0.04):
        (gv, gi, gn), res = api.bml_graph_chebyshev_ellpack(gpu(H), tgpu(offs), tgpu(nodes), tau, 0.0, 3.0, 16, 16, 0.0, 700,
                                                           700)
        assert res.status == 0
        Dg = hm.ellpack_to_dense(gv.cpu().numpy(), gi.cpu().numpy(), gn.cpu().numpy())
        errs.append(np.linalg.norm(Dg - D_full) / np.linalg.norm(D_full))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 0.2 * errs[0]


def test_graph_table2_size_workload(api):
    """The workload bench.py times (graph_n12800: the sizes of the paper's Table II, P:527-538 -- 4 parts, core 3200,
    core+halo 5600).  The plain-series oracle cannot finish a 5600-node part in test time, so: index work against the
    oracle exactly (part sizes), D through properties and against the dense expansion of the WHOLE matrix computed by
    bml_chebyshev_dense (itself oracle-checked at the sizes the oracle reaches): the difference is the graph
    approximation, 1e-5 relative on the small variant of the same model."""
    import torch

    w = hm.WORKLOADS["graph_n12800"]
    H = hm.make_ellpack("graph_n12800")
    N = w.N
    offs, nodes = hm.regular_core_partition(N, w.n_parts)
    Hg = gpu(H)
    sizes = api.bml_graph_core_halo(Hg, tgpu(offs), tgpu(nodes), w.graph_tol)[2].cpu().numpy()
    ref_sizes = [og.core_halo(*H, nodes[offs[p]: offs[p + 1]], w.graph_tol)[0].size for p in range(w.n_parts)]
    assert sizes[:, 0].tolist() == ref_sizes == [5600] * 4 and sizes[:, 1].tolist() == [3200] * 4
    (gv, gi, gn), res = api.bml_graph_chebyshev_ellpack(Hg, tgpu(offs), tgpu(nodes), w.graph_tol, w.mu, w.beta, w.k, w.m,
                                                       w.drop_tol, w.M_out, 5600)
    assert res.status == 0 and res.n_products == 4 * 30
    assert int(gn.max()) <= w.M_out and int(gn.min()) >= 1
    # rows ascending, unused slots zero
    mask = torch.arange(w.M_out, device="cuda").unsqueeze(0) < gn.unsqueeze(1)
    assert bool(((gi[:, 1:] > gi[:, :-1]) | ~mask[:, 1:]).all()) and bool((gv[~mask] == 0).all())
    # against the dense expansion of the whole matrix
    Hd = torch.zeros((N, N), dtype=torch.float64, device="cuda")
    hmask = torch.arange(w.M, device="cuda").unsqueeze(0) < Hg[2].unsqueeze(1)
    rows = torch.arange(N, device="cuda").unsqueeze(1).expand(N, w.M)
    Hd[rows[hmask], Hg[1][hmask].long()] = Hg[0][hmask]
    D_full, r = api.bml_chebyshev_dense(Hd, w.mu, w.beta, w.k, w.m)
    assert r.status == 0
    Dg = torch.zeros((N, N), dtype=torch.float64, device="cuda")
    rows = torch.arange(N, device="cuda").unsqueeze(1).expand(N, w.M_out)
    Dg[rows[mask], gi[mask].long()] = gv[mask]
    kept = D_full.abs() >= w.drop_tol
    err = (torch.linalg.norm(Dg - D_full * kept) / torch.linalg.norm(D_full)).item()
    assert err < 1e-4, err
    assert abs(Dg.trace().item() - r.trace) < 1e-3 * N
