"""GPU parity, sparse ELLPACK-R path.  The kernels keep the oracle's canonical accumulation order (ascending slot p
of row i, one fma per contribution), so stored values, column indices and row lengths are compared BIT-EXACTLY; the
reduced scalars (traces, norms) are compared to round-off."""
import numpy as np
import pytest

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


def to_gpu(X):
    import torch

    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in X)


def to_cpu(X):
    return tuple(a.cpu().numpy() for a in X)


def assert_ell_equal(A, B):
    assert np.array_equal(A[2], B[2]), "row lengths differ"
    assert np.array_equal(A[1], B[1]), "column indices differ"
    assert np.array_equal(A[0], B[0]), "stored values differ (expected bit-exact)"


def rescaled(oracle_mod, H):
    lo, hi = oracle_mod.gershgorin_ellpack(*H)
    xv, xi, xn, bad = oracle_mod.rescale_ellpack(*H, lo, hi)
    assert bad < 0
    return (xv, xi, xn), lo, hi


def test_gershgorin_and_trace_ellpack(api, oracle_mod):
    H = hm.small_sparse_model((7, 7, 8), M=160)
    lo, hi = oracle_mod.gershgorin_ellpack(*H)
    b = api.bml_gershgorin(to_gpu(H)).cpu().numpy()
    assert (b[0], b[1]) == (lo, hi)
    assert abs(api.bml_trace(to_gpu(H)).item() - oracle_mod.trace_ellpack(*H)) < 1e-10


@pytest.mark.parametrize("L,M", [((7, 7, 8), 400), ((8, 7, 9), 512)])
@pytest.mark.parametrize("tau", [0.0, 1e-6, 1e-3])
@pytest.mark.parametrize("branch", [0, 1])
def test_x2_ellpack_one_product_bit_exact(api, oracle_mod, L, M, tau, branch):
    H = hm.small_sparse_model(L, M=M)
    X, _, _ = rescaled(oracle_mod, H)
    pv, pi, pn, bad, mx = oracle_mod.x2_ellpack(*X, tau)
    assert bad < 0
    if branch:
        ev, ei, en, bad, mxu = oracle_mod.update_ellpack(X, (pv, pi, pn), tau)
        assert bad < 0
        mx = max(mx, mxu)
    else:
        ev, ei, en = pv, pi, pn
    out, sums, info = api.bml_x2_ellpack(to_gpu(X), branch, tau)
    assert_ell_equal(to_cpu(out), (ev, ei, en))
    info = info.cpu().numpy()
    assert info[0] == np.iinfo(np.int32).max and info[1] == np.iinfo(np.int32).max and info[2] == mx
    Xd, Pd, Ed = (hm.ellpack_to_dense(*A) for A in (X, (pv, pi, pn), (ev, ei, en)))
    ref = np.array([np.trace(Pd), np.linalg.norm(Pd - Xd) ** 2, np.linalg.norm(Xd) ** 2, np.trace(Ed)])
    assert np.allclose(sums.cpu().numpy(), ref, rtol=1e-12, atol=1e-15)


def test_x2_ellpack_rows_that_outgrow_the_small_table_go_to_the_large_one(api, oracle_mod):
    """Kernel 1 runs 2048-slot tables behind an exact pre-screen (bound per 32-column block from the block maxima of
    X) and hands rows that still do not fit to the 4096-slot instance.  Here every 32-column block a row touches holds
    one entry of magnitude 0.05 - 0.1 and a few of 1e-5 (random signs), tau = 1e-6: the block bounds all pass, so the
    screen removes nothing; the first rows reach ~2100 distinct columns j >= i (more than the small table holds, fewer
    than the large one), the last rows a handful -- both instances run -- and only the large x large products survive
    the threshold, so the rows fit M.  Bit-exact against the oracle, both branches."""
    rng = np.random.default_rng(11)
    N, M, tau = 8192, 512, 1e-6
    A = np.zeros((N, N))
    nb = N // 32
    for i in range(N):
        for b in rng.choice(nb, 7, replace=False):
            cols = b * 32 + rng.choice(32, 8, replace=False)
            A[i, cols[0]] = rng.choice([-1.0, 1.0]) * rng.uniform(0.05, 0.1)
            A[i, cols[1:]] = rng.choice([-1.0, 1.0], 7) * 1e-5
    A = np.triu(A, 1)
    A = A + A.T + np.diag(rng.uniform(0.3, 0.7, N))
    X = hm.ellpack_from_dense(A, M)
    assert X[2].max() <= M
    pv, pi, pn, bad, mx = oracle_mod.x2_ellpack(*X, tau)
    assert bad < 0
    # the construction does what the docstring says: the upper part of row 0 outgrows 2048 slots before thresholding
    touched = np.unique(np.concatenate([X[1][k, : X[2][k]] for k in X[1][0, : X[2][0]]]))
    assert 2048 < touched.size < 4096
    for branch in (0, 1):
        if branch:
            ev, ei, en, bad_u, _ = oracle_mod.update_ellpack(X, (pv, pi, pn), tau)
            assert bad_u < 0
        else:
            ev, ei, en = pv, pi, pn
        out, sums, info = api.bml_x2_ellpack(to_gpu(X), branch, tau)
        assert_ell_equal(to_cpu(out), (ev, ei, en))
        info = info.cpu().numpy()
        assert info[0] == np.iinfo(np.int32).max and info[1] == np.iinfo(np.int32).max


def test_x2_ellpack_second_iterate_wider_rows(api, oracle_mod):
    """Rows after one product are several times wider (pre-threshold fill in the thousands at full size): run a
    second product on the oracle's X_1."""
    H = hm.small_sparse_model((12, 10, 8), M=512)
    X, _, _ = rescaled(oracle_mod, H)
    P = oracle_mod.x2_ellpack(*X, 1e-6)[:3]
    X1 = oracle_mod.update_ellpack(X, P, 1e-6)[:3]
    ref = oracle_mod.x2_ellpack(*X1, 1e-6)
    assert ref[3] < 0
    out, _, info = api.bml_x2_ellpack(to_gpu(X1), 0, 1e-6)
    assert_ell_equal(to_cpu(out), ref[:3])


def test_x2_ellpack_overflow_and_threshold_edges(api, oracle_mod):
    import torch

    # entry exactly tau is kept, tau - ulp dropped, small diagonal kept (readings item 8)
    N, M = 4, 4
    tau = 0.25
    A = np.zeros((N, N))
    A[0, 0] = 0.5; A[0, 1] = 0.5; A[1, 0] = 0.5; A[1, 1] = 1e-3
    A[2, 2] = 0.5; A[3, 3] = np.nextafter(0.5, 0)
    X = hm.ellpack_from_dense(A, M)
    ref = oracle_mod.x2_ellpack(*X, tau)
    out, _, _ = api.bml_x2_ellpack(to_gpu(X), 0, tau)
    assert_ell_equal(to_cpu(out), ref[:3])
    # overflow: row fill after the product exceeds M
    H = hm.small_sparse_model((7, 7, 8), M=160)
    X, _, _ = rescaled(oracle_mod, H)
    ref = oracle_mod.x2_ellpack(*X, 0.0)
    assert ref[3] >= 0
    _, _, info = api.bml_x2_ellpack(to_gpu(X), 0, 0.0)
    info = info.cpu().numpy()
    assert info[0] == ref[3] and info[2] == ref[4]


def _check_solve(api, oracle_mod, H, n_occ, tol, tau, max_products=100):
    D_ref, st = oracle_mod.sp2_ellpack(*H, n_occ, tol, tau, max_products)
    D, res = api.bml_sp2_ellpack(*to_gpu(H), n_occ, tol, tau, max_products)
    assert res.status == st["status"]
    assert res.n_products == st["n_products"] and res.m_star == st["m_star"]
    assert res.branch == st["branch"]
    assert (res.emin, res.emax) == (st["emin"], st["emax"])
    assert np.allclose(res.trace, st["trace"], rtol=0, atol=1e-9)
    assert np.array_equal(res.max_row_nnz, st["max_row_nnz"])
    if res.status >= 0:          # on an ELLPACK overflow the oracle stops before it evaluates e_m
        assert np.allclose(res.idem, st["idem"], rtol=1e-6, atol=1e-14)
        assert_ell_equal(to_cpu(D), D_ref)
    return res, st


@pytest.mark.parametrize("L,M,tau,tol", [((12, 10, 8), 512, 1e-6, 1e-8), ((7, 7, 8), 392, 0.0, 1e-10),
                                         ((12, 10, 8), 512, 1e-4, 1e-8)])
def test_sp2_ellpack_small_model_parity(api, oracle_mod, L, M, tau, tol):
    """tau = 0 with M = N (nothing dropped, no overflow possible) is the dense recursion in sparse storage."""
    H = hm.small_sparse_model(L, M=M)
    res, _ = _check_solve(api, oracle_mod, H, H[0].shape[0] // 2, tol, tau)
    assert res.status in (0, 1)


def test_sp2_ellpack_unsorted_input_rows(api, oracle_mod):
    """input rows may be in any order; D is identical (canonical order is restored by the rescale step)."""
    H = hm.small_sparse_model((7, 7, 8), M=400)
    rng = np.random.default_rng(3)
    v, i, n = (a.copy() for a in H)
    for r in range(v.shape[0]):
        perm = rng.permutation(n[r])
        v[r, : n[r]] = v[r, perm]
        i[r, : n[r]] = i[r, perm]
    _check_solve(api, oracle_mod, (v, i, n), v.shape[0] // 2, 1e-8, 1e-6)


def test_sp2_ellpack_missing_diagonal_is_inserted(api, oracle_mod):
    H = hm.small_sparse_model((7, 7, 8), M=400)
    v, i, n = (a.copy() for a in H)
    # drop the stored diagonal of row 5 (H_55 := 0, not stored)
    p = int(np.nonzero(i[5, : n[5]] == 5)[0][0])
    v[5, p:n[5] - 1] = v[5, p + 1:n[5]]; i[5, p:n[5] - 1] = i[5, p + 1:n[5]]
    n[5] -= 1
    v[5, n[5]] = 0.0; i[5, n[5]] = 0
    _check_solve(api, oracle_mod, (v, i, n), v.shape[0] // 2, 1e-8, 1e-6)


def test_sp2_ellpack_overflow_status(api, oracle_mod):
    H = hm.small_sparse_model((7, 7, 8), M=160)
    res, st = _check_solve(api, oracle_mod, H, H[0].shape[0] // 2, 1e-8, 0.0)
    assert res.status == -3 and res.overflow_row == st["overflow_row"]


def test_config5_literal_overflows_at_product0(api):
    """BASELINE.json configs[4] exactly as written: X_0^2 has 829 entries per row, all >= 1e-6 -> ELLPACK-R overflow
     at product 0.  The oracle side of this statement is tests/test_oracle_pins.py."""
    w = hm.WORKLOADS["ellpack_n65536_literal"]
    H = hm.make_ellpack("ellpack_n65536_literal")
    D, res = api.bml_sp2_ellpack(*to_gpu(H), w.n_occ, w.idem_tol, w.drop_tol)
    assert res.status == -3 and res.n_products == 1 and res.overflow_row == 0
    assert res.max_row_nnz[0] == 829


def test_config5prime_full_size_sampled_rows_and_invariants(api, oracle_mod):
    """The labelled fallback 5' at N=65536: (a) one fused product on the oracle's X_0 compared bit-exactly
    with the oracle (the oracle's row merge at this size takes seconds per product); (b) the full solve checked
    through its invariants and the expected branch string."""
    import torch

    w = hm.WORKLOADS["ellpack_n65536"]
    H = hm.make_ellpack("ellpack_n65536")
    X, lo, hi = rescaled(oracle_mod, H)
    ref = oracle_mod.x2_ellpack(*X, w.drop_tol)
    out, _, info = api.bml_x2_ellpack(to_gpu(X), 0, w.drop_tol)
    assert_ell_equal(to_cpu(out), ref[:3])
    D, res = api.bml_sp2_ellpack(*to_gpu(H), w.n_occ, w.idem_tol, w.drop_tol)
    assert res.status == 1                      # stops on the tau = 1e-6 truncation floor (S2)
    assert (res.emin, res.emax) == (lo, hi)
    import json
    import os

    g = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "sp2_expected.json")))
    g = g["ellpack_n65536"]                      # written by tests/golden/make_golden.py from the oracle
    assert res.branch == g["branch"] and res.n_products == g["n_products"] == 12
    dv, di, dn = D
    rows = torch.arange(w.N, device="cuda").unsqueeze(1)
    mask = torch.arange(w.M, device="cuda").unsqueeze(0) < dn.unsqueeze(1)
    tr = dv[(di == rows) & mask].sum().item()
    assert abs(tr - w.n_occ) < 1e-3
    assert int(dn.max()) <= w.M and int(dn.min()) >= 1
    # canonical order: columns strictly ascending within each row
    d = (di[:, 1:] - di[:, :-1])[mask[:, 1:]]
    assert bool((d > 0).all())
