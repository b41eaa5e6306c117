"""GPU parity of the Chebyshev / Paterson-Stockmeyer path (include/bml_chebyshev.h; PAPER.md IV.B, Eq. 8-14) against
oracle/chebyshev.py, through the C ABI.

Tolerances (DESIGN.md 5.5 "Error budget"): one product alpha A B + beta C + gamma I is an N-term FP64 dot product per
element in a different summation order than the oracle's BLAS call: |err| <= ~N eps * sum_k |a_ik b_kj|, asserted as
1e-13 relative to that magnitude (N <= 2048).  The resummed expansion (k + m - 2 products of matrices with
||T_i|| <= 1 and |d_ij| < 1 for these inputs) against the plain series Eq. 8: relative Frobenius error <= 1e-11."""
import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

from oracle import chebyshev as och
from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu

TOL_PRODUCT = 1e-13
TOL_D = 1e-11


@pytest.fixture(scope="module")
def api():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2401_13772_b200 import api as a

    a.load()
    return a


def relfro(A, B):
    return np.linalg.norm(A - B) / np.linalg.norm(B)


def commuting_pair(N, seed):
    """Two symmetric commuting matrices: polynomials of one random symmetric matrix with spectrum in [-1, 1]."""
    rng = np.random.default_rng(seed)
    G = rng.normal(size=(N, N)) / np.sqrt(max(N, 1))
    X = (G + G.T) / 2
    X /= max(np.abs(np.linalg.eigvalsh(X)).max(), 1e-30) * 1.01
    A = 2.0 * X @ X - np.eye(N) + 0.3 * X
    B = X @ X @ X - 0.5 * X + 0.1 * np.eye(N)
    A = np.triu(A) + np.triu(A, 1).T
    B = np.triu(B) + np.triu(B, 1).T
    C = rng.normal(size=(N, N))
    C = np.triu(C) + np.triu(C, 1).T
    return A, B, C


def check_product(got, A, B, C, alpha, beta, gamma):
    ref = och.symm_ab(A, B, C, alpha, beta, gamma)
    # the kernel computes the tiles on and above the diagonal and mirrors them: compare that triangle with the
    # oracle's, and require bitwise symmetry
    mag = abs(alpha) * (np.abs(A) @ np.abs(B)) + (abs(beta) * np.abs(C) if C is not None else 0.0) + abs(gamma)
    iu = np.triu_indices(A.shape[0])
    assert (np.abs(got - ref)[iu] <= TOL_PRODUCT * mag[iu] + 1e-300).all()
    assert np.array_equal(got, got.T)


@pytest.mark.parametrize("N", [1, 2, 7, 31, 33, 100, 256, 300, 512, 513, 640, 1000, 1024, 1025, 1283])
def test_symm_ab_one_job(api, N):
    """Sizes spanning the three tile edges (32 / 64 / 128), several tiles, ragged tails and K tails that are not a
    multiple of the 16-column slab; the K-split last wave (stream-K hand-off) is exercised by every size."""
    A, B, C = commuting_pair(N, N)
    slab, n, ld, se = api.matrix_slab([A, B, C, np.zeros((N, N))])
    api.bml_symm_ab_dense(slab, n, ld, [(0, 1, 2, 3, 2.0, -1.0, 0.25)])
    check_product(api.slab_matrix(slab, 3, n, ld).cpu().numpy(), A, B, C, 2.0, -1.0, 0.25)
    # operands untouched
    assert np.array_equal(api.slab_matrix(slab, 0, n, ld).cpu().numpy(), A)
    assert np.array_equal(api.slab_matrix(slab, 1, n, ld).cpu().numpy(), B)


@pytest.mark.parametrize("N", [96, 700, 1500])
def test_symm_ab_square_no_c_and_in_place_c(api, N):
    """a == b (one panel per diagonal tile), no C term (T_{2a} = 2 T_a T_a - I), and C == Out (Eq. 10 in place)."""
    A, B, C = commuting_pair(N, 1000 + N)
    slab, n, ld, se = api.matrix_slab([A, B, C, np.zeros((N, N))])
    api.bml_symm_ab_dense(slab, n, ld, [(0, 0, -1, 3, 2.0, 123.0, -1.0)])
    check_product(api.slab_matrix(slab, 3, n, ld).cpu().numpy(), A, A, None, 2.0, 0.0, -1.0)
    api.bml_symm_ab_dense(slab, n, ld, [(0, 1, 2, 2, 1.0, 1.0, 0.0)])
    check_product(api.slab_matrix(slab, 2, n, ld).cpu().numpy(), A, B, C, 1.0, 1.0, 0.0)


@pytest.mark.parametrize("N,n_jobs", [(64, 16), (300, 3), (520, 8), (1100, 4)])
def test_symm_ab_grouped_launch(api, N, n_jobs):
    """Several products in ONE launch (a doubling level of Eq. 13-14): the work list runs across jobs."""
    A, B, C = commuting_pair(N, 7 * N)
    mats = [A, B, C] + [np.zeros((N, N))] * n_jobs
    slab, n, ld, se = api.matrix_slab(mats)
    ops = [(0, 1), (1, 0), (0, 0), (1, 1)]
    jobs = []
    for q in range(n_jobs):
        a, b = ops[q % 4]
        jobs.append((a, b, 2 if q % 3 else -1, 3 + q, 1.0 + 0.5 * q, -1.0 + 0.1 * q, 0.01 * q))
    api.bml_symm_ab_dense(slab, n, ld, jobs)
    M = [A, B]
    for q, (a, b, c, o, al, be, ga) in enumerate(jobs):
        check_product(api.slab_matrix(slab, o, n, ld).cpu().numpy(), M[a], M[b], C if c >= 0 else None, al,
                      be if c >= 0 else 0.0, ga)


def test_symm_ab_is_bit_reproducible(api):
    A, B, C = commuting_pair(1283, 5)
    outs = []
    for _ in range(3):
        slab, n, ld, se = api.matrix_slab([A, B, C, np.zeros_like(A)])
        api.bml_symm_ab_dense(slab, n, ld, [(0, 1, 2, 3, 2.0, -1.0, 0.0)])
        outs.append(api.slab_matrix(slab, 3, n, ld).cpu().numpy())
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


def test_grouped_store_only_launches_are_bit_reproducible(api):
    """Regression test of the ring-stage release (dense_fp64_core.cuh StageRelease): grouped launches of products with
    no C term have a store-only epilogue, the consumers then run close behind the TMA producer, and a stage released
    before its last fragment loads had completed used to be refilled under them -- about 1 launch in 20 at N = 4000
    came back with a few wrong 32-byte fragment chunks.  150 launches x 8 jobs must be bitwise identical."""
    import torch

    N = 2048
    rng = np.random.default_rng(11)
    G = rng.normal(size=(N, N)) / np.sqrt(N)
    X = (G + G.T) / 4
    X2 = X @ X
    mats = [X, np.triu(X2) + np.triu(X2, 1).T, np.eye(N) - X] + [np.zeros((N, N))] * 8
    slab, n, ld, se = api.matrix_slab(mats)
    ws = api._workspace(api.load().bml_symm_ab_workspace_bytes(), "cuda")
    ops = [(0, 0), (1, 0), (1, 1), (2, 1), (2, 2), (0, 2), (1, 2), (0, 1)]
    jobs = [(a, b, -1, 3 + q, 2.0, 0.0, -1.0) for q, (a, b) in enumerate(ops)]
    api.bml_symm_ab_dense(slab, n, ld, jobs, ws)
    ref = slab[3:].clone()
    check_product(api.slab_matrix(slab, 4, n, ld).cpu().numpy(), mats[1], mats[0], None, 2.0, 0.0, -1.0)
    for it in range(150):
        api.bml_symm_ab_dense(slab, n, ld, jobs, ws)
        assert torch.equal(slab[3:], ref), f"launch {it} differs"


def test_symm_ab_rejects_bad_arguments(api):
    A, B, C = commuting_pair(40, 1)
    slab, n, ld, se = api.matrix_slab([A, B, C])
    with pytest.raises(RuntimeError):
        api.bml_symm_ab_dense(slab, n, ld, [(0, 1, 2, 0, 1.0, 1.0, 0.0)])       # output is an operand
    with pytest.raises(RuntimeError):
        api.bml_symm_ab_dense(slab, n, ld, [(0, 1, 2, 3, 1.0, 1.0, 0.0)])       # slot out of range
    with pytest.raises(RuntimeError):
        api.bml_symm_ab_dense(slab, n, ld, [])
    with pytest.raises(RuntimeError):
        api.bml_symm_ab_dense(slab, n, ld, [(0, 1, -1, 2, 1.0, 0.0, 0.0)] * 2)  # two jobs write one slot


# ------------------------------------------------ the expansion ---------------------------------------------
def to_gpu(A):
    import torch

    return torch.from_numpy(np.ascontiguousarray(A)).cuda()


def check_solve(api, H, mu, beta, k, m):
    D_ref, info = och.chebyshev_serial(H, mu, beta, k * m - 1)
    D, res = api.bml_chebyshev_dense(to_gpu(H), mu, beta, k, m)
    assert res.status == 0
    assert res.n_products == k + m - 2 and res.L == k * m - 1
    assert res.emin == pytest.approx(info["emin"], rel=1e-14) and res.emax == pytest.approx(info["emax"], rel=1e-14)
    assert np.max(np.abs(res.c - info["c"])) <= 1e-13
    # d_{i,j}: (a) as a representation of the same polynomial: Eq. 10 evaluated on scalars = Eq. 8; (b) entry by entry
    # within the conditioning of the division by T_k: writing a degree-(m-1) Chebyshev series in y = T_k in powers of y
    # amplifies the last-bit differences of c_n (device vs numpy exp / cos) by up to (1 + sqrt 2)^(m-1) -- measured
    # 3e-10 at m = 16 -- without harming (a), which is what the matrices see
    x = np.linspace(-1.0, 1.0, 401)
    assert np.max(np.abs(och.ps_eval_scalar(res.d, x) - npcheb.chebval(x, info["c"]))) <= 1e-12
    assert np.max(np.abs(res.d - och.ps_coeffs(info["c"], k))) <= 1e-13 + 2e-15 * (1.0 + np.sqrt(2.0)) ** (m - 1)
    Dg = D.cpu().numpy()
    assert relfro(Dg, D_ref) <= TOL_D
    assert np.array_equal(Dg, Dg.T)
    assert abs(res.trace - np.trace(D_ref)) <= 1e-10 * H.shape[0]
    assert res.trace == pytest.approx(np.trace(Dg), rel=1e-13)
    return Dg, res


@pytest.mark.parametrize("k,m", [(2, 1), (2, 2), (3, 5), (8, 8), (16, 4), (5, 16), (16, 16), (32, 8), (9, 1)])
def test_chebyshev_factorisations(api, k, m):
    """All branches of the launch sequence: m = 1 (no nesting step), k not a power of two (ragged doubling levels),
    k = 32 (16 products in one level), against the plain series Eq. 8 of the same order."""
    H = hm.lattice_dense((6, 5, 5), 0.0, 0.2, 1.0, lambda r: -1.0, seed=3)
    check_solve(api, H, 0.1, 1.5, k, m)


@pytest.mark.parametrize("N", [2, 3, 17, 100, 257, 600, 1100])
def test_chebyshev_sizes(api, N):
    rng = np.random.default_rng(N)
    G = rng.normal(size=(N, N)) / np.sqrt(N)
    H = (G + G.T) / 2 + np.diag(rng.uniform(-1, 1, N))
    check_solve(api, H, 0.05, 2.0, 8, 8)


def test_chebyshev_fig3_size_against_oracle_and_exact(api):
    """The N = 2000 workload bench.py times (Fig. 3 size): element-wise against the oracle, and against the
    LAPACK Fermi operator within the truncation error (1.2e-10 relative measured by the oracle pin at N = 500)."""
    w = hm.WORKLOADS["cheby_n2000"]
    H = hm.make_dense("cheby_n2000")
    D_ref, info = och.chebyshev_ps(H, w.mu, w.beta, w.k, w.m)
    D, res = api.bml_chebyshev_dense(to_gpu(H), w.mu, w.beta, w.k, w.m)
    assert res.status == 0 and res.n_products == 30
    Dg = D.cpu().numpy()
    assert relfro(Dg, D_ref) <= TOL_D
    assert np.array_equal(Dg, Dg.T)
    assert relfro(Dg, och.fermi_exact(H, w.mu, w.beta)) <= 1e-9
    # the launch sequence: 4 doubling levels for k = 16 + 15 nesting steps
    assert res.n_launches == 4 + 15


def test_chebyshev_n4000_properties(api):
    """N = 4000 (the largest Fig. 3 size) through properties that need no O(N^3) CPU work per check beyond one LAPACK
    diagonalisation: D against U f(Lambda) U^T, trace against sum f(eps_i), commutation with H."""
    import torch

    w = hm.WORKLOADS["cheby_n4000"]
    H = hm.make_dense("cheby_n4000")
    Hg = to_gpu(H)
    D, res = api.bml_chebyshev_dense(Hg, w.mu, w.beta, w.k, w.m)
    assert res.status == 0
    assert torch.equal(D, D.T)
    ev = np.linalg.eigvalsh(H)
    assert abs(res.trace - och.fermi(ev, w.mu, w.beta).sum()) <= 1e-6
    assert (torch.linalg.norm(Hg @ D - D @ Hg) / torch.linalg.norm(Hg)).item() < 1e-11
    # f(H)(1 - f(H)) has the spectrum f(1-f) in [0, 1/4]: D is not idempotent at finite temperature, but D - D^2 is PSD
    X = D - D @ D
    assert torch.linalg.eigvalsh(X).min().item() > -1e-9


def test_chebyshev_status_codes(api):
    import torch

    H = to_gpu(np.eye(8) * 3.0)
    D, res = api.bml_chebyshev_dense(H, 0.0, 1.0, 4, 4)
    assert res.status == -2                                   # e_max - e_min = 0
    Hn = hm.lattice_dense((4, 4, 4), 0.0, 0.2, 1.0, lambda r: -1.0, seed=0)
    for k, m in [(1, 4), (33, 2), (4, 0), (4, 33)]:
        assert api.bml_chebyshev_dense(to_gpu(Hn), 0.0, 1.0, k, m)[1].status == -1
    assert api.bml_chebyshev_dense(to_gpu(Hn), 0.0, -1.0, 4, 4)[1].status == -1
    Ha = Hn.copy()
    Ha[1, 2] += 1e-9
    assert api.bml_chebyshev_dense(to_gpu(Ha), 0.0, 1.0, 4, 4, flags=api.FLAG_CHECK_SYMMETRY)[1].status == -5
    assert api.bml_chebyshev_dense(to_gpu(Hn), 0.0, 1.0, 4, 4, flags=api.FLAG_CHECK_SYMMETRY)[1].status == 0


def test_chebyshev_strided_input_and_repeat(api):
    """H with ld > N, and the same solver object reused (workspace flags and epochs start over)."""
    import torch

    H = hm.lattice_dense((7, 6, 5), 0.0, 0.2, 1.0, lambda r: -1.0, seed=9)
    N = H.shape[0]
    big = torch.zeros((N, N + 24), dtype=torch.float64, device="cuda")
    big[:, :N] = to_gpu(H)
    solver = api.ChebyshevSolver(N, 8, 4)
    D1 = solver.solve(big[:, :N], 0.2, 1.0)[0].clone()
    D2 = solver.solve(to_gpu(H), 0.2, 1.0)[0].clone()
    assert torch.equal(D1, D2)
    D_ref, _ = och.chebyshev_serial(H, 0.2, 1.0, 31)
    assert relfro(D1.cpu().numpy(), D_ref) <= TOL_D


def test_chebyshev_graph_replay_on_a_side_stream(api):
    """On a non-default stream small expansions are captured once and replayed as a CUDA graph (chebyshev.cu): the
    replays must give the bits of the plainly enqueued solve, also after the INPUT CONTENT changes under the same
    pointers, and for several shapes alternating in one cache."""
    import torch

    H1 = hm.lattice_dense((7, 6, 5), 0.0, 0.2, 1.0, lambda r: -1.0, seed=1)
    H2 = hm.lattice_dense((7, 6, 5), 0.3, 0.1, 1.0, lambda r: -1.0, seed=2)
    N = H1.shape[0]
    ref1 = api.bml_chebyshev_dense(to_gpu(H1), 0.1, 2.0, 8, 8)[0].clone()     # default stream: plain enqueue
    ref2 = api.bml_chebyshev_dense(to_gpu(H2), 0.1, 2.0, 8, 8)[0].clone()
    side = torch.cuda.Stream()
    solver = api.ChebyshevSolver(N, 8, 8)
    solver_b = api.ChebyshevSolver(N, 4, 4)
    Hbuf = to_gpu(H1)
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        for it in range(6):
            Hbuf.copy_(to_gpu(H1 if it % 2 == 0 else H2))
            D, res = solver.solve(Hbuf, 0.1, 2.0)
            assert res.status == 0 and res.n_launches == 3 + 7
            assert torch.equal(D, ref1 if it % 2 == 0 else ref2), f"replay {it}"
            Db, rb = solver_b.solve(Hbuf, 0.1, 2.0)
            assert rb.status == 0 and rb.n_products == 6
    torch.cuda.synchronize()
    D_ref_b, _ = och.chebyshev_serial(H2, 0.1, 2.0, 15)
    assert relfro(Db.cpu().numpy(), D_ref_b) <= TOL_D
