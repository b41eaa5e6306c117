"""GPU parity, dense path: the CUDA kernels (through the C ABI binding) against the CPU oracle, element by element
on the same seeded inputs.  FP64 tolerance: relative Frobenius error of D <= 1e-10 (BASELINE.json north_star);
branch string and product count bit-exact."""
import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu


def _golden(name):
    import json
    import os

    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "sp2_expected.json")
    gold = json.load(open(path))
    if name not in gold:
        pytest.skip(f"{name} not in the golden file yet (run tests/golden/make_golden.py {name})")
    return gold[name]

TOL_D = 1e-10          # north_star: relFro(D_gpu - D_oracle) <= 1e-10 in FP64
TOL_P = 1e-13          # one product: |P_gpu - P_oracle| <= 1e-13 * ||X||_F-scale (sum of <= 8192 products, eps 1e-16)


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


def to_gpu(A):
    import torch

    return torch.from_numpy(np.ascontiguousarray(A)).cuda()


# ------------------------------------------------------------------------------------------------ D0, trace
@pytest.mark.parametrize("N,ld", [(2, 2), (3, 5), (97, 97), (256, 300), (1000, 1000)])
def test_gershgorin_and_trace_dense(api, oracle_mod, N, ld):
    import torch

    rng = np.random.default_rng(N)
    A = rng.normal(size=(N, N))
    A = A + A.T
    buf = np.zeros((N, ld))
    buf[:, :N] = A
    g = torch.from_numpy(buf).cuda()[:, :N]
    lo, hi = oracle_mod.gershgorin_dense(A)
    b = api.bml_gershgorin(g).cpu().numpy()
    # compensated row sums on both sides: the bounds agree to the last bit
    assert (b[0], b[1]) == (lo, hi)
    t = api.bml_trace(g).item()
    assert abs(t - oracle_mod.trace_dense(A)) <= 1e-13 * np.abs(np.diag(A)).sum()


# ------------------------------------------------------------------------------------------------ D3 + D4
@pytest.mark.parametrize("N", [1, 2, 7, 128, 129, 200, 384, 515, 640, 1000, 1100, 1283])
@pytest.mark.parametrize("branch", [0, 1])
def test_x2_dense_one_product_elementwise(api, oracle_mod, N, branch):
    """One fused product on sizes that span several tiles with ragged tails (and the degenerate N=1,2): 32 x 32 tiles
    up to N = 512, 64 x 64 up to 1024, and above that the persistent 128 x 128 kernel, whose 45 / 66 tiles at
    N = 1100 / 1283 are all split along K across the 148 CTAs (stream-K hand-off of partial accumulators)."""
    rng = np.random.default_rng(1000 + N)
    X = rng.uniform(-1, 1, size=(N, N)) / np.sqrt(N)
    X = np.triu(X) + np.triu(X, 1).T
    P = oracle_mod.x2_dense(X)
    Xg = api.padded_dense(X)
    Xn, sums = api.bml_x2_dense(Xg, branch)
    Xn = Xn.cpu().numpy()
    expect = 2.0 * X - P if branch else P
    scale = max(np.abs(P).max(), np.abs(X).max())
    assert np.abs(Xn - expect).max() <= TOL_P * scale * 10
    assert np.array_equal(Xn, Xn.T), "X' must be bitwise symmetric (mirrored write)"
    s = sums.cpu().numpy()
    ref = np.array([np.trace(P), np.linalg.norm(P - X) ** 2, np.linalg.norm(X) ** 2, np.trace(expect)])
    assert np.allclose(s, ref, rtol=1e-12, atol=1e-14)


def test_x2_dense_rejects_bad_arguments(api):
    import torch

    X = torch.zeros((20, 20), dtype=torch.float64, device="cuda")   # ld = 20 is not a multiple of 16
    with pytest.raises(RuntimeError):
        api.bml_x2_dense(X, 0)


# ------------------------------------------------------------------------------------------------ full SP2
def _check_solve(api, oracle_mod, H, n_occ, tol, max_products=100):
    D_ref, st = oracle_mod.sp2_dense(H, n_occ, tol, max_products)
    D, res = api.bml_sp2_dense(to_gpu(H), n_occ, tol, max_products)
    D = D.cpu().numpy()
    assert res.status == st["status"]
    assert res.n_products == st["n_products"] and res.m_star == st["m_star"]
    assert res.branch == st["branch"], "SP2 branch sequence must match the oracle bit for bit"
    assert (res.emin, res.emax) == (st["emin"], st["emax"])
    assert np.allclose(res.trace, st["trace"], rtol=0, atol=1e-9)
    assert np.allclose(res.idem, st["idem"], rtol=1e-6, atol=1e-14)
    assert relfro(D, D_ref) <= TOL_D
    assert np.array_equal(D, D.T)
    return D, res, st


def test_sp2_worked_2x2_tie_break(api, oracle_mod):
    """tr X_0 == N_occ exactly: the '<=' of Listing 2 must pick 2X - X^2 on the device too."""
    H = np.array([[1.5, -1.0], [-1.0, -1.5]])
    D, res, _ = _check_solve(api, oracle_mod, H, 1, 1e-10)
    assert res.branch == "1001010110" and res.n_products == 11
    assert relfro(D, 0.5 * (np.eye(2) - H / np.sqrt(3.25))) < 1e-10


@pytest.mark.parametrize("N,n_occ,seed", [(3, 1, 0), (33, 11, 3), (100, 37, 5), (333, 200, 6)])
def test_sp2_planted_gap_parity(api, oracle_mod, N, n_occ, seed):
    H, _ = hm.planted_gap(N, n_occ, gap=1.0, width=2.0, seed=seed)
    D, res, _ = _check_solve(api, oracle_mod, H, n_occ, 1e-10)
    assert res.status == 0
    assert abs(np.trace(D) - n_occ) < 1e-8


def test_sp2_config1_n256(api, oracle_mod):
    w = hm.WORKLOADS["dense_n256"]
    H = hm.make_dense("dense_n256")
    _, res, _ = _check_solve(api, oracle_mod, H, w.n_occ, w.idem_tol)
    assert res.branch == "10010110010110" and res.n_products == 15


def test_sp2_small_long_range(api, oracle_mod):
    H = hm.small_long_range((8, 8, 6))
    _check_solve(api, oracle_mod, H, H.shape[0] // 2, 1e-10)


def test_sp2_config2_n2048_full_parity(api, oracle_mod):
    """BASELINE.json configs[1] at full size, in the launch configuration bench.py times."""
    w = hm.WORKLOADS["dense_n2048"]
    H = hm.make_dense("dense_n2048")
    D, res, _ = _check_solve(api, oracle_mod, H, w.n_occ, w.idem_tol)
    assert res.branch == "011010011010010110" and res.n_products == 19
    assert abs(np.trace(D) - w.n_occ) < 1e-8
    assert np.linalg.norm(H @ D - D @ H) / np.linalg.norm(H) < 1e-12      # [H, D] = 0


def test_sp2_status_paths(api, oracle_mod):
    import torch

    # S3: max_products reached
    H = hm.make_dense("dense_n256")
    _, res, _ = _check_solve(api, oracle_mod, H, 128, 1e-10, max_products=5)
    assert res.status == 2 and res.n_products == 5
    _, res, _ = _check_solve(api, oracle_mod, H, 128, 1e-10, max_products=1)
    assert res.status == 2 and res.n_products == 1 and res.branch == ""
    # degenerate bounds
    D, res = api.bml_sp2_dense(torch.eye(8, dtype=torch.float64, device="cuda") * 3.0, 4, 1e-10)
    assert res.status == -2
    # invalid arguments
    Hg = to_gpu(H)
    assert api.bml_sp2_dense(Hg, 0, 1e-10)[1].status == -1
    assert api.bml_sp2_dense(Hg, 256, 1e-10)[1].status == -1
    assert api.bml_sp2_dense(Hg, 128, 0.0)[1].status == -1
    assert api.bml_sp2_dense(Hg, 128, 1e-10, max_products=129)[1].status == -1
    # symmetry check flag
    Hbad = H.copy()
    Hbad[3, 200] += 1e-9
    assert api.bml_sp2_dense(to_gpu(Hbad), 128, 1e-10, flags=api.FLAG_CHECK_SYMMETRY)[1].status == -5
    assert api.bml_sp2_dense(Hg, 128, 1e-10, flags=api.FLAG_CHECK_SYMMETRY)[1].status == 0


def test_sp2_gapless_terminates_like_the_oracle(api, oracle_mod):
    """P:175 'known challenges in the case of a vanishing electronic bandgap': must end in S3, not hang.  Clean ring,
    N_occ = 2 cuts through the degenerate k = +/-1 pair (gap exactly zero); margins here are NOT round-off safe, so
    only termination, status and the product count are compared."""
    H = hm.ring_dense(64, 0.0, 0.0, 0.0)
    D_ref, st = oracle_mod.sp2_dense(H, 2, 1e-10, 60)
    D, res = api.bml_sp2_dense(to_gpu(H), 2, 1e-10, 60)
    assert st["status"] == 2
    assert res.status == 2 and res.n_products == 60 and res.idem[-1] > 1e-2


def test_sp2_strided_input_and_output_reuse(api, oracle_mod):
    """H with ld > N; a DenseSolver reused for two different H of the same size gives independent results."""
    import torch

    N = 200
    H1, _ = hm.planted_gap(N, 80, seed=11)
    H2, _ = hm.planted_gap(N, 80, seed=12)
    buf = torch.zeros((N, 256), dtype=torch.float64, device="cuda")
    buf[:, :N] = torch.from_numpy(H1).cuda()
    solver = api.DenseSolver(N)
    D1, r1 = solver.solve(buf[:, :N], 80, 1e-10)
    D1 = D1.cpu().numpy().copy()
    D2, r2 = solver.solve(to_gpu(H2), 80, 1e-10)
    D2 = D2.cpu().numpy()
    assert relfro(D1, oracle_mod.sp2_dense(H1, 80, 1e-10)[0]) <= TOL_D
    assert relfro(D2, oracle_mod.sp2_dense(H2, 80, 1e-10)[0]) <= TOL_D


# ------------------------------------------------------------------------------------------------ full size, sampled
def test_config3_n8192_one_product_sampled_and_solve_invariants(api, oracle_mod):
    """BASELINE.json configs[2] (N=8192) is beyond what the oracle finishes in seconds: (a) one fused product on the
    oracle's X_0 is compared with the oracle on sampled entries (each a compensated N-term dot product), incl. tile
    corners; (b) the full solve is checked through properties that hold at any size and against the branch string
    of the scalar recursion recorded in BASELINE.md."""
    import torch

    w = hm.WORKLOADS["dense_n8192"]
    H = hm.make_dense("dense_n8192")
    N = w.N
    lo, hi = oracle_mod.gershgorin_dense(H)
    X0 = oracle_mod.rescale_dense(H, lo, hi)
    Xg = api.padded_dense(X0)
    rng = np.random.default_rng(5)
    rows = np.concatenate([rng.integers(0, N, 400), [0, 127, 128, 8191, 8191, 4095, 4096, 300]])
    cols = np.concatenate([rng.integers(0, N, 400), [0, 128, 127, 8191, 0, 4096, 4095, 300]])
    ref = oracle_mod.x2_dense_sampled(X0, rows, cols)
    for branch in (0, 1):
        Xn, sums = api.bml_x2_dense(Xg, branch)
        got = Xn[torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()].cpu().numpy()
        expect = 2.0 * X0[rows, cols] - ref if branch else ref
        assert np.abs(got - expect).max() <= 1e-13
        got_t = Xn[torch.from_numpy(cols).cuda(), torch.from_numpy(rows).cuda()].cpu().numpy()
        assert np.array_equal(got, got_t)
    D, res = api.bml_sp2_dense(to_gpu(H), w.n_occ, w.idem_tol)
    assert res.status == 0
    assert (res.emin, res.emax) == (lo, hi)
    g = _golden("dense_n8192")                   # written by tests/golden/make_golden.py from the oracle
    assert res.branch == g["branch"] and res.n_products == g["n_products"] == 32
    assert abs(torch.trace(D).item() - w.n_occ) < 1e-7
    assert torch.equal(D, D.T)
    D2 = D @ D                                   # torch/cuBLAS used only to CHECK idempotency of the result
    assert (torch.linalg.norm(D2 - D) / torch.linalg.norm(D)).item() < 10 * w.idem_tol
    Hg = to_gpu(H)
    assert (torch.linalg.norm(Hg @ D - D @ Hg) / torch.linalg.norm(Hg)).item() < 1e-12


# ------------------------------------------------------------------------------------------------ properties (T3)
def test_sp2_persistent_kernel_full_parity_n1152(api, oracle_mod):
    """N = 1152 (> 1024) runs the persistent 128 x 128 kernel: 45 tiles on 148 CTAs, every tile split along K and
    reassembled from FP64 partials.  Full solve against the oracle, element by element."""
    H = hm.small_long_range((12, 12, 8))
    D, res, _ = _check_solve(api, oracle_mod, H, H.shape[0] // 2, 1e-10)
    assert res.status == 0
    assert np.linalg.norm(H @ D - D @ H) / np.linalg.norm(H) < 1e-12


@pytest.mark.parametrize("a,b", [(3.0, 0.0), (0.25, -7.5), (1.0, 100.0)])
def test_sp2_shift_scale_invariance_on_gpu(api, a, b):
    """H -> a H + b I (a > 0) leaves X_0, hence the branch string, m* and D unchanged (SURVEY 8(c) pins)."""
    H, _ = hm.planted_gap(150, 60, gap=1.0, width=2.0, seed=11)
    D0, r0 = api.bml_sp2_dense(to_gpu(H), 60, 1e-10)
    D1, r1 = api.bml_sp2_dense(to_gpu(a * H + b * np.eye(150)), 60, 1e-10)
    assert r0.status == r1.status == 0
    assert r1.branch == r0.branch and r1.n_products == r0.n_products
    assert relfro(D1.cpu().numpy(), D0.cpu().numpy()) < 1e-11


def test_sp2_permutation_similarity_on_gpu(api):
    """H -> P H P^T gives P D P^T with the same branch string (tile assignment must not matter)."""
    N, n_occ = 700, 300          # 64 x 64 tiles, ragged
    H, _ = hm.planted_gap(N, n_occ, gap=1.0, width=2.0, seed=12)
    perm = np.random.default_rng(1).permutation(N)
    Hp = H[np.ix_(perm, perm)]
    D0, r0 = api.bml_sp2_dense(to_gpu(H), n_occ, 1e-10)
    D1, r1 = api.bml_sp2_dense(to_gpu(Hp), n_occ, 1e-10)
    assert r0.status == r1.status == 0 and r1.branch == r0.branch
    assert relfro(D1.cpu().numpy(), D0.cpu().numpy()[np.ix_(perm, perm)]) < 1e-11


def test_sp2_dense_is_bit_reproducible(api):
    """Fixed-order reductions and the fixed stream-K summation order: two solves of the same H give the same bits."""
    H = hm.small_long_range((12, 12, 8))
    D0, r0 = api.bml_sp2_dense(to_gpu(H), 576, 1e-10)
    D0 = D0.clone()
    D1, r1 = api.bml_sp2_dense(to_gpu(H), 576, 1e-10)
    import torch

    assert torch.equal(D0, D1)
    assert np.array_equal(r0.trace, r1.trace) and np.array_equal(r0.idem, r1.idem)


def test_sp2_square_kernel_many_launches_bit_reproducible(api):
    """The persistent FP64 kernel repeated 300 times on one iterate (N = 2048, every tile K-split; and N = 3000, full
    waves + a split wave): any race in the TMA ring (dense_fp64_core.cuh StageRelease) or in the split-tile hand-off
    would show as a launch whose output differs in a few elements."""
    import torch

    for N in (2048, 3000):
        rng = np.random.default_rng(N)
        G = rng.normal(size=(N, N)) / np.sqrt(N)
        X = api.padded_dense((G + G.T) / 4 + 0.5 * np.eye(N))
        Xn = torch.empty_strided(X.shape, X.stride(), dtype=X.dtype, device="cuda")
        ws = api._workspace(api.load().bml_x2_dense_workspace_bytes(N, 0), "cuda")
        api.bml_x2_dense(X, 0, 0, Xn, ws)
        ref = Xn.clone()
        for it in range(300):
            _, sums = api.bml_x2_dense(X, 0, 0, Xn, ws)
            assert torch.equal(Xn, ref), f"N={N}: launch {it} differs"


def test_sp2_small_matrix_graph_replay_on_a_side_stream(api, oracle_mod):
    """On a non-default stream the prelude and the first batch of product launches of a small dense solve are captured
    once and replayed as a CUDA graph (api.cu): replays give the bits of the plainly enqueued solve, also when the
    input content changes under the same pointers, with and without the Lanczos flag, and for solves that need more
    products than the first batch holds."""
    import torch

    cases = [(hm.make_dense("dense_n256"), 128, 1e-10), (hm.small_long_range((8, 8, 6)), 192, 1e-10)]
    side = torch.cuda.Stream()
    for H1, n_occ, tol in cases:
        H2 = H1 + np.diag(np.linspace(-0.05, 0.05, H1.shape[0]))
        refs = []
        for Hx in (H1, H2):
            D, r = api.bml_sp2_dense(to_gpu(Hx), n_occ, tol)          # default stream: plain enqueue
            refs.append((D.clone(), r))
        assert refs[1][1].n_products > 16 or H1.shape[0] == 256      # the long-range case outlasts the first batch
        solver = api.DenseSolver(H1.shape[0], "cuda", 0)
        Hbuf = to_gpu(H1)
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            for it in range(6):
                Hbuf.copy_(to_gpu(H1 if it % 2 == 0 else H2))
                D, r = solver.solve(Hbuf, n_occ, tol)
                D0, r0 = refs[it % 2]
                assert r.status == r0.status == 0 and r.branch == r0.branch and r.n_products == r0.n_products
                assert np.array_equal(r.idem, r0.idem)
                assert torch.equal(D, D0), f"replay {it}"
            Dl, rl = solver.solve(Hbuf, n_occ, tol, flags=api.FLAG_LANCZOS_BOUNDS(16))
            Dl2, rl2 = solver.solve(Hbuf, n_occ, tol, flags=api.FLAG_LANCZOS_BOUNDS(16))
            assert rl.status == 0 and rl.branch == rl2.branch and (rl.emin, rl.emax) == (rl2.emin, rl2.emax)
            assert rl.n_products <= refs[1][1].n_products
        torch.cuda.synchronize()
