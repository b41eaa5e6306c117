"""GPU parity, dense mixed-precision mode (BASELINE.json configs[3]; readings item 17): tcgen05 products of
16-bit planes of X (precision 1: two scaled FP16 planes, the default; precision 2: three BF16 planes) on CTA pairs
(cta_group::2), the leading term's FP32 TMEM accumulation promoted to FP64 every 512 columns, the small cross terms in an
accumulator of their own, FP64 traces / norms / updates.

The oracle of this mode is the FP64 CPU oracle run with the mixed config's tolerance (1e-6).  Required (north_star):
identical branch string and product count, relative Frobenius error of D <= 1e-5.  One product is held to
relFro <= 3e-6 (DESIGN.md 5.3 "Error budget": the planes keep 22-24 mantissa bits, the dropped cross terms are
<= 2^-22, and the truncating FP32 accumulation of the leading term over a 512-column chunk adds a one-sided bias that
stays below 3e-6 relFro on mixed-sign data; all-positive inputs, the worst case, are held to the bounds derived in
test_x2_mixed_sampled_over_several_chunks_and_periods; the diagonal of X^2 is computed in FP64)."""
import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm

pytestmark = pytest.mark.gpu

TOL_D_MIXED = 1e-5     # north_star
TOL_P_MIXED = 3e-6     # one product, relative Frobenius
TOL_MIXED_IDEM = 1e-6  # BASELINE.json configs[3]


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


PRECISIONS = [1, 2]


@pytest.mark.parametrize("N", [1, 2, 7, 128, 129, 200, 384, 515])
@pytest.mark.parametrize("branch", [0, 1])
@pytest.mark.parametrize("precision", PRECISIONS)
def test_x2_mixed_one_product(api, oracle_mod, N, branch, precision):
    """One fused mixed-precision product on sizes spanning several 128x128 tiles, ragged tails and a K tail that is
    not a multiple of the 32-column slab or of the 512-column promotion chunk (the 2048 columns after which the BF16
    split's small-term accumulators alternate are covered by the sampled test below)."""
    import torch

    rng = np.random.default_rng(100 + N)
    A = rng.normal(size=(N, N)) / np.sqrt(N)
    X = (A + A.T) / 2 + np.diag(rng.uniform(0.0, 1.0, N))
    P = oracle_mod.x2_dense(X)
    ref = 2.0 * X - P if branch else P
    Xn, sums = api.bml_x2_dense(api.padded_dense(X), branch, precision)
    got = Xn.cpu().numpy()
    scale = np.linalg.norm(P)
    assert np.linalg.norm(got - ref) <= TOL_P_MIXED * scale
    assert np.array_equal(got, got.T), "mirrored write must make X' bitwise symmetric"
    s = sums.cpu().numpy()
    expect = np.array([np.trace(P), np.linalg.norm(P - X) ** 2, np.linalg.norm(X) ** 2, np.trace(ref)])
    assert abs(s[2] - expect[2]) <= 1e-12 * expect[2]          # ||X||^2 is pure FP64
    assert np.allclose(s, expect, rtol=2e-5, atol=1e-5 * abs(expect[0]))
    # "FP64 traces": the diagonal of X^2 comes from the FP64 master iterate, so tr(X^2) is exact to FP64 round-off
    assert abs(s[0] - expect[0]) <= 1e-12 * max(1.0, abs(expect[0]))
    # the trace the kernel reports is the trace of the matrix it wrote (it decides the next branch)
    assert abs(s[3] - np.trace(got)) <= 1e-12 * max(1.0, np.abs(np.diag(got)).sum())


@pytest.mark.parametrize("N,same_sign", [(1100, False), (2200, False), (4300, False), (4300, True)])
@pytest.mark.parametrize("precision", PRECISIONS)
def test_x2_mixed_sampled_over_several_chunks_and_periods(api, oracle_mod, N, same_sign, precision):
    """One product at sizes the dense oracle cannot finish in seconds, on sampled entries (each an N-term compensated dot
    product of the oracle): several 512-column promotion chunks with a ragged last one (N = 1100: 3 chunks; 2200: 5),
    two and three 2048-column periods of the BF16 split's small-term accumulators (4300: the third period re-uses the
    first accumulator, so the MMA issuer's wait on its drain is exercised), an odd number of tile rows (34 at 4300: the
    last pair has one CTA beyond the grid), tile corners and the pair on the diagonal.  `same_sign`: all entries positive,
    the worst case of the tensor core's truncating accumulate (every update loses up to one ulp in the same direction);
    SP2 iterates are not of that kind (their off-diagonal sums have mixed signs and the diagonal of X^2 is computed in
    FP64), so the solve-level numbers of DESIGN.md 5.3 are those of the mixed-sign rows."""
    import torch

    rng = np.random.default_rng(700 + N + int(same_sign))
    if same_sign:
        A = rng.uniform(0.0, 1.0, size=(N, N)) / N
        X = (A + A.T) / 2 + np.diag(rng.uniform(0.0, 0.5, N))
    else:
        A = rng.normal(size=(N, N)) / np.sqrt(N)
        X = (A + A.T) / 2 + np.diag(rng.uniform(0.0, 1.0, N))
    rows = np.concatenate([rng.integers(0, N, 200), [0, 127, 128, 255, 256, N - 1, N - 1, 0, 129, 300]])
    cols = np.concatenate([rng.integers(0, N, 200), [0, 128, 127, 256, 255, N - 1, 0, N - 1, 130, 300]])
    ref = oracle_mod.x2_dense_sampled(X, rows, cols)
    mag = np.einsum("ik,ik->i", np.abs(X[rows]), np.abs(X[:, cols].T))
    Xg = api.padded_dense(X)
    r_t, c_t = torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()
    for branch in (0, 1):
        Xn, sums = api.bml_x2_dense(Xg, branch, precision)
        got = Xn[r_t, c_t].cpu().numpy()
        expect = 2.0 * X[rows, cols] - ref if branch else ref
        # bound per entry, relative to sum_k |x_ik x_kj|: planes 2^-22, then per 512-column chunk 32 truncating updates of
        # an accumulator that (same-sign terms) grows to the chunk sum, <= 32 x 2^-23 = 3.8e-6, and as much again for the
        # truncated alignment of the 16 products inside each MMA: 8e-6 in the worst case (measured: max 6.3e-6, mean bias
        # -2.8e-6 for FP16 x 2, -1.0e-6 for BF16 x 3); mixed-sign data stay far below (4e-6 asserted, ~1e-7 measured)
        assert (np.abs(got - expect) <= (8e-6 if same_sign else 4e-6) * mag + 1e-12).all()
        assert np.array_equal(got, Xn[c_t, r_t].cpu().numpy())
        # relative Frobenius error over the sample, against the one-product bound
        assert np.linalg.norm(got - expect) <= (5e-6 if same_sign else TOL_P_MIXED) * np.linalg.norm(ref)
        s = sums.cpu().numpy()
        assert abs(s[2] - np.linalg.norm(X) ** 2) <= 1e-12 * np.linalg.norm(X) ** 2
        assert abs(s[3] - torch.trace(Xn).item()) <= 1e-12 * max(1.0, torch.diagonal(Xn).abs().sum().item())
        del Xn


def _check_mixed_solve(api, oracle_mod, H, n_occ, precision, tol=TOL_MIXED_IDEM):
    D_ref, st = oracle_mod.sp2_dense(H, n_occ, tol)
    D, res = api.bml_sp2_dense(to_gpu(H), n_occ, tol, 100, precision)
    assert st["status"] == 0 and res.status == 0
    assert res.n_products == st["n_products"] and res.m_star == st["m_star"]
    assert res.branch == st["branch"]
    assert (res.emin, res.emax) == (st["emin"], st["emax"])
    Dg = D.cpu().numpy()
    assert relfro(Dg, D_ref) <= TOL_D_MIXED
    assert np.array_equal(Dg, Dg.T)
    assert abs(np.trace(Dg) - n_occ) <= 1e-5 * n_occ
    return res, st


@pytest.mark.parametrize("precision", PRECISIONS)
def test_sp2_mixed_config1_model_n256(api, oracle_mod, precision):
    _check_mixed_solve(api, oracle_mod, hm.make_dense("dense_n256"), 128, precision)


@pytest.mark.parametrize("N,n_occ,seed", [(64, 20, 1), (200, 77, 2), (333, 100, 3)])
@pytest.mark.parametrize("precision", PRECISIONS)
def test_sp2_mixed_planted_gap(api, oracle_mod, N, n_occ, seed, precision):
    H, _ = hm.planted_gap(N, n_occ, gap=1.0, width=1.0, seed=seed)
    _check_mixed_solve(api, oracle_mod, H, n_occ, precision)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_sp2_mixed_small_long_range(api, oracle_mod, precision):
    """Reduced-size stand-in of the configs[3] Hamiltonian model (same hopping law, 8x8x6 box)."""
    H = hm.small_long_range((8, 8, 6))
    _check_mixed_solve(api, oracle_mod, H, H.shape[0] // 2, precision)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_sp2_mixed_config2_model_n2048(api, oracle_mod, precision):
    w = hm.WORKLOADS["dense_n2048"]
    _check_mixed_solve(api, oracle_mod, hm.make_dense("dense_n2048"), w.n_occ, precision)


def test_mixed_rejects_sparse_and_bad_precision(api):
    import torch

    X = api.padded_dense(np.eye(4))
    with pytest.raises(RuntimeError):
        api.bml_x2_dense(X, 0, 3)


@pytest.mark.parametrize("precision", PRECISIONS)
def test_config4_n16384_sampled_product_and_solve(api, oracle_mod, precision):
    """BASELINE.json configs[3] at full size (N=16384, mixed precision, tol 1e-6), in the launch configuration
    bench.py times.  The CPU oracle cannot finish an N=16384 solve in test time, so: (a) one fused mixed product on
    the oracle's X_0 is compared with the oracle on sampled entries (each an N-term compensated dot product), incl.
    tile corners; (b) the solve is checked through properties that hold at any size, against the branch string of
    the FP64 oracle's full solve stored in tests/golden (21,521 s of oracle time on 7 threads) and against the FP64
    DMMA path of this library (itself oracle-checked element by element at the sizes the oracle reaches, and against
    the oracle's first four products at this size in tests/test_golden.py)."""
    import torch

    w = hm.WORKLOADS["mixed_n16384"]
    H = hm.make_dense("mixed_n16384")
    N = w.N
    lo, hi = oracle_mod.gershgorin_dense(H)
    X0 = oracle_mod.rescale_dense(H, lo, hi)
    rng = np.random.default_rng(7)
    rows = np.concatenate([rng.integers(0, N, 300), [0, 127, 128, N - 1, N - 1, 8191, 8192, 300]])
    cols = np.concatenate([rng.integers(0, N, 300), [0, 128, 127, N - 1, 0, 8192, 8191, 300]])
    ref = oracle_mod.x2_dense_sampled(X0, rows, cols)
    Xg = api.padded_dense(X0)
    # |x_ik x_kj| summed over k bounds what the truncating FP32 accumulation and the dropped cross terms can lose
    mag = np.einsum("ik,ik->i", np.abs(X0[rows]), np.abs(X0[:, cols].T))
    for branch in (0, 1):
        Xn, sums = api.bml_x2_dense(Xg, branch, precision)
        got = Xn[torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()].cpu().numpy()
        expect = 2.0 * X0[rows, cols] - ref if branch else ref
        assert (np.abs(got - expect) <= 4e-6 * mag + 1e-12).all()
        got_t = Xn[torch.from_numpy(cols).cuda(), torch.from_numpy(rows).cuda()].cpu().numpy()
        assert np.array_equal(got, got_t)
        del Xn
    del Xg
    Hg = to_gpu(H)
    D, res = api.bml_sp2_dense(Hg, w.n_occ, w.idem_tol, 100, precision)
    assert res.status == 0
    assert (res.emin, res.emax) == (lo, hi)
    import json
    import os

    here = os.path.dirname(os.path.abspath(__file__))
    gold = json.load(open(os.path.join(here, "golden", "sp2_expected.json")))["mixed_n16384"]
    if True:
        # the FP64 oracle's full solve of configs[3] at the mixed tolerance (tests/golden/make_golden.py mixed_n16384):
        # same branch string and product count, D within the mixed tolerance over every entry (Gaussian probe)
        assert res.branch == gold["branch"] and res.n_products == gold["n_products"] and res.m_star == gold["m_star"]
        y = torch.from_numpy(np.loadtxt(os.path.join(here, "golden", gold["Dv_file"]))).cuda()
        v = torch.from_numpy(np.random.default_rng(gold["probe_seed"]).standard_normal(N)).cuda()
        assert (torch.linalg.norm(D @ v - y) / gold["D_fro"]).item() <= 3 * TOL_D_MIXED
        for i, j, val in gold["D_samples"]:
            assert abs(D[i, j].item() - val) <= TOL_D_MIXED * gold["D_fro"]
    assert res.n_products == 30
    assert res.idem[-1] < w.idem_tol
    assert abs(torch.trace(D).item() - w.n_occ) < 1e-5 * w.n_occ
    assert torch.equal(D, D.T)
    Dm = D.clone()
    D64, r64 = api.bml_sp2_dense(Hg, w.n_occ, w.idem_tol, 100, 0)
    assert r64.status == 0 and r64.branch == res.branch and r64.n_products == res.n_products
    assert (torch.linalg.norm(Dm - D64) / torch.linalg.norm(D64)).item() <= TOL_D_MIXED
    assert (torch.linalg.norm(Hg @ Dm - Dm @ Hg) / torch.linalg.norm(Hg)).item() < 1e-5
