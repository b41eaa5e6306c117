"""Pins of the tighter-spectral-bounds oracle (oracle/bounds.py) against what the mathematics fixes.  CPU only."""
import numpy as np
import pytest

from oracle import bounds as ob
from oracle import chebyshev as och
from paper_2401_13772_b200 import hamiltonians as hm


def test_splitmix64_first_output_of_the_published_generator():
    """SplitMix64 seeded with 0 yields 0xE220A8397B1DCDAF first (the test vector published with the generator)."""
    assert ob.splitmix64(0) == 0xE220A8397B1DCDAF
    u = ob.start_vector(1000, 3)
    assert u.min() >= -1.0 and u.max() < 1.0 and abs(u.mean()) < 0.1 and len(set(u.tolist())) == 1000


def test_lanczos_matches_moments_of_the_start_vector():
    """K steps of Lanczos reproduce the moments v0^T H^p v0 = e1^T T^p e1 for p <= 2K - 1 (the defining property of
    the recursion): catches a wrong sign or index in the three-term recurrence."""
    rng = np.random.default_rng(0)
    G = rng.normal(size=(40, 40))
    H = (G + G.T) / 2
    K = 4
    alpha, beta = ob.lanczos(H, K, seed=5)
    T = np.diag(alpha) + np.diag(beta[1:K], 1) + np.diag(beta[1:K], -1)
    u = ob.start_vector(40, 5)
    v0 = u / np.linalg.norm(u)
    for p in range(2 * K):
        assert np.linalg.matrix_power(T, p)[0, 0] == pytest.approx(v0 @ np.linalg.matrix_power(H, p) @ v0, rel=1e-10)


def test_full_length_recursion_gives_the_spectrum():
    rng = np.random.default_rng(1)
    G = rng.normal(size=(12, 12))
    H = (G + G.T) / 2
    alpha, beta = ob.lanczos(H, 12)
    T = np.diag(alpha) + np.diag(beta[1:12], 1) + np.diag(beta[1:12], -1)
    assert np.allclose(np.linalg.eigvalsh(T), np.linalg.eigvalsh(H), atol=1e-8)


def test_two_by_two_closed_form():
    """K = N = 2: T is similar to H, beta_2 = 0, so the bounds are the exact eigenvalues widened by the 1% pad."""
    H = np.array([[1.0, 2.0], [2.0, -3.0]])
    lo, hi, info = ob.lanczos_bounds(H, 2)
    ev = np.array([-1.0 - np.sqrt(8.0), -1.0 + np.sqrt(8.0)])
    assert info["beta"][2] == pytest.approx(0.0, abs=1e-14)
    pad = 0.01 * (ev[1] - ev[0])
    assert lo == pytest.approx(ev[0] - pad, rel=1e-12) and hi == pytest.approx(ev[1] + pad, rel=1e-12)


@pytest.mark.parametrize("K", [8, 16, 24, 32])
@pytest.mark.parametrize("name", ["ring", "nn_lattice", "long_range", "planted", "gapless", "sparse5p"])
def test_bounds_enclose_the_spectrum_and_beat_gershgorin(name, K):
    H = {
        "ring": lambda: hm.make_dense("dense_n256"),
        "nn_lattice": lambda: hm.lattice_dense((8, 8, 6), 1.5, 0.2, 1.0, lambda r: -1.0),
        "long_range": lambda: hm.small_long_range((8, 8, 6)),
        "planted": lambda: hm.planted_gap(200, 77, seed=2)[0],
        "gapless": lambda: hm.lattice_dense((8, 8, 6), 0.0, 0.2, 1.0, lambda r: -1.0),
        "sparse5p": lambda: hm.ellpack_to_dense(*hm.small_sparse_model((8, 7, 8))),
    }[name]()
    w = np.linalg.eigvalsh(H)
    glo, ghi = och.gershgorin(H)
    for seed in (0, 1, 2):
        lo, hi, info = ob.lanczos_bounds(H, K, seed)
        assert lo <= w[0] and hi >= w[-1], (lo, w[0], w[-1], hi)
        assert lo >= glo and hi <= ghi
        assert info["theta"][0] >= w[0] - 1e-9 and info["theta"][-1] <= w[-1] + 1e-9      # Ritz values interlace
    if name in ("long_range", "ring"):
        assert (hi - lo) < 0.8 * (ghi - glo)


def test_sp2_with_the_tighter_bounds_returns_the_same_projector_in_fewer_products(oracle_mod):
    H = hm.small_long_range((8, 8, 6))
    n_occ = H.shape[0] // 2
    D0, s0 = oracle_mod.sp2_dense(H, n_occ, 1e-10)
    lo, hi, _ = ob.lanczos_bounds(H, 20)
    D1, s1 = oracle_mod.sp2_dense(H, n_occ, 1e-10, bounds=(lo, hi))
    assert s0["status"] == 0 and s1["status"] == 0
    assert (s1["emin"], s1["emax"]) == (lo, hi)
    assert s1["n_products"] < s0["n_products"] - 3
    assert np.linalg.norm(D1 - D0) / np.linalg.norm(D0) < 1e-9
    # bounds=None is the Gershgorin path, bit for bit
    D2, s2 = oracle_mod.sp2_dense(H, n_occ, 1e-10, bounds=None)
    assert np.array_equal(D2, D0) and s2["branch"] == s0["branch"]
