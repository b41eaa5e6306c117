"""Pins of the Chebyshev / Paterson-Stockmeyer oracle (oracle/chebyshev.py) against what the paper and the mathematics
fix: closed forms, library routines that are NOT the ones the oracle calls, the exact result within the measured
truncation error, and invariants.  CPU only.

Each pin names the mistake it is meant to catch."""
import math

import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

from oracle import chebyshev as ch
from paper_2401_13772_b200 import hamiltonians as hm


def relfro(A, B):
    return np.linalg.norm(A - B) / np.linalg.norm(B)


# ------------------------------------------------ coefficients (Eq. 8, reading C3) ----------------------
@pytest.mark.parametrize("n0", [0, 1, 3, 7])
def test_coeffs_of_a_chebyshev_polynomial_are_a_unit_vector(n0):
    """f = T_{n0}  =>  c_n = [n = n0]: catches a wrong c_0 weight (the 1/2 of the n = 0 term) and wrong nodes."""
    L = 11
    x = ch.gauss_nodes(2 * (L + 1))
    c = ch.cheb_coeffs_from_samples(npcheb.chebval(x, np.eye(L + 1)[n0]), L)
    assert np.allclose(c, np.eye(L + 1)[n0], atol=1e-14)


def test_coeffs_of_exp_are_modified_bessel_functions():
    """exp(x) = I_0(1) + 2 sum_n I_n(1) T_n(x) (textbook closed form): catches a wrong normalisation or cosine
    argument; I_n(1) from its power series, not from the oracle."""
    def bessel_i(n, z=1.0):
        return sum((z / 2) ** (2 * j + n) / (math.factorial(j) * math.factorial(j + n)) for j in range(40))

    L = 15
    x = ch.gauss_nodes(2 * (L + 1))
    c = ch.cheb_coeffs_from_samples(np.exp(x), L)
    expect = np.array([bessel_i(0)] + [2.0 * bessel_i(n) for n in range(1, L + 1)])
    assert np.allclose(c, expect, rtol=0, atol=1e-15)


def test_fermi_series_reproduces_the_fermi_function_on_the_interval():
    """sum_n c_n T_n(x(eps)) = f_mu(eps) within the truncation error: catches a swapped interval map (x <-> -x),
    a wrong sign of beta or mu."""
    emin, emax, mu, beta, L = -3.0, 5.0, 0.7, 4.0, 127
    c = ch.cheb_coeffs(emin, emax, mu, beta, L)
    eps = np.linspace(emin, emax, 2001)
    x = (2.0 * eps - (emax + emin)) / (emax - emin)
    assert np.max(np.abs(npcheb.chebval(x, c) - 1.0 / (1.0 + np.exp(beta * (eps - mu))))) < 1e-10
    assert abs(ch.fermi(np.array([mu]), mu, beta)[0] - 0.5) < 1e-16
    assert ch.fermi(np.array([emin]), mu, beta)[0] > 0.99 and ch.fermi(np.array([emax]), mu, beta)[0] < 1e-7


# ------------------------------------------------ d_{i,j} (Eq. 10-12, reading C4) -----------------------
@pytest.mark.parametrize("k,m", [(2, 1), (2, 3), (3, 3), (4, 4), (5, 2), (8, 8), (16, 16), (16, 3), (7, 9), (32, 8)])
def test_resummed_form_equals_the_series_on_scalars(k, m):
    """Eq. 10 with the oracle's d_{i,j} = Eq. 8 evaluated by numpy.polynomial.chebyshev.chebval (Clenshaw, a
    different algorithm): catches a wrong index or sign in the division by T_k (the T_{|n-2k|} term)."""
    rng = np.random.default_rng(k * 100 + m)
    c = rng.normal(size=k * m) * 0.7 ** np.arange(k * m)
    d = ch.ps_coeffs(c, k)
    assert d.shape == (k, m)
    x = np.concatenate([np.linspace(-1, 1, 101), rng.uniform(-1, 1, 50)])
    ref = npcheb.chebval(x, c)
    assert np.max(np.abs(ch.ps_eval_scalar(d, x) - ref)) < 1e-12 * max(1.0, np.abs(c).sum())


def test_ps_coeffs_hand_example():
    """k = 2, m = 2 worked by hand from Eq. 11: T_2 = T_2 T_0, T_3 = 2 T_2 T_1 - T_1, so
    c_0 T_0 + c_1 T_1 + c_2 T_2 + c_3 T_3 = (c_0 T_0 + (c_1 - c_3) T_1) + T_2 (c_2 T_0 + 2 c_3 T_1)."""
    c = np.array([0.3, -1.1, 0.8, 0.25])
    d = ch.ps_coeffs(c, 2)
    assert np.allclose(d, [[0.3, 0.8], [-1.1 - 0.25, 0.5]], atol=0, rtol=0)


# ------------------------------------------------ T_i (Eq. 11, 13, 14, reading C5) ----------------------
def test_doubling_gives_chebyshev_polynomials_of_the_matrix():
    """T_i(H~) = U T_i(lambda) U^T with T_i(lambda) = cos(i arccos lambda): catches a wrong (a, b) split or a wrong
    subtracted term T_{a-b}."""
    rng = np.random.default_rng(5)
    A = rng.normal(size=(40, 40))
    H = (A + A.T) / 2
    emin, emax = ch.gershgorin(H)
    Ht = ch.map_to_unit(H, emin, emax)
    w, U = np.linalg.eigh(Ht)
    assert w.min() >= -1.0 and w.max() <= 1.0
    T = ch.cheb_T_doubling(Ht, 13)
    assert len(T) == 14
    for i, Ti in enumerate(T):
        assert np.allclose(Ti, (U * np.cos(i * np.arccos(w))) @ U.T, atol=1e-12)


def test_gershgorin_matches_the_sp2_oracle(oracle_mod):
    H = hm.small_long_range((6, 5, 4))
    assert ch.gershgorin(H) == pytest.approx(oracle_mod.gershgorin_dense(H), rel=1e-15)


# ------------------------------------------------ D (Eq. 8 / Eq. 10) ------------------------------------
@pytest.mark.parametrize("k,m", [(8, 8), (16, 4), (4, 16), (16, 16)])
def test_serial_and_resummed_agree_and_approximate_the_fermi_operator(k, m):
    """chebyshev_ps (Eq. 10-14) = chebyshev_serial (Eq. 8-9) to round-off, and both equal U f(Lambda) U^T (LAPACK)
    within the truncation error of the scalar series measured on a fine grid."""
    H = hm.lattice_dense((6, 6, 5), 0.0, 0.2, 1.0, lambda r: -1.0, seed=1)
    mu, beta, L = 0.1, 3.0, k * m - 1
    Ds, info = ch.chebyshev_serial(H, mu, beta, L)
    Dp, info_p = ch.chebyshev_ps(H, mu, beta, k, m)
    assert info_p["n_products"] == k + m - 2 and info["n_products"] == L - 1
    assert relfro(Dp, Ds) < 1e-13
    assert np.allclose(Dp, Dp.T, atol=1e-14)
    eps = np.linspace(info["emin"], info["emax"], 4001)
    x = (2.0 * eps - (info["emax"] + info["emin"])) / (info["emax"] - info["emin"])
    trunc = np.max(np.abs(npcheb.chebval(x, info["c"]) - ch.fermi(eps, mu, beta)))
    De = ch.fermi_exact(H, mu, beta)
    # ||p(H) - f(H)||_2 <= max |p - f| on the spectrum
    assert np.linalg.norm(Ds - De, 2) <= trunc + 1e-13
    assert abs(np.trace(Ds) - ch.fermi(np.linalg.eigvalsh(H), mu, beta).sum()) <= H.shape[0] * (trunc + 1e-14)


def test_particle_hole_mirror():
    """f_mu(eps) + f_{-mu}(-eps) = 1  =>  D(H, mu) + D(-H, -mu) = I up to twice the truncation error: catches a sign
    error in the interval map that the scalar test cannot see once matrices are involved."""
    H = hm.lattice_dense((5, 4, 4), 0.0, 0.3, 1.0, lambda r: -1.0, seed=2)
    k, m, mu, beta = 8, 8, 0.4, 2.0
    D1, _ = ch.chebyshev_ps(H, mu, beta, k, m)
    D2, _ = ch.chebyshev_ps(-H, -mu, beta, k, m)
    assert np.allclose(D1 + D2, np.eye(H.shape[0]), atol=1e-9)


def test_cold_limit_is_the_sp2_projector(oracle_mod):
    """At beta * gap >> 1 the Fermi operator is the projector on the occupied subspace, which is what the SP2
    oracle returns (Eq. 5-7): ties the two oracles together."""
    N, n_occ = 48, 20
    H, eps = hm.planted_gap(N, n_occ, gap=2.0, width=0.5, seed=4)
    D_sp2, st = oracle_mod.sp2_dense(H, n_occ, 1e-12)
    assert st["status"] in (0, 1)
    D, _ = ch.chebyshev_ps(H, 0.0, 20.0, 32, 32)       # f(+-gap/2) is e^-20 away from {1, 0}; L = 1023
    assert relfro(D, D_sp2) < 1e-7
    assert abs(np.trace(D) - n_occ) < 1e-6


def test_symm_ab_is_the_plain_definition():
    rng = np.random.default_rng(0)
    A, B, C = rng.normal(size=(3, 6, 6))
    out = ch.symm_ab(A, B, C, 2.0, -1.0, 0.5)
    ref = np.zeros((6, 6))
    for i in range(6):
        for j in range(6):
            ref[i, j] = 2.0 * sum(A[i, q] * B[q, j] for q in range(6)) - C[i, j] + (0.5 if i == j else 0.0)
    assert np.allclose(out, ref, atol=1e-14)
    assert np.allclose(ch.symm_ab(A, B, None, 1.0, 0.0, 0.0), A @ B, atol=1e-14)
