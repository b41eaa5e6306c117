"""CPU oracle for the Chebyshev / Paterson-Stockmeyer density-matrix path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain numpy, FP64.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module; it imports nothing from ``paper_2401_13772_b200``.

What the path computes (section IV.B):

    f_mu(H) ~ sum_{n=0}^{L} c_n T_n(H~)                                      Eq. 8
    T_{n+1} = 2 H~ T_n - T_{n-1}                                             Eq. 9
    sum_n c_n T_n = S_0 + T_k (S_1 + T_k (S_2 + ... + T_k S_{m-1}))          Eq. 10,  L + 1 = k m
    T_n T_m = (T_{n+m} + T_{|n-m|}) / 2                                      Eq. 11
    S_j = sum_{i<k} d_{i,j} T_i                                              Eq. 12
    T_2 = 2 T_1 T_1 - T_0;  T_3 = 2 T_2 T_1 - T_1;  T_4 = 2 T_2 T_2 - T_0    Eq. 13-14

The resummed form (Eq. 10) reaches, up to rounding order, the same matrix as the plain sum (Eq. 8), so the parity
target is ``chebyshev_serial`` -- Eq. 8 evaluated by the recursion Eq. 9, the definition written out.
``chebyshev_ps`` follows Eq. 10-14 step by step in the paper's order and is pinned against it.

Readings of the paper (listed in DESIGN.md "Readings", Chebyshev items):
  C1. H~ = (2 H - (e_max + e_min) I) / (e_max - e_min) maps the Gershgorin interval onto [-1, 1] (the paper writes
      T_n(H); Chebyshev polynomials need the spectrum in [-1, 1]; bounds as in the SP2 path).
  C2. f_mu(eps) = 1 / (1 + exp(beta (eps - mu))), beta = 1 / (k_B T), mu given ("using a known chemical
      potential", Fig. 3 caption P:247).
  C3. c_n by Chebyshev-Gauss quadrature on N_q = 2 (L + 1) nodes x_q = cos(pi (q + 1/2) / N_q):
      c_n = (2 - [n = 0]) / N_q * sum_q f(x_q) cos(n pi (q + 1/2) / N_q)   (the paper does not say how c_n is obtained).
  C4. d_{i,j}: "can be determined from the Chebyshev coefficients c_n" via Eq. 11 (the construction itself is in
      Ref. 37, not in the paper): divide the series by T_k using T_n = 2 T_k T_{n-k} - T_{|n-2k|} (Eq. 11 with
      (n, m) = (k, n - k)), highest n first; the remainder is S_0, the quotient is divided again.
  C5. T_i, 2 <= i <= k, by Eq. 11 with the most balanced split: T_i = 2 T_a T_b - T_{a-b}, a = ceil(i / 2),
      b = floor(i / 2) (this is Eq. 13-14 for i = 2, 3, 4).

Pins (tests/test_oracle_chebyshev.py): closed-form coefficients (T_3 itself; exp(x) -> modified Bessel functions),
Eq. 10 against numpy.polynomial.chebyshev.chebval on scalars for many (k, m), T_i(H~) against the spectral
decomposition, D against U f(Lambda) U^T from LAPACK within the measured truncation error of the scalar series,
particle-hole mirror D(H, mu) + D(-H, -mu) = I, the zero-temperature limit against the SP2 oracle's projector.
"""
from __future__ import annotations

import numpy as np


# ------------------------------------------------ scalars ------------------------------------------------
def fermi(eps, mu, beta):
    """f_mu(eps) = 1 / (1 + exp(beta (eps - mu))) (reading C2), written to avoid overflow of exp."""
    z = beta * (np.asarray(eps, dtype=np.float64) - mu)
    out = np.empty_like(z)
    pos = z >= 0
    ez = np.exp(-z[pos])
    out[pos] = ez / (1.0 + ez)
    out[~pos] = 1.0 / (1.0 + np.exp(z[~pos]))
    return out


def gauss_nodes(Nq):
    """x_q = cos(pi (q + 1/2) / N_q), q = 0..N_q-1 (reading C3)."""
    q = np.arange(Nq, dtype=np.float64)
    return np.cos(np.pi * (q + 0.5) / Nq)


def cheb_coeffs_from_samples(fx, L):
    """c_0..c_L of the Chebyshev series of a function sampled at gauss_nodes(len(fx)) (reading C3)."""
    fx = np.asarray(fx, dtype=np.float64)
    Nq = fx.size
    q = np.arange(Nq, dtype=np.float64)
    c = np.empty(L + 1)
    for n in range(L + 1):
        c[n] = (1.0 if n == 0 else 2.0) / Nq * np.sum(fx * np.cos(n * np.pi * (q + 0.5) / Nq))
    return c


def cheb_coeffs(emin, emax, mu, beta, L):
    """Eq. 8 coefficients of eps -> f_mu(eps) on [e_min, e_max] mapped to x in [-1, 1] (readings C1-C3)."""
    Nq = 2 * (L + 1)
    x = gauss_nodes(Nq)
    eps = 0.5 * (emax - emin) * x + 0.5 * (emax + emin)
    return cheb_coeffs_from_samples(fermi(eps, mu, beta), L)


def ps_coeffs(c, k):
    """d[i, j] of Eq. 10 / Eq. 12 from c_0..c_L, L + 1 = k m (reading C4).

    One division step: p = sum_{n<=deg} p_n T_n = T_k q + r with deg r < k.  For n > k, Eq. 11 with (k, n - k) gives
    T_n = 2 T_k T_{n-k} - T_{|n-2k|}; for n = k, T_k = T_k T_0.  Going down from the highest n, p_n is moved into
    q_{n-k} (times 2, or times 1 when n = k) and subtracted from p_{|n-2k|}, which is of lower degree than n.
    """
    c = np.asarray(c, dtype=np.float64)
    assert k >= 2 and c.size % k == 0
    m = c.size // k
    d = np.zeros((k, m))
    p = c.copy()
    for j in range(m):
        q = np.zeros(max(p.size - k, 0))
        for n in range(p.size - 1, k, -1):
            q[n - k] += 2.0 * p[n]
            p[abs(n - 2 * k)] -= p[n]
        if p.size > k:
            q[0] += p[k]
        d[:, j] = p[:k]
        p = q
    assert p.size == 0
    return d


def ps_eval_scalar(d, x):
    """Right-hand side of Eq. 10 at scalars x in [-1, 1] (used by the pins)."""
    x = np.asarray(x, dtype=np.float64)
    k, m = d.shape
    T = [np.ones_like(x), x]
    for i in range(2, k + 1):
        T.append(2.0 * x * T[i - 1] - T[i - 2])
    R = np.zeros_like(x)
    for j in range(m - 1, -1, -1):
        S = sum(d[i, j] * T[i] for i in range(k))
        R = T[k] * R + S
    return R


# ------------------------------------------------ matrices -----------------------------------------------
def gershgorin(H):
    """(e_min, e_max) by Gershgorin circles, same definition as the SP2 oracle's."""
    H = np.asarray(H, dtype=np.float64)
    dg = np.diag(H)
    off = np.sum(np.abs(H), axis=1) - np.abs(dg)
    return float(np.min(dg - off)), float(np.max(dg + off))


def map_to_unit(H, emin, emax):
    """H~ of reading C1."""
    H = np.asarray(H, dtype=np.float64)
    return (2.0 * H - (emax + emin) * np.eye(H.shape[0])) / (emax - emin)


def chebyshev_serial(H, mu, beta, L):
    """D = sum_n c_n T_n(H~), Eq. 8 by the recursion Eq. 9 -- the definition; L products.  Returns (D, info)."""
    emin, emax = gershgorin(H)
    c = cheb_coeffs(emin, emax, mu, beta, L)
    Ht = map_to_unit(H, emin, emax)
    N = Ht.shape[0]
    Tm, Tc = np.eye(N), Ht
    D = c[0] * Tm
    if L >= 1:
        D = D + c[1] * Tc
    for n in range(2, L + 1):
        Tm, Tc = Tc, 2.0 * (Ht @ Tc) - Tm          # Eq. 9
        D = D + c[n] * Tc
    return D, {"emin": emin, "emax": emax, "c": c, "n_products": max(L - 1, 0)}


def cheb_T_doubling(Ht, k):
    """[T_0, ..., T_k](H~) by Eq. 11 with the balanced split of reading C5 (Eq. 13-14); k - 1 products."""
    N = Ht.shape[0]
    T = [np.eye(N), Ht]
    for i in range(2, k + 1):
        a, b = (i + 1) // 2, i // 2
        T.append(2.0 * (T[a] @ T[b]) - T[a - b])
    return T


def chebyshev_ps(H, mu, beta, k, m):
    """D by the resummed form Eq. 10, step by step: T_0..T_k (Eq. 13-14), S_j (Eq. 12), nested products (Eq. 10).
    k + m - 2 products.  Returns (D, info)."""
    L = k * m - 1
    emin, emax = gershgorin(H)
    c = cheb_coeffs(emin, emax, mu, beta, L)
    d = ps_coeffs(c, k)
    Ht = map_to_unit(H, emin, emax)
    T = cheb_T_doubling(Ht, k)
    S = [sum(d[i, j] * T[i] for i in range(k)) for j in range(m)]
    R = S[m - 1]
    for j in range(m - 2, -1, -1):
        R = T[k] @ R + S[j]
    return R, {"emin": emin, "emax": emax, "c": c, "d": d, "n_products": k + m - 2}


def symm_ab(A, B, C, alpha, beta, gamma):
    """alpha A B + beta C + gamma I -- the one matrix operation Eq. 10, 13, 14 are made of."""
    A = np.asarray(A, dtype=np.float64)
    out = alpha * (A @ np.asarray(B, dtype=np.float64)) + gamma * np.eye(A.shape[0])
    if C is not None:
        out = out + beta * np.asarray(C, dtype=np.float64)
    return out


def fermi_exact(H, mu, beta):
    """U f_mu(Lambda) U^T by LAPACK diagonalisation -- what Eq. 8 approximates (used by the pins only)."""
    w, U = np.linalg.eigh(np.asarray(H, dtype=np.float64))
    return (U * fermi(w, mu, beta)) @ U.T
