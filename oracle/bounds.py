"""CPU oracle for the tighter spectral bounds -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain numpy, FP64.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this module; it imports nothing from ``paper_2401_13772_b200``.

Eq. 5 of the paper rescales H with its EXACT extreme eigenvalues eps_1, eps_N; Listing 2 consumes unexplained
`emin`, `emax` and the only bound the paper names is Gershgorin's, which is what the SP2 path uses by
default (reading 1).  Gershgorin is loose by a factor ~2 on the long-range models, which costs SP2 about a third more
products.  This module is the optional tighter bound:

    K steps of the Lanczos recursion on H from a fixed pseudo-random start vector           (textbook Lanczos)
    T_K = tridiag(alpha_0..alpha_{K-1}; beta_1..beta_{K-1}),  (theta_i, s_i) its eigenpairs  (LAPACK)
    r_max = |beta_K s_{K-1,max}|, r_min = |beta_K s_{K-1,min}|                               (Ritz residual norms)
    e_max = min(Gershgorin, theta_max + r_max + pad),  e_min = max(Gershgorin, theta_min - r_min - pad),
    pad = 0.01 (theta_max - theta_min)

Readings (DESIGN.md "Readings" B1-B3):
  B1. theta_max + r_max is the safeguarded upper bound of Zhou & Li's k-step Lanczos estimator: an eigenvalue lies
      within r of every Ritz value, and for the extreme Ritz values of a generic start vector that eigenvalue is the
      extreme one.  It is not a theorem for every start vector, hence the pad of 1% of the Ritz width, and the result is
      never looser than Gershgorin.  The pins check enclosure on every model in this repository for K >= 8 (with K = 2..4
      an outlying band is missed on three of them, which is why the product interface rejects K < 8).
  B2. The start vector is counter-based so that the oracle and the CUDA path draw the same numbers without sharing
      code: u_i = 2 * (splitmix64(seed + i) >> 11) * 2^-53 - 1, v_0 = u / ||u||.
  B3. Full reorthogonalisation: after the three-term step, w is orthogonalised against ALL previous Lanczos vectors by
      two passes of classical Gram-Schmidt.  Without it the recursion loses orthogonality as soon as one extreme Ritz
      value converges, and the residual term |beta_K s_K| of the other end is then reproduced to two digits only -- two
      correct implementations would disagree by 1e-3 of the width (measured).  With it the tridiagonal matrix is
      reproducible to round-off.  alpha_j is the coefficient of the three-term step (the Gram-Schmidt corrections are
      not folded into it).  An exact breakdown (beta_{j+1} = 0) ends the recursion with K = j + 1.
"""
from __future__ import annotations

import numpy as np

from . import chebyshev as _och

_MASK = (1 << 64) - 1


def splitmix64(x: int) -> int:
    """One step of the SplitMix64 generator (Steele, Lea, Flood 2014) on the 64-bit counter x."""
    x = (x + 0x9E3779B97F4A7C15) & _MASK
    z = x
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return z ^ (z >> 31)


def start_vector(N: int, seed: int = 0):
    """u_i of reading B2, not normalised."""
    return np.array([2.0 * ((splitmix64(seed + i) >> 11) * 2.0 ** -53) - 1.0 for i in range(N)])


def lanczos(H, K: int, seed: int = 0):
    """K steps of the Lanczos recursion (reading B3).  Returns (alpha[K'], beta[K' + 1]) with beta[0] = 0 and
    beta[K'] the norm of the last residual; K' < K after a breakdown."""
    H = np.asarray(H, dtype=np.float64)
    N = H.shape[0]
    u = start_vector(N, seed)
    v = u / np.sqrt(np.dot(u, u))
    v_prev = np.zeros(N)
    alpha, beta = [], [0.0]
    V = []
    for j in range(min(K, N)):
        V.append(v)
        w = H @ v
        a = float(np.dot(v, w))
        w = w - a * v - beta[j] * v_prev
        for _ in range(2):                                   # two passes of classical Gram-Schmidt (reading B3)
            c = [float(np.dot(q, w)) for q in V]
            for ci, q in zip(c, V):
                w = w - ci * q
        b = float(np.sqrt(np.dot(w, w)))
        alpha.append(a)
        beta.append(b)
        if b == 0.0:
            break
        v_prev, v = v, w / b
    return np.array(alpha), np.array(beta)


def lanczos_bounds(H, K: int, seed: int = 0):
    """(e_min, e_max) of the module docstring for a dense symmetric H.  Returns (e_min, e_max, info)."""
    H = np.asarray(H, dtype=np.float64)
    glo, ghi = _och.gershgorin(H)
    alpha, beta = lanczos(H, K, seed)
    Kp = alpha.size
    T = np.diag(alpha) + np.diag(beta[1:Kp], 1) + np.diag(beta[1:Kp], -1)
    theta, S = np.linalg.eigh(T)
    r_min, r_max = abs(beta[Kp] * S[Kp - 1, 0]), abs(beta[Kp] * S[Kp - 1, Kp - 1])
    pad = 0.01 * (theta[Kp - 1] - theta[0])
    lo = max(glo, theta[0] - r_min - pad)
    hi = min(ghi, theta[Kp - 1] + r_max + pad)
    return float(lo), float(hi), {"alpha": alpha, "beta": beta, "theta": theta, "r_min": r_min, "r_max": r_max,
                                  "gershgorin": (glo, ghi), "steps": Kp}
