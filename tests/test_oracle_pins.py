"""Pins for the CPU oracle (no GPU).  The paper prints no worked numeric example, so the oracle is
pinned to what the paper and the mathematics fix: the Fermi-step eigenprojector of Eq. 2 by a
brute-force Jacobi solver, closed forms, projector invariants, the scalar recursion on eigenvalues, invariances,
library routines for single steps, and hand-built threshold / overflow cases."""
from fractions import Fraction

import numpy as np
import pytest

from paper_2401_13772_b200 import hamiltonians as hm
from tests._pins import fermi_projector, gershgorin_np, jacobi_eigh, scalar_sp2


def relfro(A, B):
    return np.linalg.norm(A - B) / np.linalg.norm(B)


def fp_bound(st):
    """D = X_{m*} passed e_{m*} < tol; to first order ||X - D*||_F = ||X^2 - X||_F, so the distance to the exact
    projector is bounded by the recorded e_{m*} (plus round-off)."""
    return 1.1 * st["idem"][-1] + 1e-13


# ------------------------------------------------------------------ fixed point: brute force ----------
@pytest.mark.parametrize("N,n_occ,seed", [(8, 3, 1), (16, 8, 2), (33, 11, 3), (64, 40, 4)])
def test_fixed_point_vs_jacobi_eigenprojector(oracle_mod, N, n_occ, seed):
    H, _ = hm.planted_gap(N, n_occ, gap=1.0, width=2.0, seed=seed)
    w, V = jacobi_eigh(H)
    assert np.linalg.norm(V @ np.diag(w) @ V.T - H) < 1e-12 * np.linalg.norm(H)
    Dstar = fermi_projector(w, V, n_occ)
    D, st = oracle_mod.sp2_dense(H, n_occ, 1e-10)
    assert st["status"] == 0
    # D = X_{m*} is the iterate that PASSED the test e < tol, so to first order ||X - D*||_F = ||X^2 - X||_F
    # (|l^2 - l| ~ |l - round(l)| for eigenvalues l near 0 or 1): the error is bounded by the recorded e_{m*}.
    e_star = st["idem"][-1]
    assert e_star < 1e-10
    assert relfro(D, Dstar) <= fp_bound(st)
    # one more purification step lands on the projector to round-off (quadratic convergence)
    D2, st2 = oracle_mod.sp2_dense(H, n_occ, 1e-10 * max(e_star, 1e-6))
    assert relfro(D2, Dstar) <= 1e-13 or st2["status"] == 1


def test_jacobi_helper_against_lapack():
    H, eps = hm.planted_gap(24, 10, seed=7)
    w, _ = jacobi_eigh(H)
    assert np.allclose(w, np.linalg.eigvalsh(H), atol=1e-13)


# ------------------------------------------------------------------ closed forms ----------------------
def test_diagonal_H_gives_indicator_of_lowest_levels(oracle_mod):
    rng = np.random.default_rng(0)
    h = rng.permutation(np.concatenate([rng.uniform(-3, -1, 5), rng.uniform(1, 3, 7)]))
    D, st = oracle_mod.sp2_dense(np.diag(h), 5, 1e-12)
    assert st["status"] == 0
    expect = np.diag((h < 0).astype(float))
    assert np.abs(D - expect).max() < 1e-14
    # SP2 on a diagonal matrix IS the scalar recursion: same branch string
    bits, m_star, status, _, _ = scalar_sp2(h, 5, st["emin"], st["emax"], 1e-12)
    assert (bits, m_star, status) == (st["branch"], st["m_star"], 0)


@pytest.mark.parametrize("a,b", [(1.5, -1.0), (0.3, 2.0), (-0.7, 0.1)])
def test_two_by_two_closed_form(oracle_mod, a, b):
    H = np.array([[a, b], [b, -a]])
    D, st = oracle_mod.sp2_dense(H, 1, 1e-10)
    assert st["status"] == 0
    assert relfro(D, 0.5 * (np.eye(2) - H / np.sqrt(a * a + b * b))) <= fp_bound(st)


def test_worked_2x2_exact_rational_recursion_and_tie_break(oracle_mod):
    """H=[[1.5,-1],[-1,-1.5]], N_occ=1: Gershgorin [-2.5,2.5], X0=[[.2,.2],[.2,.8]], tr X0 == N_occ EXACTLY, so the
    '<=' of Listing 2 must pick 2X-X^2.  The recursion is replayed in exact rational arithmetic."""
    H = np.array([[1.5, -1.0], [-1.0, -1.5]])
    D, st = oracle_mod.sp2_dense(H, 1, 1e-10)
    assert (st["emin"], st["emax"]) == (-2.5, 2.5)
    X = [[Fraction(1, 5), Fraction(1, 5)], [Fraction(1, 5), Fraction(4, 5)]]
    bits, traces = "", []
    for m in range(st["n_products"]):
        t = X[0][0] + X[1][1]
        traces.append(float(t))
        P = [[sum(X[i][k] * X[k][j] for k in range(2)) for j in range(2)] for i in range(2)]
        if m == st["m_star"]:
            break
        b = t - 1 <= 0
        bits += "1" if b else "0"
        X = [[2 * X[i][j] - P[i][j] if b else P[i][j] for j in range(2)] for i in range(2)]
    assert bits[0] == "1" and traces[0] == 1.0
    assert st["branch"] == bits
    assert np.allclose(st["trace"], traces, rtol=0, atol=1e-14)
    assert np.abs(D - np.array([[float(v) for v in r] for r in X])).max() < 1e-14


def test_staggered_ring_closed_form_via_fft(oracle_mod):
    """Clean bipartite ring, staggered +/-Delta, NN hopping t: H^2 = T^2 + Delta^2 I is circulant, the gap is
    2*Delta with mu=0, so D = (I - H (H^2)^(-1/2))/2, with the circulant inverse square root done by FFT."""
    N, Delta = 64, 1.5
    H = hm.ring_dense(N, Delta, 0.0, 0.0)
    H2 = H @ H
    c = H2[0]
    assert all(np.allclose(np.roll(c, i), H2[i]) for i in range(N))
    g = np.real(np.fft.ifft(1.0 / np.sqrt(np.real(np.fft.fft(c)))))
    G = np.array([np.roll(g, i) for i in range(N)])
    Dexact = 0.5 * (np.eye(N) - H @ G)
    D, st = oracle_mod.sp2_dense(H, N // 2, 1e-10)
    assert st["status"] == 0
    assert relfro(D, Dexact) <= fp_bound(st)


# ------------------------------------------------------------------ invariants ------------------------
@pytest.fixture(scope="module")
def cfg1(oracle_mod):
    H = hm.make_dense("dense_n256")
    D, st = oracle_mod.sp2_dense(H, 128, 1e-10)
    return H, D, st


def _check_projector(H, D, n_occ, tol):
    assert abs(np.trace(D) - n_occ) <= 1e-9
    assert np.linalg.norm(D @ D - D) / np.linalg.norm(D) <= 10 * tol
    assert np.linalg.norm(H @ D - D @ H) / np.linalg.norm(H) <= 1e-12
    assert np.array_equal(D, D.T)
    assert np.abs(np.diag(D) - (D * D).sum(1)).max() <= 1e-12
    w = np.linalg.eigvalsh(D)
    assert np.all((np.abs(w) < 1e-9) | (np.abs(w - 1) < 1e-9))


def test_invariants_config1(cfg1):
    H, D, st = cfg1
    assert st["status"] == 0
    _check_projector(H, D, 128, 1e-10)


def test_invariants_small_long_range(oracle_mod):
    H = hm.small_long_range((8, 8, 6))
    n = H.shape[0]
    D, st = oracle_mod.sp2_dense(H, n // 2, 1e-10)
    assert st["status"] == 0
    _check_projector(H, D, n // 2, 1e-10)


# ------------------------------------------------------------------ branch sequence: scalar recursion -
def test_branch_string_vs_scalar_recursion_jacobi(oracle_mod):
    H, _ = hm.planted_gap(40, 17, gap=0.8, width=3.0, seed=11)
    w, _ = jacobi_eigh(H)
    D, st = oracle_mod.sp2_dense(H, 17, 1e-10)
    bits, m_star, status, tr, idem = scalar_sp2(w, 17, st["emin"], st["emax"], 1e-10)
    assert (st["branch"], st["m_star"], st["status"]) == (bits, m_star, status)
    assert np.allclose(st["trace"], tr, rtol=0, atol=1e-10)


def test_branch_string_vs_scalar_recursion_config1(cfg1):
    H, D, st = cfg1
    w = np.linalg.eigvalsh(H)  # LAPACK, cross-check only; never linked into the oracle
    bits, m_star, status, tr, idem = scalar_sp2(w, 128, st["emin"], st["emax"], 1e-10)
    assert (st["branch"], st["m_star"], st["status"]) == (bits, m_star, status)
    assert np.allclose(st["trace"], tr, rtol=0, atol=1e-9)
    # e_m of the matrix recursion equals the eigenvalue formula while it is above round-off
    big = idem > 1e-9
    assert np.allclose(st["idem"][big], idem[big], rtol=1e-6)


def test_config2_full_oracle_vs_scalar_recursion(oracle_mod):
    """BASELINE.json configs[1] end to end on the CPU (about 10 s): branch string, m*, invariants."""
    H = hm.make_dense("dense_n2048")
    D, st = oracle_mod.sp2_dense(H, 1024, 1e-10)
    w = np.linalg.eigvalsh(H)
    bits, m_star, status, tr, _ = scalar_sp2(w, 1024, st["emin"], st["emax"], 1e-10)
    assert (st["branch"], st["m_star"], st["status"]) == (bits, m_star, status)
    assert st["n_products"] == 19
    _check_projector(H, D, 1024, 1e-10)
    Vo = np.linalg.eigh(H)[1][:, :1024]
    assert relfro(D, Vo @ Vo.T) <= fp_bound(st)


# ------------------------------------------------------------------ invariances -----------------------
def test_shift_scale_and_permutation_invariance(oracle_mod):
    H = hm.small_long_range((6, 6, 4), seed=3)
    n = H.shape[0]
    D, st = oracle_mod.sp2_dense(H, n // 2, 1e-10)
    D2, st2 = oracle_mod.sp2_dense(2.0 * H + 0.75 * np.eye(n), n // 2, 1e-10)  # exact in binary floating point
    assert st2["branch"] == st["branch"] and st2["m_star"] == st["m_star"]
    assert relfro(D2, D) < 1e-12
    perm = np.random.default_rng(5).permutation(n)
    Hp = H[np.ix_(perm, perm)]
    Dp, stp = oracle_mod.sp2_dense(Hp, n // 2, 1e-10)
    assert stp["branch"] == st["branch"] and stp["m_star"] == st["m_star"]
    assert relfro(Dp, D[np.ix_(perm, perm)]) < 1e-12


# ------------------------------------------------------------------ single steps vs library routines --
def test_gershgorin_closed_form_and_numpy(oracle_mod):
    clean = hm.lattice_dense((16, 16, 8), 1.5, 0.0, 1.0, lambda r: -1.0)
    assert oracle_mod.gershgorin_dense(clean) == (-7.5, 7.5)  # +/-(Delta + 6|t|)
    H = hm.make_dense("dense_n2048")
    lo, hi = oracle_mod.gershgorin_dense(H)
    assert -7.7 <= lo and hi <= 7.7
    assert np.allclose((lo, hi), gershgorin_np(H), rtol=1e-15)
    v, ix, nz = hm.ellpack_from_dense(H[:128, :128], 128)
    assert np.allclose(oracle_mod.gershgorin_ellpack(v, ix, nz), gershgorin_np(H[:128, :128]), rtol=1e-15)


def test_x2_and_rescale_against_numpy(oracle_mod):
    rng = np.random.default_rng(1)
    A = rng.normal(size=(77, 77))
    X = A + A.T
    P = oracle_mod.x2_dense(X)
    assert np.abs(P - X @ X).max() < 1e-12 * np.abs(P).max()
    assert np.array_equal(P, P.T)  # bitwise symmetric: products commute, same k order
    r, c = rng.integers(0, 77, 50), rng.integers(0, 77, 50)
    assert np.allclose(oracle_mod.x2_dense_sampled(X, r, c), (X @ X)[r, c], rtol=1e-13, atol=1e-13)
    lo, hi = oracle_mod.gershgorin_dense(X)
    X0 = oracle_mod.rescale_dense(X, lo, hi)
    assert np.allclose(X0, (hi * np.eye(77) - X) / (hi - lo), rtol=1e-15, atol=1e-16)
    w = np.linalg.eigvalsh(X0)
    assert w.min() >= -1e-14 and w.max() <= 1 + 1e-14  # Eq. 5 maps the spectrum into [0,1]
    assert abs(oracle_mod.trace_dense(X0) - np.trace(X0)) < 1e-13


# ------------------------------------------------------------------ degenerate / failure cases --------
def test_status_codes(oracle_mod):
    H = hm.make_dense("dense_n256")
    assert oracle_mod.sp2_dense(3.0 * np.eye(8), 4, 1e-10)[1]["status"] == -2  # e_max == e_min
    assert oracle_mod.sp2_dense(H, 0, 1e-10)[1]["status"] == -1
    assert oracle_mod.sp2_dense(H, 256, 1e-10)[1]["status"] == -1
    assert oracle_mod.sp2_dense(H, 128, 0.0)[1]["status"] == -1
    Hb = H.copy()
    Hb[3, 5] += 1e-9
    assert oracle_mod.sp2_dense(Hb, 128, 1e-10)[1]["status"] == -5
    st = oracle_mod.sp2_dense(H, 128, 1e-10, max_products=5)[1]
    assert (st["status"], st["n_products"], st["m_star"]) == (2, 5, 4)


def test_gapless_metal_does_not_converge_but_terminates(oracle_mod):
    """SP2 has 'known challenges in the case of a vanishing electronic bandgap'.  A clean ring has doubly
    degenerate levels -2cos(2 pi k/N); N_occ = 2 cuts through the k = +/-1 pair, so the gap is exactly zero."""
    H = hm.ring_dense(64, 0.0, 0.0, 0.0)
    D, st = oracle_mod.sp2_dense(H, 2, 1e-10, max_products=60)
    assert st["status"] == 2 and st["n_products"] == 60 and st["idem"][-1] > 1e-2


# ------------------------------------------------------------------ ELLPACK-R: thresholds, overflow ---
def _ell(rows, N, M):
    v = np.zeros((N, M)); ix = np.zeros((N, M), dtype=np.int32); nz = np.zeros(N, dtype=np.int32)
    for i, r in enumerate(rows):
        for p, (j, x) in enumerate(r):
            ix[i, p], v[i, p] = j, x
        nz[i] = len(r)
    return v, ix, nz


def test_threshold_semantics_hand_built(oracle_mod):
    """keep iff |v| >= tau or j == i (P:74 'discard small matrix elements'; Eq. 15's '>= tau' sense)."""
    tau = 0.25
    # X = [[a, b, 0],[b, 0.5, c],[0, c, d]]: P_02 = b*c, P_00 = a^2+b^2, ...
    a, b, c, d = 0.125, 0.5, 0.5, 0.0625
    X = _ell([[(0, a), (1, b)], [(0, b), (1, 0.5), (2, c)], [(1, c), (2, d)]], 3, 3)
    pv, pi, pn, bad, mx = oracle_mod.x2_ellpack(*X, tau)
    P = hm.ellpack_to_dense(pv, pi, pn)
    Xd = hm.ellpack_to_dense(*X)
    full = Xd @ Xd
    assert full[0, 2] == 0.25 and P[0, 2] == 0.25  # exactly tau: kept
    assert bad == -1
    below = np.nextafter(tau, 1.0)  # a threshold one ulp above the value drops it
    pv2, pi2, pn2, _, _ = oracle_mod.x2_ellpack(*X, below)
    P2 = hm.ellpack_to_dense(pv2, pi2, pn2)
    assert P2[0, 2] == 0.0 and 2 not in pi2[0, : pn2[0]]
    # diagonal below tau is kept: P_22 = c^2 + d^2 = 0.2539 > tau; use a bigger tau
    pv3, pi3, pn3, _, _ = oracle_mod.x2_ellpack(*X, 10.0)
    assert [list(pi3[i, : pn3[i]]) for i in range(3)] == [[0], [1], [2]]
    assert np.allclose(np.diag(hm.ellpack_to_dense(pv3, pi3, pn3)), np.diag(full))
    # rows come out in ascending column order
    for i in range(3):
        assert list(pi[i, : pn[i]]) == sorted(pi[i, : pn[i]])


def test_update_union_pattern_and_threshold(oracle_mod):
    X = _ell([[(0, 1.0), (2, 0.5)], [(1, 0.2)], [(0, 0.5), (2, 0.3)]], 3, 3)
    P = _ell([[(0, 0.9), (1, 0.3)], [(1, 0.39)], [(2, 0.1)]], 3, 3)
    ov, oi, on, bad, mx = oracle_mod.update_ellpack(X, P, 0.05)
    got = hm.ellpack_to_dense(ov, oi, on)
    want = 2 * hm.ellpack_to_dense(*X) - hm.ellpack_to_dense(*P)
    want[np.abs(want) < 0.05] = 0.0
    want[1, 1] = 2 * 0.2 - 0.39  # diagonal kept although |0.01| < tau
    assert np.array_equal(got, want) and bad == -1
    assert list(oi[1, : on[1]]) == [1]


def test_sparse_tau0_equals_dense_oracle(oracle_mod):
    H = hm.small_long_range((6, 5, 4), seed=2)
    n = H.shape[0]
    D, st = oracle_mod.sp2_dense(H, n // 2, 1e-10)
    (dv, di, dn), sts = oracle_mod.sp2_ellpack(*hm.ellpack_from_dense(H, n), n // 2, 1e-10, 0.0)
    assert sts["status"] == 0 and sts["branch"] == st["branch"] and sts["m_star"] == st["m_star"]
    assert relfro(hm.ellpack_to_dense(dv, di, dn), D) < 1e-13
    assert np.allclose(sts["trace"], st["trace"], rtol=0, atol=1e-11)


def test_sparse_row_order_invariance(oracle_mod):
    """'the ELLPACK-R format is unsorted' — shuffling entries within input rows must not change D."""
    v, ix, nz = hm.small_sparse_model((8, 8, 7), M=512)
    n = v.shape[0]
    (dv, di, dn), st = oracle_mod.sp2_ellpack(v, ix, nz, n // 2, 1e-8, 1e-6)
    rng = np.random.default_rng(9)
    v2, ix2 = v.copy(), ix.copy()
    for i in range(n):
        p = rng.permutation(nz[i])
        v2[i, : nz[i]], ix2[i, : nz[i]] = v[i, p], ix[i, p]
    (ev, ei, en), st2 = oracle_mod.sp2_ellpack(v2, ix2, nz, n // 2, 1e-8, 1e-6)
    assert st2["branch"] == st["branch"] and st2["status"] == st["status"]
    assert np.array_equal(ei, di) and np.array_equal(en, dn) and np.array_equal(ev, dv)


def test_sparse_thresholded_sp2_close_to_exact_projector(oracle_mod):
    v, ix, nz = hm.small_sparse_model((8, 8, 7), M=512)
    n = v.shape[0]
    H = hm.ellpack_to_dense(v, ix, nz)
    (dv, di, dn), st = oracle_mod.sp2_ellpack(v, ix, nz, n // 2, 1e-8, 1e-6)
    assert st["status"] in (0, 1)
    Vo = np.linalg.eigh(H)[1][:, : n // 2]
    D = hm.ellpack_to_dense(dv, di, dn)
    assert relfro(D, Vo @ Vo.T) < 1e-4  # truncation-limited, not round-off limited
    assert abs(np.trace(D) - n // 2) < 1e-4
    assert np.abs(D - D.T).max() < 1e-5


def test_ellpack_overflow_is_a_failure(oracle_mod):
    """a growing number of non-zeroes 'may reach the limit M and lead to a failure'."""
    v, ix, nz = hm.lattice_ellpack((8, 8, 8), 1.5, 0.2, 2.0, lambda r: -np.exp(-r), 64)  # 33/row; X0^2 has > 64
    (dv, di, dn), st = oracle_mod.sp2_ellpack(v, ix, nz, 256, 1e-8, 1e-6)
    assert st["status"] == -3 and st["overflow_row"] == 0 and st["n_products"] == 1
    assert st["max_row_nnz"][0] > 64


def test_config5_literal_overflows_at_product0_with_fill_829(oracle_mod):
    """BASELINE.json configs[4] as literally written: the 123-point r<=3 stencil convolved with itself has 829
    points, all >= 1e-6 after the rescale, so M=512 overflows at the first product."""
    v, ix, nz = hm.make_ellpack("ellpack_n65536_literal")
    lo, hi = oracle_mod.gershgorin_ellpack(v, ix, nz)
    assert abs(lo + 15.892109) < 1e-5 and abs(hi - 15.892112) < 1e-5
    xv, xi, xn, bad = oracle_mod.rescale_ellpack(v, ix, nz, lo, hi)
    assert bad == -1
    pv, pi, pn, bad, mx = oracle_mod.x2_ellpack(xv, xi, xn, 1e-6)
    assert bad == 0 and mx == 829


# ------------------------------------------------------------------ rule R1 == variant R2 -------------
@pytest.mark.parametrize("seed,N,n_occ", [(21, 48, 7), (22, 48, 24), (23, 61, 50)])
def test_rule_R1_picks_the_candidate_whose_trace_is_nearer_n_occ(oracle_mod, seed, N, n_occ):
    """DESIGN.md reading 4: with a = tr X - n_occ and d = tr X - tr X^2 >= 0 the two candidates of Eq. 6-7 have traces
    n_occ + a - d (X^2) and n_occ + a + d (2X - X^2), so "take the candidate whose trace is nearer n_occ" (variant R2 of
    P:169's "other variants") is a < 0 => 2X - X^2, a > 0 => X^2: Listing 2's rule except on the tie a = 0.
    Brute force: replay the oracle's branch string with numpy and form BOTH candidates at every step."""
    H, _ = hm.planted_gap(N, n_occ, gap=0.6, width=4.0, seed=seed)
    D, st = oracle_mod.sp2_dense(H, n_occ, 1e-10)
    assert st["status"] == 0
    X = (st["emax"] * np.eye(N) - H) / (st["emax"] - st["emin"])
    for m in range(st["m_star"]):
        P = X @ X
        cand = (P, 2.0 * X - P)                        # b = 0, b = 1
        dist = [abs(np.trace(c) - n_occ) for c in cand]
        b = int(st["branch"][m])
        assert dist[b] <= dist[1 - b]
        assert abs(np.trace(X) - st["trace"][m]) <= 1e-10
        assert np.trace(X) - np.trace(P) >= -1e-12     # d >= 0: the spectrum of X lies in [0, 1]
        X = cand[b]
    assert relfro(X, D) <= 1e-10


# ---------------------------------------------------------------------------------------------------------------
# Pins added in round 2 ("parity unpinned" items i and ii)
# ---------------------------------------------------------------------------------------------------------------
def test_rescale_ellpack_inserts_a_missing_diagonal_hand_example(oracle_mod):
    """Eq. 5 on ELLPACK-R with a row whose diagonal is NOT stored (H_11 = 0): the diagonal slot must appear,
    in ascending-column position, with value s (e_max - 0).  Every expected slot and value is written out by hand:
    e_min = -2, e_max = 3, s = 1 / 5."""
    M = 4
    hv = np.zeros((3, M)); hi = np.zeros((3, M), dtype=np.int32); hn = np.zeros(3, dtype=np.int32)
    # row 0: (0, 2.0), (1, 1.0)      row 1 (unsorted, no diagonal): (2, -0.5), (0, 1.0)      row 2: (1, -0.5), (2, -1.0)
    hv[0, :2] = [2.0, 1.0]; hi[0, :2] = [0, 1]; hn[0] = 2
    hv[1, :2] = [-0.5, 1.0]; hi[1, :2] = [2, 0]; hn[1] = 2
    hv[2, :2] = [-0.5, -1.0]; hi[2, :2] = [1, 2]; hn[2] = 2
    xv, xi, xn, bad = oracle_mod.rescale_ellpack(hv, hi, hn, -2.0, 3.0)
    assert bad < 0
    assert xn.tolist() == [2, 3, 2]
    assert xi.tolist() == [[0, 1, 0, 0], [0, 1, 2, 0], [1, 2, 0, 0]]
    s = 1.0 / (3.0 - -2.0)
    want = [[s * (3.0 - 2.0), -s * 1.0, 0.0, 0.0],           # X_00 = s (e_max - H_00), X_01 = -s H_01
            [-s * 1.0, s * (3.0 - 0.0), -s * -0.5, 0.0],     # inserted X_11 = s e_max = 0.6 between columns 0 and 2
            [-s * -0.5, s * (3.0 - -1.0), 0.0, 0.0]]
    assert xv.tolist() == want
    assert want[1][1] == 0.6000000000000001 and want[1][2] == 0.1           # the literal numbers
    assert oracle_mod.trace_ellpack(xv, xi, xn) == pytest.approx(0.2 + 0.6 + 0.8, abs=1e-15)
    # a full row without its diagonal cannot take the inserted slot: that row is reported, lowest first
    hv2 = np.ones((2, 2)); hi2 = np.array([[1, 0], [0, 0]], dtype=np.int32); hn2 = np.array([2, 1], dtype=np.int32)
    hi2[1, 0] = 0                                             # row 1 = {(0, 1.0)}: one free slot, diagonal fits
    hv3 = np.ones((2, 1)); hi3 = np.array([[1], [0]], dtype=np.int32); hn3 = np.array([1, 1], dtype=np.int32)
    assert oracle_mod.rescale_ellpack(hv2, hi2, hn2, -2.0, 3.0)[3] < 0
    assert oracle_mod.rescale_ellpack(hv3, hi3, hn3, -2.0, 3.0)[3] == 0      # M = 1, both rows lack the diagonal


def test_idempotency_norm_over_the_union_of_two_different_patterns(oracle_mod):
    """Reading 8: e_m = ||thr(X X) - X||_F / ||X||_F runs over the UNION of the two patterns, an absent entry counting as
    0.  A small random sparse H and a large tau give entries that are in X only (their product entry was dropped) and
    entries in thr(X X) only (fill-in); the expected value is computed in exact rational arithmetic from the definition
    on the dense 8 x 8 matrices -- no sparse merge, no floating point."""
    from fractions import Fraction

    N, M, tau = 8, 8, 0.02
    rng = np.random.default_rng(11)
    A = np.zeros((N, N))
    for i in range(N):
        A[i, i] = rng.uniform(-1, 1)
        for j in (i + 1, i + 3):
            if j < N:
                A[i, j] = A[j, i] = rng.uniform(-1, 1)
    H = hm.ellpack_from_dense(A, M)
    lo, hi = oracle_mod.gershgorin_ellpack(*H)
    xv, xi, xn, bad = oracle_mod.rescale_ellpack(*H, lo, hi)
    assert bad < 0
    X = [[Fraction(0)] * N for _ in range(N)]
    inX = [[False] * N for _ in range(N)]
    for i in range(N):
        for p in range(xn[i]):
            X[i][xi[i, p]] = Fraction(float(xv[i, p]))
            inX[i][xi[i, p]] = True
    e2 = x2 = Fraction(0)
    only_x = only_p = 0
    for i in range(N):
        for j in range(N):
            touched = any(inX[i][k] and inX[k][j] for k in range(N))
            pij = sum(X[i][k] * X[k][j] for k in range(N))
            keep = touched and (abs(pij) >= Fraction(tau) or i == j)
            only_x += inX[i][j] and not keep
            only_p += keep and not inX[i][j]
            e2 += ((pij if keep else 0) - X[i][j]) ** 2
            x2 += X[i][j] ** 2
    assert only_x >= 2 and only_p >= 2          # the case exercises both kinds of mismatch
    _, st = oracle_mod.sp2_ellpack(*H, N // 2, 1e-12, tau, max_products=1)
    assert st["n_products"] == 1
    want = float(e2) ** 0.5 / float(x2) ** 0.5
    assert st["idem"][0] == pytest.approx(want, rel=1e-13)
    # and the two norms move the value: ignoring either kind of one-sided entry would miss by far more than 1e-13
    e2_wrong = sum(((sum(X[i][k] * X[k][j] for k in range(N)) - X[i][j]) ** 2 for i in range(N) for j in range(N)
                    if inX[i][j]), Fraction(0))
    assert abs(float(e2_wrong) ** 0.5 / float(x2) ** 0.5 - want) > 1e-6
