"""Independent reference computations used to PIN the oracle (none of them calls oracle/ or the CUDA path).

* ``jacobi_eigh``      — brute-force cyclic Jacobi eigensolver (textbook), for tiny N.
* ``fermi_projector``  — D* = sum_{i<=N_occ} v_i v_i^T, Eq. 2 of the paper with the beta->infinity step function
                         (PAPER.md P:118-126).
* ``scalar_sp2``       — the SP2 recursion Eq. 5-7 applied to a vector of eigenvalues: in exact arithmetic
                         tr X_m = sum_i f_m(lambda_i) and ||X_m^2 - X_m||_F^2 = sum_i (f_m^2 - f_m)^2, so the branch
                         string and m* of the matrix recursion must agree with it whenever margins >> round-off.
"""
import numpy as np


def jacobi_eigh(A, tol=1e-15, max_sweeps=60):
    A = np.array(A, dtype=np.float64, copy=True)
    n = A.shape[0]
    V = np.eye(n)
    for _ in range(max_sweeps):
        off = np.linalg.norm(A - np.diag(np.diag(A)))
        if off < tol * max(1.0, np.linalg.norm(A)):
            break
        for p in range(n - 1):
            for q in range(p + 1, n):
                if abs(A[p, q]) < 1e-300:
                    continue
                theta = (A[q, q] - A[p, p]) / (2.0 * A[p, q])
                t = np.sign(theta) / (abs(theta) + np.sqrt(theta * theta + 1.0)) if theta != 0 else 1.0
                c = 1.0 / np.sqrt(t * t + 1.0)
                s = t * c
                Ap, Aq = A[:, p].copy(), A[:, q].copy()
                A[:, p], A[:, q] = c * Ap - s * Aq, s * Ap + c * Aq
                Ap, Aq = A[p, :].copy(), A[q, :].copy()
                A[p, :], A[q, :] = c * Ap - s * Aq, s * Ap + c * Aq
                Vp, Vq = V[:, p].copy(), V[:, q].copy()
                V[:, p], V[:, q] = c * Vp - s * Vq, s * Vp + c * Vq
    w = np.diag(A).copy()
    order = np.argsort(w)
    return w[order], V[:, order]


def fermi_projector(w, V, n_occ):
    Vo = V[:, :n_occ]
    return Vo @ Vo.T


def gershgorin_np(H):
    d = np.diag(H)
    rad = np.abs(H).sum(1) - np.abs(d)
    return float((d - rad).min()), float((d + rad).max())


def scalar_sp2(eigs, n_occ, emin, emax, tol, max_products=100):
    lam = (emax - np.asarray(eigs, dtype=np.longdouble)) / (emax - emin)
    bits, tr, idem = [], [], []
    status = 2
    for m in range(max_products):
        t = lam.sum()
        l2 = lam * lam
        e = np.sqrt(((l2 - lam) ** 2).sum()) / np.sqrt(l2.sum())
        tr.append(float(t))
        idem.append(float(e))
        if e < tol:
            status = 0
            break
        if m >= 2 and e < 1e-2 and e >= idem[m - 2]:
            status = 1
            break
        if m + 1 == max_products:
            break
        b = 1 if t - n_occ <= 0 else 0
        bits.append(str(b))
        lam = 2 * lam - l2 if b else l2
    return "".join(bits), len(tr) - 1, status, np.array(tr), np.array(idem)
