"""Textbook fp64 Krylov iterations for the reference tier of the oracle.  Test infrastructure only.

``lanczos_sqrt``  y = A^{1/2} w for a symmetric positive definite operator, Chow & Saad (ref. 28 of the paper, PAPER.md:427,
                  912): v_1 = w/|w|, T_m = V_m^T A V_m tridiagonal, y_m = |w| V_m T_m^{1/2} e_1; full re-orthogonalisation
                  (this is a checker, not a fast code), stop when |y_m - y_{m-1}| <= tol |y_m|.
``gmres``         x with |b - A x| <= tol |b|, no restart, x_0 = 0: Arnoldi with modified Gram-Schmidt (twice) and the small
                  least-squares problem solved by numpy at every iteration.
Shares nothing with paper_1709_06946_b200/csrc/krylov.cu.
"""
import numpy as np
from scipy.linalg import eigh_tridiagonal


def lanczos_sqrt(matvec, w, tol=1e-10, maxit=300):
    w = np.asarray(w, dtype=np.float64).ravel()
    wn = np.linalg.norm(w)
    if wn == 0.0:
        return np.zeros_like(w), 0
    V = [w / wn]
    alpha, beta = [], []
    y_prev = None
    for m in range(1, maxit + 1):
        u = np.asarray(matvec(V[-1]), dtype=np.float64).ravel()
        alpha.append(float(V[-1] @ u))
        u = u - alpha[-1] * V[-1] - (beta[-1] * V[-2] if beta else 0.0)
        for _ in range(2):                                   # full re-orthogonalisation
            for v in V:
                u -= (v @ u) * v
        lam, Q = eigh_tridiagonal(np.array(alpha), np.array(beta)) if m > 1 else (np.array(alpha), np.ones((1, 1)))
        coef = wn * (Q * np.sqrt(np.clip(lam, 0.0, None))) @ Q[0]          # |w| T^{1/2} e_1
        y = np.stack(V, axis=1) @ coef
        if y_prev is not None and np.linalg.norm(y - y_prev) <= tol * np.linalg.norm(y):
            return y, m
        y_prev = y
        b = float(np.linalg.norm(u))
        if b <= 1e-14 * abs(alpha[0]):
            return y, m
        beta.append(b)
        V.append(u / b)
    raise RuntimeError('lanczos_sqrt: no convergence')


def gmres(matvec, b, tol=1e-10, maxit=200):
    b = np.asarray(b, dtype=np.float64).ravel()
    bn = np.linalg.norm(b)
    if bn == 0.0:
        return np.zeros_like(b), 0
    V = [b / bn]
    H = np.zeros((maxit + 1, maxit))
    for m in range(1, maxit + 1):
        u = np.asarray(matvec(V[-1]), dtype=np.float64).ravel()
        for _ in range(2):
            for j, v in enumerate(V):
                hj = float(v @ u)
                H[j, m - 1] += hj
                u = u - hj * v
        H[m, m - 1] = np.linalg.norm(u)
        e1 = np.zeros(m + 1); e1[0] = bn
        y, *_ = np.linalg.lstsq(H[:m + 1, :m], e1, rcond=None)
        res = np.linalg.norm(H[:m + 1, :m] @ y - e1)
        if res <= tol * bn or H[m, m - 1] <= 1e-300:
            return np.stack(V, axis=1) @ y, m
        V.append(u / H[m, m - 1])
    raise RuntimeError('gmres: no convergence')
