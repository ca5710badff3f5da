"""Least-squares fit of the basis coefficients, R X = b - G_C I_C (Eq. 6;
PAPER.md:116 for the solver choice).

Oracle-side (test infrastructure).  The paper names normal equations and Gram-Schmidt QR; the
oracle uses neither: Householder QR (LAPACK via numpy) of the stacked, column-equilibrated,
Tikhonov-augmented matrix (reading O5; weights, scaling, lambda and chi^2 are not in
the paper; lambda = 0 reproduces Eq. 6 exactly).
"""
import numpy as np


def fit(resp, d, sigma, lam):
    """minimise |W (resp X - d)|^2 + lam^2 M sum_l (s_l X_l)^2, W = diag(1/sigma),
    s_l = |W resp[:, l]|_2.  Returns (X, chi2, status) ; status 3 = rank deficient."""
    M, nb = resp.shape
    A = resp / sigma[:, None]
    y = d / sigma
    s = np.sqrt(np.sum(A * A, axis=0))
    keep = s > 0.0
    X = np.zeros(nb)
    finite = np.all(np.isfinite(A)) and np.all(np.isfinite(y))
    if not finite:
        return X, np.nan, 2          # include/ptefit.h: status 2 = non-finite data
    if not keep.any():
        return X, np.nan, 3          # status 3 = singular fit
    Ae = A[:, keep] / s[keep]
    k = Ae.shape[1]
    S = np.vstack([Ae, lam * np.sqrt(M) * np.eye(k)])
    rhs = np.concatenate([y, np.zeros(k)])
    Q, Rm = np.linalg.qr(S)
    dg = np.abs(np.diag(Rm))
    if np.any(dg < 1e-13 * dg[0]):
        return X, np.nan, 3
    xe = np.linalg.solve(Rm, Q.T @ rhs)
    X[keep] = xe / s[keep]
    res = A @ X - y
    return X, float(res @ res), 0
