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


def fit_joint(resp, gc, b, ic_meas, sigma, sigma_ic, lam):
    """Joint fit of the basis coefficients and the coil currents, Eq. 7: the coil
    currents become free parameters I_C' and the measured currents enter as extra rows,

        [ R   G_C ] [ X    ]   [ b   ]
        [ 0    I  ] [ I_C' ] = [ I_C ]

    (the printed Eq. 7 stacks [R; G_C] as one column; dimensionally it must be this block matrix --
    SURVEY.md 8(c) O5, reading O5b).  Weights: measurement rows 1/sigma (as in fit), coil
    rows 1/sigma_ic (the paper gives no weights).  The Tikhonov term of fit() acts on X only, in the same
    equilibrated coordinates.  Householder QR of the stacked system.
    Returns (X, I_C', chi2 over the measurement rows, status)."""
    M, nb = resp.shape
    nc = gc.shape[1]
    A1 = resp / sigma[:, None]
    A2 = gc / sigma[:, None]
    y = np.concatenate([b / sigma, ic_meas / sigma_ic])
    X = np.zeros(nb)
    icf = np.array(ic_meas, np.float64, copy=True)
    if not (np.all(np.isfinite(A1)) and np.all(np.isfinite(y))):
        return X, icf, np.nan, 2
    s = np.sqrt(np.sum(A1 * A1, axis=0))
    keep = s > 0.0
    if not keep.any():
        return X, icf, np.nan, 3
    k = int(keep.sum())
    top = np.hstack([A1[:, keep] / s[keep], A2])                       # measurement rows
    mid = np.hstack([np.zeros((nc, k)), np.diag(1.0 / sigma_ic)])      # measured coil currents
    bot = np.hstack([lam * np.sqrt(M) * np.eye(k), np.zeros((k, nc))])  # regularisation of X
    S = np.vstack([top, mid, bot])
    t = np.sqrt(np.sum(S[:, k:] ** 2, axis=0))                          # coil columns equilibrated too
    S[:, k:] /= t
    rhs = np.concatenate([y, np.zeros(k)])
    Q, Rm = np.linalg.qr(S)
    dg = np.abs(np.diag(Rm))
    if np.any(dg < 1e-13 * dg[0]):
        return X, icf, np.nan, 3
    sol = np.linalg.solve(Rm, Q.T @ rhs)
    X[keep] = sol[:k] / s[keep]
    icf = sol[k:] / t
    res = A1 @ X + A2 @ icf - b / sigma
    return X, icf, float(res @ res), 0
