"""Polynomial P'/FF' current basis with edge subtraction (Eq. 8-11).

Oracle-side (test infrastructure).  Reading of the garbled Eq. 8-11 (O4): "p' with k
terms" means N_P' = k and k coefficients a_0..a_{k-1}, columns R (x^i - x^k), i = 0..k-1;
FF' likewise with factor mu0/R (Eq. 10).  Columns are multiplied by the plasma mask and by
dA = dR dZ so that J_b X is the filament current of every node in amperes (Eq. 2 is written
with the area element implicit).
"""
import numpy as np

MU0 = 4.0e-7 * np.pi


def tension_spline_cardinals(x, knots, tau):
    """Cardinal tension splines phi_q(x), q = 0..len(knots)-1, on the knot set `knots`.

    BASELINE.json configs[4] names "5-knot tension-spline FF' edge terms"; they are NOT in the
    paper, so the definition is SURVEY.md 8(c) O4's (reading O4c): on every knot
    interval the fourth derivative of phi equals tau^2 times its second derivative, phi is C2
    across the knots, phi_q(k_r) = delta_qr, the second derivative vanishes at both end knots,
    and phi_q(x) = 0 for x outside [k_0, k_last].
    Closed form on [k_r, k_r + h], t = (x - k_r)/h, with m = second derivative at the knots:
      y_r (1-t) + y_{r+1} t + (m_r/tau^2) [sinh(tau h (1-t))/sinh(tau h) - (1-t)]
                             + (m_{r+1}/tau^2) [sinh(tau h t)/sinh(tau h) - t],
    and m solves the tridiagonal system that makes the first derivative continuous:
      a_{r-1} m_{r-1} + (b_{r-1} + b_r) m_r + a_r m_{r+1} = (y_{r+1}-y_r)/h_r - (y_r-y_{r-1})/h_{r-1},
      a_r = (1/h_r - tau/sinh(tau h_r))/tau^2,  b_r = (tau cosh(tau h_r)/sinh(tau h_r) - 1/h_r)/tau^2.
    Returns an array of shape x.shape + (len(knots),)."""
    k = np.asarray(knots, np.float64)
    n = len(k)
    h = np.diff(k)
    a = (1.0 / h - tau / np.sinh(tau * h)) / tau**2
    b = (tau * np.cosh(tau * h) / np.sinh(tau * h) - 1.0 / h) / tau**2
    T = np.zeros((n, n))
    T[0, 0] = T[n - 1, n - 1] = 1.0                      # natural ends: m = 0
    for r in range(1, n - 1):
        T[r, r - 1], T[r, r], T[r, r + 1] = a[r - 1], b[r - 1] + b[r], a[r]
    Y = np.eye(n)                                        # column q = knot values of phi_q
    rhs = np.zeros((n, n))
    rhs[1:-1] = (Y[2:] - Y[1:-1]) / h[1:, None] - (Y[1:-1] - Y[:-2]) / h[:-1, None]
    Mq = np.linalg.solve(T, rhs)                         # Mq[r, q] = second derivative of phi_q at k_r
    x = np.asarray(x, np.float64)
    r = np.clip(np.searchsorted(k, x, side="right") - 1, 0, n - 2)
    hr = h[r]
    t = np.clip((x - k[r]) / hr, 0.0, 1.0)       # outside [k_0, k_last] the value is zeroed below
    sh = np.sinh(tau * hr)
    A = np.sinh(tau * hr * (1.0 - t)) / sh - (1.0 - t)
    Bc = np.sinh(tau * hr * t) / sh - t
    out = (Y[r] * (1.0 - t)[..., None] + Y[r + 1] * t[..., None]
           + Mq[r] * (A / tau**2)[..., None] + Mq[r + 1] * (Bc / tau**2)[..., None])
    inside = (x >= k[0]) & (x <= k[-1])
    return out * inside[..., None]


def basis_columns(psin, mask, r, dA, n_p, n_ff, spline=None):
    """J_b[nz, nr, n_p+n_ff(+n_spline)] per Eq. 10.  spline = dict(knots, tension,
    terms) appends FF'-type columns (mu0/R) phi_q(x) dA for q in terms (config 5 only)."""
    nz, nr = psin.shape
    R = np.broadcast_to(r[None, :], (nz, nr))
    x = psin
    cols = []
    for i in range(n_p):
        cols.append(R * (x ** i - x ** n_p))
    for j in range(n_ff):
        cols.append(MU0 / R * (x ** j - x ** n_ff))
    if spline is not None:
        phi = tension_spline_cardinals(x, spline["knots"], spline["tension"])
        for q in spline["terms"]:
            cols.append(MU0 / R * phi[..., q])
    Jb = np.stack(cols, axis=-1) * dA
    return Jb * mask[..., None]


def delz_column(Jb_poly, X_prev, nz, nr, dz):
    """Vertical-shift term (reading O4b; not in the paper, which only notes that the
    Picard iteration displaces the plasma vertically).  With I' = J_b(psin^k) X^{k-1}
    the node currents the previous coefficients give on the current flux map,
    column[j, i] = -(I'[j+1, i] - I'[j-1, i]) / (2 dZ)   (amperes per metre of upward shift),
    zero on the first and last row.  Jb_poly is [nz*nr, n_p+n_ff]."""
    Ip = (Jb_poly @ X_prev).reshape(nz, nr)
    col = np.zeros((nz, nr))
    col[1:-1, :] = -(Ip[2:, :] - Ip[:-2, :]) / (2.0 * dz)
    return col.reshape(-1)
