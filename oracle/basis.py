"""Polynomial P'/FF' current basis with edge subtraction (Eq. 8-11).

Oracle-side (test infrastructure).  Reading of the garbled Eq. 8-11 (O4): "p' with k
terms" means N_P' = k and k coefficients a_0..a_{k-1}, columns R (x^i - x^k), i = 0..k-1;
FF' likewise with factor mu0/R (Eq. 10).  Columns are multiplied by the plasma mask and by
dA = dR dZ so that J_b X is the filament current of every node in amperes (Eq. 2 is written
with the area element implicit).
"""
import numpy as np

MU0 = 4.0e-7 * np.pi


def basis_columns(psin, mask, r, dA, n_p, n_ff):
    """J_b[nz, nr, n_p+n_ff] per Eq. 10."""
    nz, nr = psin.shape
    R = np.broadcast_to(r[None, :], (nz, nr))
    x = psin
    cols = []
    for i in range(n_p):
        cols.append(R * (x ** i - x ** n_p))
    for j in range(n_ff):
        cols.append(MU0 / R * (x ** j - x ** n_ff))
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
