"""Finite-difference Grad-Shafranov solve, Delta* psi = -mu0 R J_phi (Eq. 1,
PAPER.md:118-120 Sec. II.C), by a banded LU of the full 5-point ("pentadiagonal") matrix.

Oracle-side (test infrastructure).  The paper says only "finite differences ... pentadiagonal
... Dirichlet boundary conditions"; reading O6 fixes the EFIT-style centred stencil

  (1+dR/2R_i)/dR^2 psi[i-1,j] + (1-dR/2R_i)/dR^2 psi[i+1,j] - (2/dR^2+2/dZ^2) psi[i,j]
     + (psi[i,j-1] + psi[i,j+1])/dZ^2 = -mu0 R_i I[i,j]/dA

i.e. Delta* = d2/dR2 - (1/R) d/dR + d2/dZ2 with centred differences.  The product path solves
the same linear system by DST-in-Z + tridiagonal-in-R; this file deliberately does NOT.
Arrays are indexed [j, i] (Z-major), flat n = j*nr + i.
"""
import numpy as np
from scipy.linalg import lapack

MU0 = 4.0e-7 * np.pi


class GSOperator:
    """Banded LU (LAPACK dgbtrf, factored once) of the interior 5-point Delta* matrix."""

    def __init__(self, nr, nz, rmin, rmax, zmin, zmax):
        self.nr, self.nz = nr, nz
        self.dr = (rmax - rmin) / (nr - 1)
        self.dz = (zmax - zmin) / (nz - 1)
        self.r = rmin + self.dr * np.arange(nr)
        self.z = zmin + self.dz * np.arange(nz)
        ni, nj = nr - 2, nz - 2
        self.ni, self.nj = ni, nj
        n = ni * nj
        dr, dz = self.dr, self.dz
        ri = self.r[1:-1]
        self.cw = (1.0 + dr / (2.0 * ri)) / dr**2   # multiplies psi[i-1, j]
        self.ce = (1.0 - dr / (2.0 * ri)) / dr**2   # multiplies psi[i+1, j]
        self.cc = -(2.0 / dr**2 + 2.0 / dz**2)
        self.cz = 1.0 / dz**2
        kl = ku = ni
        ab = np.zeros((2 * kl + ku + 1, n))
        # unknown u = (j-1)*ni + (i-1); LAPACK band storage ab[kl+ku+row-col, col]
        u = np.arange(n)
        iu = u % ni
        ab[kl + ku, u] = self.cc
        m = iu > 0        # row u, col u-1: west
        ab[kl + ku + 1, u[m] - 1] = self.cw[iu[m]]
        m = iu < ni - 1   # row u, col u+1: east
        ab[kl + ku - 1, u[m] + 1] = self.ce[iu[m]]
        m = u >= ni       # row u, col u-ni: south
        ab[kl + ku + ni, u[m] - ni] = self.cz
        m = u < n - ni    # row u, col u+ni: north
        ab[kl + ku - ni, u[m] + ni] = self.cz
        self.kl, self.ku = kl, ku
        lu, piv, info = lapack.dgbtrf(ab, kl, ku)
        assert info == 0
        self.lu, self.piv = lu, piv

    def apply(self, psi):
        """Discrete Delta* at the interior nodes of psi[nz, nr] -> [nz-2, nr-2]."""
        p = psi
        return (self.cw[None, :] * p[1:-1, :-2] + self.ce[None, :] * p[1:-1, 2:]
                + self.cc * p[1:-1, 1:-1] + self.cz * (p[:-2, 1:-1] + p[2:, 1:-1]))

    def solve(self, rhs_int, psi_edge):
        """Solve Delta*_h psi = rhs_int at interior nodes with Dirichlet data taken from the
        edge entries of psi_edge[nz, nr].  Returns psi[nz, nr] (edges copied from psi_edge)."""
        f = np.array(rhs_int, dtype=np.float64, copy=True)
        f[:, 0] -= self.cw[0] * psi_edge[1:-1, 0]
        f[:, -1] -= self.ce[-1] * psi_edge[1:-1, -1]
        f[0, :] -= self.cz * psi_edge[0, 1:-1]
        f[-1, :] -= self.cz * psi_edge[-1, 1:-1]
        x, info = lapack.dgbtrs(self.lu, self.kl, self.ku, f.reshape(-1, 1), self.piv)
        assert info == 0
        out = np.array(psi_edge, dtype=np.float64, copy=True)
        out[1:-1, 1:-1] = x.reshape(self.nj, self.ni)
        return out

    def solve_current(self, I_node, psi_bdry_edge):
        """Delta* psi = -mu0 R I/dA (Eq. 1) for node currents I_node[nz, nr] in amperes."""
        rhs = -MU0 * self.r[None, 1:-1] * I_node[1:-1, 1:-1] / (self.dr * self.dz)
        return self.solve(rhs, psi_bdry_edge)


def boundary_nodes(nr, nz):
    """Flat indices of the N_b = 2(nr+nz)-4 edge nodes in the order include/ptefit.h fixes:
    bottom row j=0 (i=0..nr-1), top row j=nz-1, left column i=0 (j=1..nz-2), right column."""
    i = np.arange(nr)
    j = np.arange(1, nz - 1)
    return np.concatenate([i, (nz - 1) * nr + i, j * nr, j * nr + nr - 1])
