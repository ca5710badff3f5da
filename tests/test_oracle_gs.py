"""Pins for oracle/gs_solve.py (Eq. 1; Sec. II.C)."""
import os

import numpy as np

from oracle.gs_solve import GSOperator, boundary_nodes, MU0

HERE = os.path.dirname(__file__)


def solovev(R, Z, c=1.0, E=1.8, R0=0.8):
    return -c * (R**2 * Z**2 / E**2 + (R**2 - R0**2) ** 2 / 4) + 0.3 * (R**2 * np.log(R) - Z**2) + 0.1 * Z * R**2


def test_solovev_convergence_matches_golden():
    errs = {}
    for line in open(os.path.join(HERE, "golden", "solovev_errors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, e = line.split()
        errs[int(n)] = float(e)
    got = {}
    for n, e in errs.items():
        op = GSOperator(n, n, 0.15, 1.6, -1.5, 1.5)
        R, Z = np.meshgrid(op.r, op.z)
        pa = solovev(R, Z)
        p = op.solve(-(2 / 1.8**2 + 2) * R[1:-1, 1:-1] ** 2, pa)
        got[n] = np.max(np.abs(p - pa)) / np.max(np.abs(pa))
        assert abs(got[n] / e - 1) < 0.01, (n, got[n], e)
    assert 3.9 < got[33] / got[65] < 4.1    # second order


def test_quadratic_in_z_is_exact_and_sign_of_dR_term():
    """psi = R^2 gives Delta* psi = 2 - 2 = 0; psi = R^4 gives 12R^2 - 4R^2 = 8R^2; the centred
    stencil is exact for polynomials up to degree 2 in R for d2/dR2 and the (1/R)d/dR term;
    psi = Z^2 gives 2.  A flipped sign on the (1/R) d/dR term fails the first identity."""
    op = GSOperator(17, 13, 0.3, 1.4, -0.7, 0.9)
    R, Z = np.meshgrid(op.r, op.z)
    assert np.max(np.abs(op.apply(R**2))) < 1e-11
    assert np.max(np.abs(op.apply(Z**2) - 2.0)) < 1e-11
    assert np.max(np.abs(op.apply(R**2 * Z + 3.0))) < 1e-11


def test_dense_solve_9x9_and_residual():
    rng = np.random.default_rng(0)
    op = GSOperator(9, 9, 0.15, 1.6, -1.5, 1.5)
    I = rng.normal(size=(9, 9))
    edge = rng.normal(size=(9, 9))
    p = op.solve_current(I, edge)
    # dense matrix built independently, node by node
    idx = -np.ones((9, 9), int)
    idx[1:-1, 1:-1] = np.arange(49).reshape(7, 7)
    A = np.zeros((49, 49))
    f = np.zeros(49)
    dr, dz = op.dr, op.dz
    for j in range(1, 8):
        for i in range(1, 8):
            u = idx[j, i]
            Ri = op.r[i]
            f[u] = -MU0 * Ri * I[j, i] / (dr * dz)
            for (jj, ii, cf) in ((j, i - 1, (1 + dr / (2 * Ri)) / dr**2), (j, i + 1, (1 - dr / (2 * Ri)) / dr**2),
                                 (j - 1, i, 1 / dz**2), (j + 1, i, 1 / dz**2), (j, i, -2 / dr**2 - 2 / dz**2)):
                if idx[jj, ii] >= 0:
                    A[u, idx[jj, ii]] += cf
                else:
                    f[u] -= cf * edge[jj, ii]
    x = np.linalg.solve(A, f)
    assert np.max(np.abs(p[1:-1, 1:-1].ravel() - x)) < 1e-12 * np.max(np.abs(x))
    rhs = -MU0 * op.r[None, 1:-1] * I[1:-1, 1:-1] / (dr * dz)
    assert np.max(np.abs(op.apply(p) - rhs)) < 1e-12 * abs(op.cc) * np.max(np.abs(p))
    assert np.array_equal(p[0], edge[0]) and np.array_equal(p[:, -1], edge[:, -1])


def test_filament_flux_matches_greens_function():
    """A single node current with Green's-function Dirichlet data reproduces the free-space
    filament flux away from the source (O(h^2) + log-singularity smoothing)."""
    from oracle.greens import psi_filament
    n = 65
    op = GSOperator(n, n, 0.15, 1.6, -1.5, 1.5)
    R, Z = np.meshgrid(op.r, op.z)
    I = np.zeros((n, n))
    I[30, 28] = 1e5
    exact = 1e5 * psi_filament(op.r[28], op.z[30], R, Z + 0.0)
    exact[30, 28] = 0
    p = op.solve_current(I, exact)
    far = np.hypot(R - op.r[28], Z - op.z[30]) > 0.3
    assert np.max(np.abs(p - exact)[far]) / np.max(np.abs(exact[far])) < 2e-3
    assert p[30, 28] > 0     # COCOS 7: positive current -> flux maximum


def test_boundary_order():
    b = boundary_nodes(5, 4)
    assert list(b) == [0, 1, 2, 3, 4, 15, 16, 17, 18, 19, 5, 10, 9, 14]
