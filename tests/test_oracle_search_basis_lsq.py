"""Pins for oracle/search.py, basis.py, lsq.py."""
import numpy as np

from oracle import basis as B, lsq as L, search as S
from oracle.gs_solve import MU0


def test_fit_weights_are_the_integer_table():
    """PAPER.md:128 'preconstructing normal equations and inverting': the pseudo-inverse has the
    closed-form integer weights."""
    P = S.fit_design_pinv()
    st = lambda f: np.array([[f(x, y) for x in (-1, 0, 1)] for y in (-1, 0, 1)], float).ravel()
    assert np.allclose(P[0], st(lambda x, y: (5 if (x, y) == (0, 0) else 2 if x * y == 0 else -1)) / 9)
    assert np.allclose(P[1], st(lambda x, y: x) / 6)
    assert np.allclose(P[2], st(lambda x, y: y) / 6)
    assert np.allclose(P[3], st(lambda x, y: (1 if x else -2)) / 6)
    assert np.allclose(P[4], st(lambda x, y: x * y) / 4)
    assert np.allclose(P[5], st(lambda x, y: (1 if y else -2)) / 6)


def _quad_field(nr, nz, c, i0, j0):
    i, j = np.meshgrid(np.arange(nr), np.arange(nz))
    x, y = i - i0, j - j0
    return c[0] + c[1] * x + c[2] * y + c[3] * x * x + c[4] * x * y + c[5] * y * y


def test_exact_recovery_of_quadratics_and_classification():
    # maximum at (6.3, 5.2): O-point, det > 0 ; saddle at same place: det < 0
    for c, kind in (((2.0, 0, 0, -0.3, 0.1, -0.2), "O"), ((1.0, 0, 0, -0.3, 0.05, 0.25), "X")):
        psi = _quad_field(12, 11, c, 6.3, 5.2)
        f = S.quad_fit(psi)
        jj, ii = 5 - 1, 6 - 1
        assert abs(f["xs"][jj, ii] - 0.3) < 1e-12 and abs(f["ys"][jj, ii] - 0.2) < 1e-12
        assert abs(f["ps"][jj, ii] - c[0]) < 1e-12
        assert (f["det"][jj, ii] > 0) == (kind == "O")
        assert np.allclose(f["cxx"], c[3]) and np.allclose(f["cxy"], c[4]) and np.allclose(f["cyy"], c[5])


def _setup(n=33):
    r = np.linspace(0.15, 1.6, n)
    z = np.linspace(-1.5, 1.5, n)
    R, Z = np.meshgrid(r, z)
    th = 2 * np.pi * np.arange(64) / 64
    lr, lz = 0.8 + 0.55 * np.cos(th), 1.1 * np.sin(th)
    lim = ((R - 0.8) / 0.55) ** 2 + (Z / 1.1) ** 2 < 0.97
    return r, z, R, Z, lr, lz, lim


def test_limited_plasma_and_brute_force():
    r, z, R, Z, lr, lz, lim = _setup()
    psi = 1.0 - ((R - 0.83) / 0.5) ** 2 - ((Z - 0.04) / 0.9) ** 2
    o = S.search(psi, r, z, lim, lim, lr, lz, 1)
    assert o["status"] == 0 and o["limited"] == 1 and o["n_cand"] == 0
    assert abs(o["axis"][2] - 0.83) < 1e-12 and abs(o["axis"][3] - 0.04) < 1e-12 and abs(o["axis"][4] - 1.0) < 1e-12
    # brute force: boundary flux = max over limiter vertices of bilinear psi
    pv = [S.bilinear(psi, r, z, a, b) for a, b in zip(lr, lz)]
    assert o["psi_b"] == max(pv)
    m = o["mask"]
    assert np.all(lim[m]) and np.all(psi[m] > o["psi_b"]) and np.all(~m[lim & (psi <= o["psi_b"])])
    assert np.all((o["psin"][m] >= 0) & (o["psin"][m] <= 1)) and np.all(o["psin"][~m] == 0)
    x = (psi - 1.0) / (o["psi_b"] - 1.0)
    assert np.allclose(o["psin"][m], np.clip(x[m], 0, 1), atol=1e-14)


def test_xpoint_found_and_mirror_symmetry():
    r, z, R, Z, lr, lz, lim = _setup(65)
    # flux with a maximum near (0.8, 0.05) and a saddle below: cubic in Z
    zc, zx = 0.05, -0.8
    g = lambda Zv: -(Zv - zc) ** 2 * (Zv - (1.5 * zx - 0.5 * zc)) / (zc - (1.5 * zx - 0.5 * zc))   # g'(zc)=g'(zx)=0
    psi = 1.0 - ((R - 0.8) / 0.45) ** 2 + g(Z) / 0.9**2
    o = S.search(psi, r, z, lim, lim, lr, lz, 1)
    assert o["status"] == 0 and o["limited"] == 0
    assert abs(o["xpt"][2] - 0.8) < 2e-3 and abs(o["xpt"][3] - zx) < 2e-3
    assert abs(o["axis"][3] - zc) < 2e-3
    assert not o["mask"][Z < zx - 0.05].any()          # nothing behind the X-point
    # mirror image in Z gives the mirror image result
    o2 = S.search(psi[::-1].copy(), r, z, lim[::-1].copy(), lim[::-1].copy(), lr, -lz, 1)
    assert o2["limited"] == 0 and abs(o2["xpt"][3] + o["xpt"][3]) < 1e-12 and abs(o2["psi_b"] - o["psi_b"]) < 1e-13
    assert np.array_equal(o2["mask"], o["mask"][::-1])
    # negative plasma current: the search of -psi with s=-1 is identical
    o3 = S.search(-psi, r, z, lim, lim, lr, lz, -1)
    assert np.array_equal(o3["mask"], o["mask"]) and abs(o3["psi_b"] + o["psi_b"]) < 1e-15


def test_status_codes():
    r, z, R, Z, lr, lz, lim = _setup()
    assert S.search(R * 0 + np.nan, r, z, lim, lim, lr, lz, 1)["status"] == 2
    assert S.search(R + 0.0, r, z, lim, lim, lr, lz, 1)["status"] == 1     # no extremum inside


def test_basis_columns_closed_form():
    """Eq. 10 at hand-computable points: x=0 -> (R, 0, mu0/R, 0); x=1 -> 0."""
    r = np.array([0.5, 1.0, 2.0])
    psin = np.array([[0.0, 0.5, 1.0]])
    mask = np.array([[True, True, True]])
    Jb = B.basis_columns(psin, mask, r, 0.01, 2, 2)
    assert np.allclose(Jb[0, 0], [0.5 * 0.01, 0, MU0 / 0.5 * 0.01, 0])
    assert np.allclose(Jb[0, 1], [1.0 * (1 - 0.25) * 0.01, 1.0 * (0.5 - 0.25) * 0.01, MU0 * 0.75 * 0.01, MU0 * 0.25 * 0.01])
    assert np.all(Jb[0, 2] == 0)
    assert np.all(B.basis_columns(psin, ~mask, r, 0.01, 3, 1) == 0)
    J3 = B.basis_columns(psin, mask, r, 1.0, 3, 1)
    assert np.allclose(J3[0, 1], [1 - 0.125, 0.5 - 0.125, 0.25 - 0.125, MU0 * 0.5])


def test_delz_column_is_minus_dIdZ():
    nz, nr, dz = 7, 3, 0.1
    z = np.arange(nz) * dz
    Jb = np.zeros((nz * nr, 2))
    Jb[:, 0] = np.repeat(z**2, nr)
    col = B.delz_column(Jb, np.array([2.0, 5.0]), nz, nr, dz).reshape(nz, nr)
    assert np.allclose(col[1:-1], -(4.0 * z[1:-1])[:, None]) and np.all(col[[0, -1]] == 0)


def test_lsq_normal_equations_and_recovery():
    rng = np.random.default_rng(4)
    M, nb = 60, 4
    A = rng.normal(size=(M, nb)) * np.array([1.0, 10.0, 1e6, 1e7])
    sig = rng.uniform(0.5, 2.0, M)
    xt = np.array([1.0, -0.2, 3e-6, 1e-7])
    X, chi2, st = L.fit(A, A @ xt, sig, 0.0)          # exact data, lambda = 0 -> truth (Eq. 6)
    assert st == 0 and np.allclose(X, xt, rtol=1e-9) and chi2 < 1e-18
    d = A @ xt + sig * rng.normal(size=M)
    lam = 0.05
    X, chi2, st = L.fit(A, d, sig, lam)
    W = A / sig[:, None]
    s = np.sqrt((W * W).sum(0))
    # stationarity: (WA)^T (WA X - W d) + lam^2 M S^2 X = 0
    g = W.T @ (W @ X - d / sig) + lam**2 * M * s**2 * X
    assert np.max(np.abs(g) / (s * np.linalg.norm(d / sig))) < 1e-12
    Xn = np.linalg.solve(W.T @ W + lam**2 * M * np.diag(s**2), W.T @ (d / sig))
    assert np.allclose(X, Xn, rtol=1e-9)
    assert abs(chi2 - np.sum(((A @ X - d) / sig) ** 2)) < 1e-9 * chi2
    # a zero column is dropped, a duplicated column is rank deficient
    A0 = A.copy(); A0[:, 1] = 0
    X0, _, st0 = L.fit(A0, d, sig, 0.0)
    assert st0 == 0 and X0[1] == 0
    A1 = A.copy(); A1[:, 1] = A1[:, 0]
    assert L.fit(A1, d, sig, 0.0)[2] == 3
