"""Synthetic device: grid, limiter, sensors, coils, eddy filaments, Green's tables.

Shapes follow BASELINE.json's five configs (grid extents, channel counts, coil counts); the
geometry itself is invented and seeded (the EXL-50U geometry is not public in the paper).
"""
import numpy as np
from scipy.special import ellipk, ellipe

MU0 = 4.0e-7 * np.pi

# name -> config (BASELINE.json configs[0..4])
CONFIGS = {
    "cfg1": dict(idx=1, lam=0.003, n=33, zmax=1.5, n_probe=40, n_loop=20, n_pf=8, n_eddy=0, n_p=2, n_ff=2,
                 batch=1, n_iter=10, precision="fp64", ic_range=20e3, shapes=("limited",)),
    "cfg2": dict(idx=2, lam=0.003, n=65, zmax=1.5, n_probe=76, n_loop=34, n_pf=12, n_eddy=0, n_p=3, n_ff=3,
                 batch=1, n_iter=15, precision="fp32", ic_range=20e3, shapes=("limited",)),
    "cfg3": dict(idx=3, n=129, zmax=1.6, n_probe=100, n_loop=40, n_pf=16, n_eddy=0, n_p=3, n_ff=3,
                 batch=1, n_iter=20, precision="fp32", ic_range=30e3, shapes=("lsn",)),
    "cfg4": dict(idx=4, n=129, zmax=1.6, n_probe=100, n_loop=40, n_pf=16, n_eddy=60, n_p=3, n_ff=3,
                 batch=512, n_iter=20, precision="fp32", ic_range=30e3,
                 shapes=("limited", "limited", "lsn", "usn", "dn")),   # 40/20/20/20 %
    "cfg5": dict(idx=5, n=257, zmax=1.6, n_probe=100, n_loop=40, n_pf=16, n_eddy=60, n_p=4, n_ff=4, spline=True,
                 batch=64, n_iter=30, precision="fp64", ic_range=30e3,
                 shapes=("limited", "limited", "lsn", "usn", "dn")),
}
RMIN, RMAX = 0.15, 1.60
LAMBDA_REG = 0.005
RELAX = 0.6


def filament_psi(a, zs, rho, zf):
    """Flux per radian at (rho, zf) per ampere in a filament (a, zs); scipy elliptic integrals."""
    z = zf - zs
    k2 = 4.0 * a * rho / ((a + rho) ** 2 + z * z)
    K, E = ellipk(k2), ellipe(k2)
    return MU0 / (2 * np.pi) * np.sqrt(a * rho) * ((2 - k2) * K - 2 * E) / np.sqrt(k2)


def filament_b(a, zs, rho, zf):
    """(B_R, B_Z) at (rho, zf) per ampere in a filament (a, zs)."""
    z = zf - zs
    s2 = (a + rho) ** 2 + z * z
    d2 = (a - rho) ** 2 + z * z
    k2 = 4.0 * a * rho / s2
    K, E = ellipk(k2), ellipe(k2)
    pref = MU0 / (2 * np.pi) / np.sqrt(s2)
    return (pref * z / rho * (-K + (a * a + rho * rho + z * z) / d2 * E),
            pref * (K + (a * a - rho * rho - z * z) / d2 * E))


def _inside_polygon(px, py, vx, vy):
    """Even-odd rule, vectorised over points."""
    inside = np.zeros(px.shape, bool)
    n = len(vx)
    for k in range(n):
        x0, y0, x1, y1 = vx[k], vy[k], vx[(k + 1) % n], vy[(k + 1) % n]
        cross = ((y0 > py) != (y1 > py))
        with np.errstate(divide="ignore", invalid="ignore"):
            xi = x0 + (py - y0) * (x1 - x0) / (y1 - y0)
        inside ^= cross & (px < xi)
    return inside


def _perimeter_point(t, zmax, margin):
    """Point at parameter t in [0,1) on the rectangle offset outward from the grid by margin,
    starting at the inboard mid-plane and running over the top to the outboard mid-plane for
    t in [0, 0.5) (the mirror half is produced by the caller)."""
    r0, r1, z1 = RMIN - margin, RMAX + margin, zmax + margin
    L = z1 + (r1 - r0) + z1
    s = 2.0 * t * L
    if s < z1:
        return r0, s
    if s < z1 + (r1 - r0):
        return r0 + (s - z1), z1
    return r1, z1 - (s - z1 - (r1 - r0))


def make_device(name, with_tables=True):
    """Returns dict(grid, geom, tables, basis, meta) -- the ptefit_create arguments as numpy
    float64 arrays plus meta (sensor/coil positions) used by make_slices."""
    c = CONFIGS[name]
    rng = np.random.default_rng(20260112 + c["idx"])
    n, zmax = c["n"], c["zmax"]
    grid = dict(nr=n, nz=n, rmin=RMIN, rmax=RMAX, zmin=-zmax, zmax=zmax)
    r = np.linspace(RMIN, RMAX, n)
    z = np.linspace(-zmax, zmax, n)
    dr, dz = r[1] - r[0], z[1] - z[0]
    R2, Z2 = np.meshgrid(r, z)
    # limiter: 64-vertex ellipse
    th = 2 * np.pi * np.arange(64) / 64
    lim_r = 0.80 + 0.55 * np.cos(th)
    lim_z = 0.77 * zmax * np.sin(th)
    lim_mask = _inside_polygon(R2, Z2, lim_r, lim_z)
    lim_mask[0, :] = lim_mask[-1, :] = False
    lim_mask[:, 0] = lim_mask[:, -1] = False
    # sensors on an ellipse enclosing the grid (tall so that R > 0): probes then loops
    M = c["n_probe"] + c["n_loop"]
    ang = np.sort(rng.uniform(0, 2 * np.pi, M))
    rng.shuffle(ang)
    sz_ax = 2.8 if zmax == 1.5 else 3.0
    sen_r = 0.875 + 0.86 * np.cos(ang)
    sen_z = sz_ax * np.sin(ang)
    alpha = rng.uniform(0, 2 * np.pi, c["n_probe"])
    # PF coils: near up-down pairs outside the grid rectangle, seeded turn counts
    npair = c["n_pf"] // 2
    tpar = (np.arange(npair) + 0.5 + rng.uniform(-0.2, 0.2, npair)) / npair * 0.5
    pf_r, pf_z = [], []
    for t in tpar:
        pr, pz = _perimeter_point(t, zmax, 0.10)
        pr = max(pr, 0.06)
        for sgn in (+1, -1):
            pf_r.append(pr + rng.uniform(-0.02, 0.02) * (pr > 0.1))
            pf_z.append(sgn * pz + rng.uniform(-0.02, 0.02))
    pf_r, pf_z = np.array(pf_r), np.array(pf_z)
    turns = rng.integers(8, 33, c["n_pf"]).astype(float)
    # eddy filaments between limiter and grid edge, nudged away from nodes
    ne = c["n_eddy"]
    te = 2 * np.pi * (np.arange(ne) + 0.5) / max(ne, 1)
    ed_r = 0.86 + 0.66 * np.cos(te)
    ed_z = 0.90 * zmax * np.sin(te)
    for k in range(ne):
        fi, fj = (ed_r[k] - RMIN) / dr, (ed_z[k] + zmax) / dz
        if abs(fi - round(fi)) < 0.25:
            ed_r[k] = RMIN + (round(fi) + 0.3) * dr
        if abs(fj - round(fj)) < 0.25:
            ed_z[k] = -zmax + (round(fj) + 0.3) * dz
    src_r = np.concatenate([pf_r, ed_r])
    src_z = np.concatenate([pf_z, ed_z])
    src_w = np.concatenate([turns, np.ones(ne)])
    geom = dict(n_meas=M, n_coil=c["n_pf"] + ne, sigma=None, lim_r=lim_r, lim_z=lim_z,
                lim_mask=lim_mask.astype(np.uint8), xpt_mask=None, ip_sign=1,
                cold_rc=0.80, cold_zc=0.0, cold_a=0.40, cold_b=0.72)
    meta = dict(cfg=c, name=name, r=r, z=z, sen_r=sen_r, sen_z=sen_z, alpha=alpha, n_probe=c["n_probe"],
                src_r=src_r, src_z=src_z, src_w=src_w, n_pf=c["n_pf"])
    basis = dict(n_p=c["n_p"], n_ff=c["n_ff"], lambda_reg=c.get("lam", LAMBDA_REG), delz=1, relax=RELAX)
    if c.get("spline"):
        # BASELINE.json configs[4]: "plus 5-knot tension-spline FF' edge terms" (7 knots
        # 0.70 .. 1.00, tension 10, the five interior cardinal functions)
        basis["spline"] = dict(knots=np.linspace(0.70, 1.00, 7), tension=10.0, terms=[1, 2, 3, 4, 5])
    out = dict(grid=grid, geom=geom, basis=basis, meta=meta, tables=None)
    if with_tables:
        out["tables"] = make_tables(meta, grid)
    return out


def sensor_response(meta, a, zs):
    """[M, len(a)] per-ampere response of every channel to filaments (a, zs)."""
    npb = meta["n_probe"]
    a = np.asarray(a)[None, :]
    zs = np.asarray(zs)[None, :]
    br, bz = filament_b(a, zs, meta["sen_r"][:npb, None], meta["sen_z"][:npb, None])
    al = meta["alpha"][:, None]
    probes = np.cos(al) * br + np.sin(al) * bz
    loops = filament_psi(a, zs, meta["sen_r"][npb:, None], meta["sen_z"][npb:, None])
    return np.concatenate([probes, loops], axis=0)


def make_tables(meta, grid):
    nr, nz = grid["nr"], grid["nz"]
    r, z = meta["r"], meta["z"]
    R2, Z2 = np.meshgrid(r, z)
    rn, zn = R2.ravel(), Z2.ravel()
    interior = np.zeros((nz, nr), bool)
    interior[1:-1, 1:-1] = True
    interior = interior.ravel()
    gp = sensor_response(meta, rn, zn) * interior[None, :]
    gc = sensor_response(meta, meta["src_r"], meta["src_z"]) * meta["src_w"][None, :]
    i = np.arange(nr)
    j = np.arange(1, nz - 1)
    bnd = np.concatenate([i, (nz - 1) * nr + i, j * nr, j * nr + nr - 1])
    gb = np.zeros((len(bnd), nr * nz))
    cols = np.nonzero(interior)[0]
    for k0 in range(0, len(bnd), 64):     # chunked to bound temporaries
        kk = bnd[k0:k0 + 64]
        gb[k0:k0 + 64, cols] = filament_psi(rn[None, cols], zn[None, cols], rn[kk, None], zn[kk, None])
    ggc = filament_psi(meta["src_r"][None, :], meta["src_z"][None, :], rn[:, None], zn[:, None]) * meta["src_w"][None, :]
    return dict(gp=gp, gc=gc, gb=gb, ggc=ggc)
