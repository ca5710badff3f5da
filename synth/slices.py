"""Seeded per-slice inputs: measurement vectors b and coil currents I_C.

`make_slices` loads the case files synth/cases/<cfg>.npz that the oracle-side script
oracle/design_cases.py wrote (converged Grad-Shafranov equilibria of the fitted current form,
DESIGN.md "Input recipe").  `truth_slice` is the seeded draw that script starts from: an analytic
D-shaped current distribution of total I_p (polynomial in a geometric flux label) plus PF-coil
currents from a small regularised least squares making the target boundary an iso-flux contour.
No Grad-Shafranov solve, no search, no basis fit happens in this module.
"""
import functools
import os

import numpy as np
from .device import CONFIGS, MU0, filament_psi, filament_b, sensor_response

IP0 = 3.0e5


def _shape(rng, kind):
    """Seeded D-shape.  'limited' shapes lean on the inboard limiter (R = 0.25 m); the null
    kinds are taller and shifted towards the null that should be active (the nulls themselves
    are the natural ones of plasma + coils; the generator does not force them)."""
    a = rng.uniform(0.35, 0.45)
    dlt = rng.uniform(0.0, 0.4)
    if kind == "limited":
        R0 = 0.25 + a + rng.uniform(0.0, 0.01)
        kap = min(rng.uniform(1.6, 2.2), 0.80 / a)
        Z0 = rng.uniform(-0.03, 0.03)
    else:
        R0 = rng.uniform(0.75, 0.85)
        kap = min(rng.uniform(0.86, 0.94) / a, 2.1)
        off = rng.uniform(0.04, 0.08)
        Z0 = {"lsn": -off, "usn": off, "dn": rng.choice([-1.0, 1.0]) * rng.uniform(0.002, 0.006)}[kind]
    return dict(kind=kind, R0=R0, a=a, kap=kap, dlt=dlt, Z0=Z0)


def _label(sh, R, Z):
    u = (Z - sh["Z0"]) / (sh["kap"] * sh["a"])
    return ((R - sh["R0"] + sh["dlt"] * sh["a"] * u * u) / sh["a"]) ** 2 + u * u


def truth_slice(dev, k):
    """Noise-free slice k: returns dict(I[N], ic[n_coil], shape, coeffs)."""
    meta, c = dev["meta"], dev["meta"]["cfg"]
    rng = np.random.default_rng((20260112 + c["idx"]) * 1000 + k)
    kind = c["shapes"][k % len(c["shapes"])]
    sh = _shape(rng, kind)
    r, z = meta["r"], meta["z"]
    dA = (r[1] - r[0]) * (z[1] - z[0])
    R2, Z2 = np.meshgrid(r, z)
    x = _label(sh, R2, Z2)
    inside = (x < 1.0) & dev["geom"]["lim_mask"].astype(bool)
    area = np.pi * sh["a"] ** 2 * sh["kap"]
    ip = IP0 * rng.uniform(0.8, 1.2)
    n_p, n_ff = c["n_p"], c["n_ff"]
    ca = rng.uniform(0.5, 1.5, n_p) * ip / (sh["R0"] * area)
    cb = rng.uniform(0.5, 1.5, n_ff) * ip * sh["R0"] / (MU0 * area)
    J = np.zeros_like(x)
    for i in range(n_p):
        J += ca[i] * R2 * (x ** i - x ** n_p)
    for j in range(n_ff):
        J += cb[j] * MU0 / R2 * (x ** j - x ** n_ff)
    I = np.where(inside, J, 0.0) * dA
    scale = ip / I.sum()
    I *= scale
    # control points on the target boundary
    nctl = 12
    th = 2 * np.pi * (np.arange(nctl) + rng.uniform(0, 1)) / nctl
    cr = sh["R0"] - sh["dlt"] * sh["a"] * np.sin(th) ** 2 + sh["a"] * np.cos(th)
    cz = sh["Z0"] + sh["kap"] * sh["a"] * np.sin(th)
    nz_idx = np.nonzero(I.ravel())[0]
    pr, pz, pI = R2.ravel()[nz_idx], Z2.ravel()[nz_idx], I.ravel()[nz_idx]
    npf = meta["n_pf"]
    sr, sz, sw = meta["src_r"], meta["src_z"], meta["src_w"]
    ne = len(sr) - npf
    i_eddy = rng.uniform(-2e3, 2e3, ne)

    def flux_fixed(qr, qz):    # plasma + eddy flux at points
        f = filament_psi(pr[None, :], pz[None, :], qr[:, None], qz[:, None]) @ pI
        if ne:
            f = f + filament_psi(sr[None, npf:], sz[None, npf:], qr[:, None], qz[:, None]) @ i_eddy
        return f

    def flux_pf(qr, qz):       # [npts, npf] per per-turn ampere
        return filament_psi(sr[None, :npf], sz[None, :npf], qr[:, None], qz[:, None]) * sw[None, :npf]

    f0, A0 = flux_fixed(cr, cz), flux_pf(cr, cz)
    rows = [A0[1:] - A0[:1]]
    rhs = [-(f0[1:] - f0[0])]
    fs = np.max(np.abs(f0)) * 0.1
    A = np.concatenate(rows, axis=0) / fs
    y = np.concatenate(rhs) / fs
    rng_ic = c["ic_range"]
    draw = rng.uniform(-rng_ic, rng_ic, npf) * 0.1
    gam = 0.3
    Areg = np.concatenate([A * rng_ic, gam * np.eye(npf)], axis=0)     # unknown u = I/range
    yreg = np.concatenate([y, gam * draw / rng_ic])
    u = np.linalg.lstsq(Areg, yreg, rcond=None)[0]
    i_pf = u * rng_ic
    ic = np.concatenate([i_pf, i_eddy])
    return dict(I=I.ravel(), ic=ic, shape=sh, ca=ca * scale, cb=cb * scale, ip=ip, ctl_r=cr, ctl_z=cz, i_eddy=i_eddy,
                draw=draw, label=x, design_resid=float(np.max(np.abs(A @ i_pf - y))))


CASE_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cases")


@functools.lru_cache(maxsize=8)
def _case_file(name):
    path = os.path.join(CASE_DIR, name + ".npz")
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} is missing: run `python -m oracle.design_cases {name}` (the case files are written "
                                "by the oracle-side design-Picard script; synth only loads them)")
    with np.load(path) as f:
        return {k: f[k] for k in f.files}


def make_slices(dev, n_slices, first=0):
    """b[n_slices, M], ic[n_slices, n_coil] (float64) for slices first..first+n_slices-1 of the config's
    case file synth/cases/<cfg>.npz (indices wrap around the stored count) and sigma[M].  The file holds
    converged Grad-Shafranov equilibria of the fitted current form + 0.5 % Gaussian noise, written by
    oracle/design_cases.py.  Fills dev['geom']['sigma'] if unset.  `truth` carries what the generator
    recorded per slice (coefficients, I_p, kind, designed axis / X-point)."""
    cf = _case_file(dev["meta"]["name"])
    n_store = cf["b"].shape[0]
    idx = (first + np.arange(n_slices)) % n_store
    if dev["geom"]["sigma"] is None:
        dev["geom"]["sigma"] = cf["sigma"].copy()
    truth = [dict(X=cf["X_true"][q], ip=float(cf["ip"][q]), kind=str(cf["kind"][q]), axis=cf["axis"][q], xpt=cf["xpt"][q],
                  limited=int(cf["limited"][q]), seed=int(cf["seed"][q])) for q in idx]
    return dict(b=cf["b"][idx].copy(), ic=cf["ic"][idx].copy(), sigma=cf["sigma"].copy(), truth=truth)
