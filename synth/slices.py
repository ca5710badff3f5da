"""Seeded per-slice inputs: measurement vectors b and coil currents I_C.

Recipe: an analytic D-shaped current distribution of total I_p
(polynomial in a geometric flux label, the shape BASELINE.json's "Solov'ev-like scale"
describes) plus PF-coil currents chosen by a small regularised least squares so that the
target boundary is an iso-flux contour of plasma + coils (and grad psi = 0 at the target
X-points).  No Grad-Shafranov solve, no search, no basis fit happens here.
"""
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
    return dict(I=I.ravel(), ic=ic, shape=sh, ca=ca * scale, cb=cb * scale, ip=ip,
                design_resid=float(np.max(np.abs(A @ i_pf - y))))


def make_slices(dev, n_slices, first=0, noise=0.005, n_cal=None):
    """b[n_slices, M], ic[n_slices, n_coil] (float64) for slices first..first+n_slices-1 and
    sigma[M]: 0.5 % of the per-group (probes / loops) RMS of the noise-free signals over the
    first n_cal slices (default min(config batch, 16)).  Fills dev['geom']['sigma'] if unset."""
    meta, c, tb = dev["meta"], dev["meta"]["cfg"], dev["tables"]
    npb = meta["n_probe"]
    if dev["geom"]["sigma"] is None:
        n_cal = n_cal or min(c["batch"], 16)
        cal = np.stack([_clean(dev, k) for k in range(n_cal)])
        sig = np.empty(cal.shape[1])
        sig[:npb] = noise * np.sqrt(np.mean(cal[:, :npb] ** 2))
        sig[npb:] = noise * np.sqrt(np.mean(cal[:, npb:] ** 2))
        dev["geom"]["sigma"] = sig
    sig = dev["geom"]["sigma"]
    b = np.empty((n_slices, len(sig)))
    ic = np.empty((n_slices, tb["gc"].shape[1]))
    truth = []
    for q in range(n_slices):
        k = first + q
        t = truth_slice(dev, k)
        rng = np.random.default_rng((20260112 + c["idx"]) * 1000 + k + 500_000_000)
        b[q] = tb["gp"] @ t["I"] + tb["gc"] @ t["ic"] + sig * rng.standard_normal(len(sig))
        ic[q] = t["ic"]
        truth.append(t)
    return dict(b=b, ic=ic, sigma=sig, truth=truth)


def _clean(dev, k):
    t = truth_slice(dev, k)
    return dev["tables"]["gp"] @ t["I"] + dev["tables"]["gc"] @ t["ic"]
