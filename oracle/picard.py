"""The per-slice EFIT Picard iteration ("repeatedly performing Picard iterations
for each time slice"; steps from Sec. II.B-II.D).

Oracle-side (test infrastructure): plain float64, one slice at a time, step by step in the
order DESIGN.md O7 states:  state = O2;  repeat n_iter times { basis (Eq. 10) -> response
R = G_P J_b (Eq. 6) -> fit -> node currents -> boundary flux G_B I -> Delta* solve -> add coil
flux -> search/normalise }.
"""
import numpy as np
from . import basis as _basis, lsq as _lsq, search as _search
from .gs_solve import GSOperator, boundary_nodes


class Device:
    """Frozen per-device data (the arguments of ptefit_create, include/ptefit.h)."""

    def __init__(self, grid, geom, tables, basis):
        self.nr, self.nz = grid["nr"], grid["nz"]
        self.op = GSOperator(self.nr, self.nz, grid["rmin"], grid["rmax"], grid["zmin"], grid["zmax"])
        self.r, self.z = self.op.r, self.op.z
        self.dA = self.op.dr * self.op.dz
        self.sigma = np.asarray(geom["sigma"], np.float64)
        self.lim_r = np.asarray(geom["lim_r"], np.float64)
        self.lim_z = np.asarray(geom["lim_z"], np.float64)
        self.lim_mask = np.asarray(geom["lim_mask"]).astype(bool).reshape(self.nz, self.nr)
        xm = geom.get("xpt_mask")
        self.xpt_mask = self.lim_mask if xm is None else np.asarray(xm).astype(bool).reshape(self.nz, self.nr)
        self.s = int(geom.get("ip_sign", 1))
        self.cold = (geom["cold_rc"], geom["cold_zc"], geom["cold_a"], geom["cold_b"])
        N = self.nr * self.nz
        interior = np.zeros((self.nz, self.nr), bool)
        interior[1:-1, 1:-1] = True
        self.interior = interior.ravel()
        self.gp = np.asarray(tables["gp"], np.float64).reshape(-1, N)
        self.gc = np.asarray(tables["gc"], np.float64)
        self.gb = np.asarray(tables["gb"], np.float64).reshape(-1, N)
        self.ggc = np.asarray(tables["ggc"], np.float64).reshape(N, -1)
        self.bnd = boundary_nodes(self.nr, self.nz)
        self.n_p, self.n_ff = basis["n_p"], basis["n_ff"]
        self.lam = basis.get("lambda_reg", 0.0)
        self.delz = int(basis.get("delz", 0))          # 1 = append the vertical-shift term
        self.relax = float(basis.get("relax", 1.0))     # psi^{k+1} = psi^k + relax (psi_new - psi^k)
        self.spline = basis.get("spline")               # dict(knots, tension, terms) or None (config 5: FF' edge terms)
        self.n_spl = 0 if self.spline is None else len(self.spline["terms"])
        self.nb = self.n_p + self.n_ff + self.n_spl + self.delz
        self.fit_coils = int(basis.get("fit_coils", 0))   # 1 = joint fit of the coil currents, Eq. 7
        self.sigma_ic = None if basis.get("sigma_ic") is None else np.asarray(basis["sigma_ic"], np.float64)


def picard_iteration(dev, psin, mask, d, psi_coil, X_prev=None, psi_prev=None, b=None, ic=None):
    """One Picard iteration from (psin, mask).  Returns dict with X, chi2, status, psi, resp,
    I (node currents), psi_bdry and the search result `srch` of the new psi.
    X_prev: previous coefficients (for the delz column); psi_prev: flux to relax towards/from
    (None = take the new flux as is)."""
    Jb = _basis.basis_columns(psin, mask, dev.r, dev.dA, dev.n_p, dev.n_ff, dev.spline)     # Eq. 10
    Jb = Jb.reshape(-1, Jb.shape[-1]) * dev.interior[:, None]                     # edge nodes carry no current
    if dev.delz:
        nj = dev.n_p + dev.n_ff + dev.n_spl
        xp = np.zeros(nj) if X_prev is None else np.asarray(X_prev)[:nj]
        col = _basis.delz_column(Jb, xp, dev.nz, dev.nr, dev.op.dz) * dev.interior
        Jb = np.concatenate([Jb, col[:, None]], axis=1)
    resp = dev.gp @ Jb                                                            # Eq. 6: R = G_P J_b
    if dev.fit_coils:                                                             # Eq. 7: coil currents fitted too,
        X, icf, chi2, st = _lsq.fit_joint(resp, dev.gc, b, ic, dev.sigma, dev.sigma_ic, dev.lam)
        psi_coil = (dev.ggc @ icf).reshape(dev.nz, dev.nr)                        # and the coil flux follows them
        out = dict(X=X, chi2=chi2, status=st, resp=resp, ic_fit=icf)
    else:
        X, chi2, st = _lsq.fit(resp, d, dev.sigma, dev.lam)
        out = dict(X=X, chi2=chi2, status=st, resp=resp)
    if st != 0:
        return out
    I = Jb @ X                                                                    # J_phi dA = J_b X
    psi_b = dev.gb @ I                                                            # Dirichlet data
    edge = np.zeros(dev.nr * dev.nz)
    edge[dev.bnd] = psi_b
    psi_pl = dev.op.solve_current(I.reshape(dev.nz, dev.nr), edge.reshape(dev.nz, dev.nr))
    psi = psi_pl + psi_coil
    if psi_prev is not None:
        psi = psi_prev + dev.relax * (psi - psi_prev)
    srch = _search.search(psi, dev.r, dev.z, dev.lim_mask, dev.xpt_mask, dev.lim_r, dev.lim_z, dev.s)
    out.update(I=I, psi_bdry=psi_b, psi=psi, srch=srch, status=srch["status"])
    return out


def reconstruct(dev, b, ic, n_iter, psi0=None, trace=False, X0=None, psi_noise=None):
    """ptefit_reconstruct for one slice.  psi0 = None -> cold start (O2), else warm start; X0 = the
    coefficients of the previous call (a warm start keeps them: they seed the vertical-shift column of the
    first iteration, which is what keeps the one-iteration-per-slice mode of PAPER.md:158 from drifting).
    psi_noise = (rel, seed): test hook of the case generator -- Gaussian noise of rel * max|psi| is added to the
    flux after every iteration, to see whether a slice's decisions survive FP32-level perturbations."""
    d = np.asarray(b, np.float64) - dev.gc @ np.asarray(ic, np.float64)           # Eq. 2 / Eq. 6 rhs
    psi_coil = (dev.ggc @ np.asarray(ic, np.float64)).reshape(dev.nz, dev.nr)
    res = dict(status=0, X=np.zeros(dev.nb) if (X0 is None or psi0 is None) else np.array(X0, np.float64), chi2=np.nan, psi=None,
               srch=None, hist=[])
    if psi0 is None:
        psin, mask = _search.cold_start(dev.r, dev.z, dev.lim_mask, *dev.cold)
        psi = np.zeros((dev.nz, dev.nr))
        if not mask.any():
            res["status"] = 1
    else:
        psi = np.array(psi0, np.float64).reshape(dev.nz, dev.nr)
        sr = _search.search(psi, dev.r, dev.z, dev.lim_mask, dev.xpt_mask, dev.lim_r, dev.lim_z, dev.s)
        res["srch"] = sr
        res["status"] = sr["status"]
        psin, mask = sr["psin"], sr["mask"]
    res["psi"] = psi
    for it in range(n_iter):
        if res["status"] != 0:
            break
        have_prev = (psi0 is not None) or it > 0     # cold start: the first flux is taken as is
        o = picard_iteration(dev, psin, mask, d, psi_coil, X_prev=res["X"],
                             psi_prev=res["psi"] if have_prev else None, b=np.asarray(b, np.float64), ic=np.asarray(ic, np.float64))
        if "ic_fit" in o:
            res["ic_fit"] = o["ic_fit"]
        res["X"], res["chi2"], res["status"] = o["X"], o["chi2"], o["status"]
        if "psi" in o and psi_noise is not None and o["status"] == 0:
            rng = np.random.default_rng(psi_noise[1] + 1000 * it)
            o["psi"] = o["psi"] + psi_noise[0] * np.max(np.abs(o["psi"])) * rng.standard_normal(o["psi"].shape)
            o["srch"] = _search.search(o["psi"], dev.r, dev.z, dev.lim_mask, dev.xpt_mask, dev.lim_r, dev.lim_z, dev.s)
            o["status"] = o["srch"]["status"]
        if "psi" in o:
            if trace:
                res["hist"].append(dict(X=o["X"], chi2=o["chi2"], dpsi=float(np.max(np.abs(o["psi"] - res["psi"]))),
                                        psi=o["psi"], resp=o["resp"], I=o["I"], psi_bdry=o["psi_bdry"], srch=o["srch"],
                                        ic_fit=o.get("ic_fit")))
            res["psi"], res["srch"] = o["psi"], o["srch"]
            psin, mask = o["srch"]["psin"], o["srch"]["mask"]
    return res
