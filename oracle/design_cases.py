"""Writes the seeded case files synth/cases/<cfg>.npz ("design Picard", SURVEY.md 8(d) "Synthetic inputs").

Oracle-side script (test infrastructure): it calls only ``oracle/`` (Grad-Shafranov solve, basis,
search) and ``synth/`` (device layout, Green's tables, seeded shape draws); ``synth.make_slices``
only loads what this script wrote.  Run:  python -m oracle.design_cases [cfg ...] [--jobs J]

For every slice a free-boundary Grad-Shafranov equilibrium is computed whose current density is
EXACTLY of the fitted form J_b(psi_N) X_true (Eq. 10) on the oracle's own 5-point
discretisation:
  repeat { I = J_b(psi_N) X_true rescaled to I_p  ->  psi_pl by oracle.gs_solve with psi_bdry = G_B I
           ->  PF currents by regularised least squares: the seeded control points of the target LCFS
               (and the target X-point, where grad psi = 0 is also asked for) at equal flux,
               regularised toward a seeded draw in the config's current range
           ->  psi = psi_pl + G_GC I_C  ->  oracle.search (axis, X-point, LCFS, psi_N) }
until the flux stops changing.  Measurements b = G_P I + G_C I_C of the converged state + Gaussian
noise, sigma = 0.5 % of the RMS of the channel group (probes / loops) over the batch.
A seed is accepted when the oracle's own reconstruction from the cold start ends with status 0, has the
labelled boundary type, contracts, and (FP32 configs) is well posed: rounding all inputs to FP32 moves the
coefficients by at most 3e-6; otherwise the next seed is tried (rejections are recorded in the file).
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth                                                    # noqa: E402
from synth.slices import truth_slice                            # noqa: E402
from synth.device import filament_psi, filament_b               # noqa: E402
from oracle import basis as OB, search as OS                    # noqa: E402
from oracle.picard import Device, reconstruct                   # noqa: E402

N_STORE = {"cfg1": 8, "cfg2": 8, "cfg3": 8, "cfg4": 512, "cfg5": 64}
CASE_DIR = os.path.join(ROOT, "synth", "cases")


def _targets(sh, rng):
    """Control points of the target LCFS (12, away from the active null) and X-point targets
    [(R, Z, active)] for the null shapes (the analytic D-shape's top / bottom, pushed out 4 %)."""
    kind = sh["kind"]
    th = 2 * np.pi * (np.arange(12) + rng.uniform(0, 1)) / 12
    xs = []
    bot = (sh["R0"] - sh["dlt"] * sh["a"], sh["Z0"] - 1.04 * sh["kap"] * sh["a"])
    top = (sh["R0"] - sh["dlt"] * sh["a"], sh["Z0"] + 1.04 * sh["kap"] * sh["a"])
    if kind == "lsn":
        xs = [(bot[0], bot[1], True)]
    elif kind == "usn":
        xs = [(top[0], top[1], True)]
    elif kind == "dn":
        low = sh["Z0"] < 0
        xs = [(bot[0], bot[1], low), (top[0], top[1], not low)]
    keep = np.ones(12, bool)
    for (_, zx, _) in xs:                           # no smooth-boundary control points next to a null
        tx = -np.pi / 2 if zx < sh["Z0"] else np.pi / 2
        d = np.abs(np.angle(np.exp(1j * (th - tx))))
        keep &= d > 0.55
    th = th[keep]
    cr = sh["R0"] - sh["dlt"] * sh["a"] * np.sin(th) ** 2 + sh["a"] * np.cos(th)
    cz = sh["Z0"] + sh["kap"] * sh["a"] * np.sin(th)
    return cr, cz, xs


def design_slice(dev, od, k, max_iter=300, tol=2e-12):
    """Converged design equilibrium of seed k, or None.  Returns dict(I, ic, X, kind, iters, ...)."""
    meta, c = dev["meta"], dev["meta"]["cfg"]
    t = truth_slice(dev, k)
    sh = t["shape"]
    rng = np.random.default_rng((20260112 + c["idx"]) * 1000 + k + 900_000_000)
    cr, cz, xts = _targets(sh, rng)
    r, z = od.r, od.z
    dr, dz = od.op.dr, od.op.dz
    npf = meta["n_pf"]
    sr_, sz_, sw = meta["src_r"], meta["src_z"], meta["src_w"]
    i_eddy = t["i_eddy"]
    X = np.concatenate([t["ca"], t["cb"]])
    ip = t["ip"]
    # iso-flux points: control points, then the active X-point target (flux equal to the boundary's)
    pr = np.concatenate([cr, [x[0] for x in xts if x[2]]])
    pz = np.concatenate([cz, [x[1] for x in xts if x[2]]])
    gpf_psi = filament_psi(sr_[None, :npf], sz_[None, :npf], pr[:, None], pz[:, None]) * sw[None, :npf]
    ged_psi = (filament_psi(sr_[None, npf:], sz_[None, npf:], pr[:, None], pz[:, None]) @ i_eddy) if len(i_eddy) else np.zeros(len(pr))
    xr = np.array([x[0] for x in xts]); xz = np.array([x[1] for x in xts])
    if len(xts):
        br, bz = filament_b(sr_[None, :], sz_[None, :], xr[:, None], xz[:, None])
        dpr, dpz = xr[:, None] * bz * sw[None, :], -xr[:, None] * br * sw[None, :]      # d psi/dR, d psi/dZ per ampere
    rng_ic = c["ic_range"]
    draw = t["draw"]
    gam = 0.05
    x0 = t["label"]
    mask = (x0 < 1.0) & od.lim_mask
    psin = np.where(mask, np.clip(x0, 0.0, 1.0), 0.0)
    ic = t["ic"].copy()
    psi_prev = None
    last = np.inf
    for it in range(max_iter):
        Jb = OB.basis_columns(psin, mask, r, od.dA, od.n_p, od.n_ff).reshape(-1, od.n_p + od.n_ff) * od.interior[:, None]
        I = Jb @ X
        tot = I.sum()
        if not np.isfinite(tot) or tot <= 0:
            return None
        fac = ip / tot
        I = I * fac
        edge = np.zeros(od.nr * od.nz)
        edge[od.bnd] = od.gb @ I
        psi_pl = od.op.solve_current(I.reshape(od.nz, od.nr), edge.reshape(od.nz, od.nr))
        # coil currents: equal flux at the iso-flux points, zero gradient at the X-point targets
        f_fix = OS.bilinear(psi_pl, r, z, pr, pz) + ged_psi
        A = gpf_psi[1:] - gpf_psi[:1]
        y = -(f_fix[1:] - f_fix[0])
        fs = max(np.max(np.abs(f_fix)), 1e-12) * 0.1
        rows, rhs = [A / fs], [y / fs]
        if len(xts):
            gR = np.zeros_like(psi_pl); gZ = np.zeros_like(psi_pl)
            gR[:, 1:-1] = (psi_pl[:, 2:] - psi_pl[:, :-2]) / (2 * dr)
            gZ[1:-1, :] = (psi_pl[2:, :] - psi_pl[:-2, :]) / (2 * dz)
            fr = OS.bilinear(gR, r, z, xr, xz) + (dpr[:, npf:] @ i_eddy if len(i_eddy) else 0.0)
            fz = OS.bilinear(gZ, r, z, xr, xz) + (dpz[:, npf:] @ i_eddy if len(i_eddy) else 0.0)
            w = sh["a"] / fs
            rows += [dpr[:, :npf] * w, dpz[:, :npf] * w]
            rhs += [-fr * w, -fz * w]
        Af = np.concatenate(rows, axis=0)
        yf = np.concatenate(rhs)
        Areg = np.concatenate([Af * rng_ic, gam * np.eye(npf)], axis=0)
        yreg = np.concatenate([yf, gam * draw / rng_ic])
        u = np.linalg.lstsq(Areg, yreg, rcond=None)[0]
        ic_new = np.concatenate([u * rng_ic, i_eddy])
        ic = ic + 0.7 * (ic_new - ic)
        psi = psi_pl + (od.ggc @ ic).reshape(od.nz, od.nr)
        if psi_prev is not None:
            psi = psi_prev + 0.7 * (psi - psi_prev)
        srch = OS.search(psi, r, z, od.lim_mask, od.xpt_mask, od.lim_r, od.lim_z, od.s)
        if srch["status"] != 0:
            return None
        if psi_prev is not None:
            last = float(np.max(np.abs(psi - psi_prev)) / np.max(np.abs(psi)))
        psi_prev = psi
        psin, mask = srch["psin"], srch["mask"]
        if last < tol:
            break
    if last > 1e-9:
        return None
    return dict(I=I, ic=ic, X=X * fac, kind=sh["kind"], iters=it + 1, resid=last, limited=srch["limited"],
                xpt=srch["xpt"], axis=srch["axis"], psi=psi, max_pf=float(np.max(np.abs(ic[:npf]))))


def _scale_into_range(d, npf, rng_ic):
    """Grad-Shafranov is linear in a common factor on I_p, all currents and psi: shrink the whole
    equilibrium so that the PF currents stay inside the config's range."""
    f = min(1.0, 0.9 * rng_ic / max(d["max_pf"], 1e-30))
    for key in ("I", "ic", "X", "psi"):
        d[key] = d[key] * f
    d["scale"] = f
    d["max_pf"] *= f
    return d


_W = {}


def _init(cfg):
    dev = synth.make_device(cfg)
    dev["geom"]["sigma"] = np.ones(dev["geom"]["n_meas"])      # placeholder, the design loop never fits
    _W["dev"] = dev
    _W["od"] = Device(dev["grid"], dev["geom"], dev["tables"], dev["basis"])


def _design_job(k):
    dev, od = _W["dev"], _W["od"]
    c = dev["meta"]["cfg"]
    d = design_slice(dev, od, k)
    if d is None:
        return k, None
    d = _scale_into_range(d, dev["meta"]["n_pf"], c["ic_range"])
    clean = od.gp @ d["I"] + od.gc @ d["ic"]
    return k, dict(ic=d["ic"], X=d["X"], clean=clean, kind=d["kind"], iters=d["iters"], limited=d["limited"],
                   xpt=np.array(d["xpt"][:4], float), axis=np.array(d["axis"][:4], float), ip=float(d["I"].sum()), max_pf=d["max_pf"])


def _design_until_ok(seed):
    nfail = 0
    while True:
        _, d = _design_job(seed)
        if d is not None:
            return seed, d, nfail
        seed += 10000
        nfail += 1


def _r32(a):
    return np.asarray(a, np.float32).astype(np.float64)


def _coef_change(Xa, Xb, n_p, dz):
    """Largest coefficient change relative to the largest coefficient of its kind (delz: relative to dZ)."""
    npoly = len(Xa) - 1
    e = max(np.max(np.abs(Xa[:n_p] - Xb[:n_p])) / np.max(np.abs(Xb[:n_p])),
            np.max(np.abs(Xa[n_p:npoly] - Xb[n_p:npoly])) / np.max(np.abs(Xb[n_p:npoly])))
    return float(max(e, abs(Xa[-1] - Xb[-1]) / dz))


def _accept_job(args):
    k, b, ic, sigma = args
    dev = _W["dev"]
    c = dev["meta"]["cfg"]
    if _W.get("od_sig") is None:
        g = dict(dev["geom"]); g["sigma"] = sigma
        _W["od_sig"] = Device(dev["grid"], g, dev["tables"], dev["basis"])
        if c["precision"] == "fp32":      # the same device with the tables rounded to FP32 (what the FP32 path sees)
            _W["od_32"] = Device(dev["grid"], g, {kk: _r32(v) for kk, v in dev["tables"].items()}, dev["basis"])
    od = _W["od_sig"]
    res = reconstruct(od, b, ic, c["n_iter"], trace=True)
    dp = [h["dpsi"] for h in res["hist"]]
    rate = (dp[-1] / dp[-6]) ** 0.2 if len(dp) >= 7 and dp[-6] > 0 else 1.0
    sens = 0.0
    if res["status"] == 0 and c["precision"] == "fp32":
        # well-posedness for an FP32 path: (a) rounding every input to FP32 (a 6e-8 perturbation) must not move the
        # coefficients by more than 3e-6 of their kind; (b) white noise of 3e-7 max|psi| on the flux after every iteration
        # (the level of an FP32 solve) must not move the final flux by more than 1e-5 -- the candidate-ownership and
        # vertex-validity rules of the search are discontinuous, and a slice that sits on such a discontinuity cannot be
        # judged at 1e-5 on any FP32 pipeline
        r2 = reconstruct(_W["od_32"], _r32(b), _r32(ic), c["n_iter"])
        sens = _coef_change(r2["X"], res["X"], od.n_p, od.op.dz) if r2["status"] == 0 else 1.0
        for seed in (11, 12, 13):
            r3 = reconstruct(od, b, ic, c["n_iter"], psi_noise=(3e-7, seed))
            dpsi = np.max(np.abs(r3["psi"] - res["psi"])) / np.max(np.abs(res["psi"])) if r3["status"] == 0 else 1.0
            sens = max(sens, 3e-6 * dpsi / 1e-5)
    return k, res["status"], rate, float(res["chi2"]) if res["status"] == 0 else np.nan, (res["srch"]["limited"] if res["srch"] else -1), sens


def generate(cfg, jobs):
    from concurrent.futures import ProcessPoolExecutor
    c = synth.CONFIGS[cfg]
    n = N_STORE[cfg]
    t0 = time.time()
    with ProcessPoolExecutor(max_workers=jobs, initializer=_init, initargs=(cfg,)) as ex:
        # phase 1: design equilibria for seeds 0..n-1 (failed seeds are replaced by k + 10000 * attempt)
        seeds = list(range(n))
        out = {}
        rejected = []
        pending = {k: k for k in seeds}                      # slot -> seed
        while pending:
            res = list(ex.map(_design_job, list(pending.values()), chunksize=1))
            nxt = {}
            for (slot, seed), (_, d) in zip(list(pending.items()), res):
                if d is None:
                    rejected.append((slot, seed, "design"))
                    nxt[slot] = seed + 10000
                else:
                    out[slot] = (seed, d)
            pending = nxt
        print(f"{cfg}: designed {n} slices, {len(rejected)} design rejections, {time.time() - t0:.0f} s", flush=True)
        # sigma: 0.5 % of the per-group RMS of the noise-free signals over the batch
        npb = c["n_probe"]
        clean = np.stack([out[s][1]["clean"] for s in range(n)])
        sigma = np.empty(clean.shape[1])
        sigma[:npb] = 0.005 * np.sqrt(np.mean(clean[:, :npb] ** 2))
        sigma[npb:] = 0.005 * np.sqrt(np.mean(clean[:, npb:] ** 2))

        def noisy(slot, seed, d):
            rng = np.random.default_rng((20260112 + c["idx"]) * 1000 + seed + 500_000_000)
            return d["clean"] + sigma * rng.standard_normal(len(sigma))
        # phase 2: acceptance by the oracle's own reconstruction from the cold start
        b = {s: noisy(s, *out[s]) for s in range(n)}
        todo = list(range(n))
        stats = {}
        while todo:
            res = list(ex.map(_accept_job, [(s, b[s], out[s][1]["ic"], sigma) for s in todo], chunksize=1))
            redo = []
            for s, (_, st, rate, chi2, lim, sens) in zip(todo, res):
                want_div = out[s][1]["kind"] != "limited"
                ok = st == 0 and rate < 0.8 and (lim == 0) == want_div and sens <= 3e-6
                if ok:
                    stats[s] = (rate, chi2, lim)
                else:
                    rejected.append((s, out[s][0], f"accept status={st} rate={rate:.2f} limited={lim} sens={sens:.1e}"))
                    redo.append(s)
            # replacement seeds for the rejected slots, designed in parallel (a worker keeps trying seed + 10000 k)
            new = list(ex.map(_design_until_ok, [out[s][0] + 10000 for s in redo], chunksize=1))
            for s, (seed, d, nfail) in zip(redo, new):
                rejected.extend((s, seed - 10000 * (k + 1), "design") for k in range(nfail))
                out[s] = (seed, d)
                b[s] = noisy(s, seed, d)
            todo = redo
    os.makedirs(CASE_DIR, exist_ok=True)
    M = c["n_probe"] + c["n_loop"]
    nb = c["n_p"] + c["n_ff"] + (5 if c.get("spline") else 0)
    np.savez_compressed(
        os.path.join(CASE_DIR, cfg + ".npz"),
        b=np.stack([b[s] for s in range(n)]), ic=np.stack([out[s][1]["ic"] for s in range(n)]), sigma=sigma,
        X_true=np.stack([out[s][1]["X"] for s in range(n)]), seed=np.array([out[s][0] for s in range(n)]),
        kind=np.array([out[s][1]["kind"] for s in range(n)]), limited=np.array([stats[s][2] for s in range(n)]),
        xpt=np.stack([out[s][1]["xpt"] for s in range(n)]), axis=np.stack([out[s][1]["axis"] for s in range(n)]),
        ip=np.array([out[s][1]["ip"] for s in range(n)]), max_pf=np.array([out[s][1]["max_pf"] for s in range(n)]),
        rate=np.array([stats[s][0] for s in range(n)]), chi2=np.array([stats[s][1] for s in range(n)]),
        dof=np.array(M - nb - 1), n_rejected=np.array(len(rejected)),
        rejected=np.array([f"{a}:{bb}:{cc}" for a, bb, cc in rejected] or [""]))
    ch = np.array([stats[s][1] for s in range(n)])
    print(f"{cfg}: wrote {n} slices; rejections {len(rejected)}; chi2/dof median {np.median(ch) / (M - nb - 1):.2f}; "
          f"contraction median {np.median([stats[s][0] for s in range(n)]):.2f}; I_p {min(out[s][1]['ip'] for s in range(n)) / 1e3:.0f}-"
          f"{max(out[s][1]['ip'] for s in range(n)) / 1e3:.0f} kA; {time.time() - t0:.0f} s", flush=True)


def revalidate(cfg, jobs):
    """Re-run the acceptance on the stored slices of synth/cases/<cfg>.npz (same sigma) and replace the slots that
    fail by new seeds, designed and accepted as in generate()."""
    from concurrent.futures import ProcessPoolExecutor
    c = synth.CONFIGS[cfg]
    path = os.path.join(CASE_DIR, cfg + ".npz")
    with np.load(path) as f:
        F = {k: f[k] for k in f.files}
    n = F["b"].shape[0]
    sigma = F["sigma"]
    t0 = time.time()
    rejected = [r for r in F["rejected"].tolist() if r]
    new_slots = {}

    def noisy(seed, d):
        rng = np.random.default_rng((20260112 + c["idx"]) * 1000 + seed + 500_000_000)
        return d["clean"] + sigma * rng.standard_normal(len(sigma))
    with ProcessPoolExecutor(max_workers=jobs, initializer=_init, initargs=(cfg,)) as ex:
        cur = {s: (int(F["seed"][s]), None, F["b"][s], F["ic"][s], str(F["kind"][s])) for s in range(n)}
        todo = list(range(n))
        stats = {}
        while todo:
            res = list(ex.map(_accept_job, [(s, cur[s][2], cur[s][3], sigma) for s in todo], chunksize=1))
            redo = []
            for s, (_, st, rate, chi2, lim, sens) in zip(todo, res):
                ok = st == 0 and rate < 0.8 and (lim == 0) == (cur[s][4] != "limited") and sens <= 3e-6
                if ok:
                    stats[s] = (rate, chi2, lim)
                else:
                    rejected.append(f"{s}:{cur[s][0]}:accept status={st} rate={rate:.2f} limited={lim} sens={sens:.1e}")
                    redo.append(s)
            new = list(ex.map(_design_until_ok, [cur[s][0] + 10000 for s in redo], chunksize=1))
            for s, (seed, d, nfail) in zip(redo, new):
                rejected.extend(f"{s}:{seed - 10000 * (k + 1)}:design" for k in range(nfail))
                cur[s] = (seed, d, noisy(seed, d), d["ic"], d["kind"])
                new_slots[s] = d
            print(f"{cfg}: revalidation round: {len(todo)} checked, {len(redo)} replaced, {time.time() - t0:.0f} s", flush=True)
            todo = redo
    for s, d in new_slots.items():
        F["b"][s] = cur[s][2]; F["ic"][s] = d["ic"]; F["X_true"][s] = d["X"]; F["seed"][s] = cur[s][0]; F["kind"][s] = d["kind"]
        F["xpt"][s] = d["xpt"]; F["axis"][s] = d["axis"]; F["ip"][s] = d["ip"]; F["max_pf"][s] = d["max_pf"]
    for s in range(n):
        F["limited"][s] = stats[s][2]; F["rate"][s] = stats[s][0]; F["chi2"][s] = stats[s][1]
    F["n_rejected"] = np.array(len(rejected)); F["rejected"] = np.array(rejected or [""])
    np.savez_compressed(path, **F)
    print(f"{cfg}: revalidated {n} slices, {len(new_slots)} replaced; rejections in total {len(rejected)}; {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("cfgs", nargs="*", default=list(N_STORE))
    ap.add_argument("--jobs", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--revalidate", action="store_true", help="keep the stored slices that still pass the acceptance, replace the others")
    a = ap.parse_args()
    for cfg in a.cfgs:
        (revalidate if a.revalidate else generate)(cfg, a.jobs)
