"""Axis / X-point / LCFS search and flux normalisation (Sec. II.D).

Oracle-side (test infrastructure).  Brute-force scans over the whole grid in float64.

What the paper fixes: a second-order polynomial fit "in the vicinity of each grid point"
with pre-inverted normal equations; O-points have det H > 0 and X-points
det H < 0; the boundary flux is found "by comparing the flux values of all
limiter vertices and X-points within the plasmas region".
What it does not fix (plasma-region rule, window size, ties) follows DESIGN.md reading O3;
those rules are **parity unpinned by the paper**.
Arrays are [j, i]; flat index n = j*nr + i; x runs along R (i), y along Z (j).
"""
import numpy as np

_XS = np.array([-1.0, 0.0, 1.0])


def fit_design_pinv():
    """Pre-inverted normal equations of the 3x3 quadratic fit:
    rows = (c0, cx, cy, cxx, cxy, cyy), columns = the 9 stencil points ordered y-major
    (y=-1: x=-1,0,1; y=0: ...; y=+1: ...).  Computed here by numpy's pinv of the design
    matrix -- NOT by the integer-weight table the CUDA path uses."""
    X, Y = np.meshgrid(_XS, _XS)  # Y varies along axis 0
    x, y = X.ravel(), Y.ravel()
    A = np.stack([np.ones(9), x, y, x * x, x * y, y * y], axis=1)
    return np.linalg.pinv(A)


_PINV = fit_design_pinv()


def quad_fit(psi):
    """Fit c0+cx x+cy y+cxx x^2+cxy xy+cyy y^2 to the 3x3 neighbourhood of every interior
    node (index units).  Returns dict of [nz-2, nr-2] arrays incl. det H/…, stationary point."""
    nz, nr = psi.shape
    st = np.stack([psi[1 + dy:nz - 1 + dy, 1 + dx:nr - 1 + dx]
                   for dy in (-1, 0, 1) for dx in (-1, 0, 1)], axis=0)  # [9, nz-2, nr-2]
    c = np.tensordot(_PINV, st, axes=(1, 0))
    c0, cx, cy, cxx, cxy, cyy = c
    det = 4.0 * cxx * cyy - cxy * cxy          # det of the Hessian [[2cxx, cxy],[cxy, 2cyy]]
    with np.errstate(divide="ignore", invalid="ignore"):
        xs = -(2.0 * cyy * cx - cxy * cy) / det   # grad = 0
        ys = -(2.0 * cxx * cy - cxy * cx) / det
    ps = c0 + 0.5 * (cx * xs + cy * ys)
    return dict(c0=c0, cx=cx, cy=cy, cxx=cxx, cxy=cxy, cyy=cyy, det=det, xs=xs, ys=ys, ps=ps)


def bilinear(psi, r, z, rr, zz):
    """Bilinear interpolation of psi[j, i] at points (rr, zz) on the uniform grid r, z."""
    dr, dz = r[1] - r[0], z[1] - z[0]
    fi = (np.asarray(rr) - r[0]) / dr
    fj = (np.asarray(zz) - z[0]) / dz
    i0 = np.clip(np.floor(fi).astype(int), 0, len(r) - 2)
    j0 = np.clip(np.floor(fj).astype(int), 0, len(z) - 2)
    tx, ty = fi - i0, fj - j0
    return ((1 - ty) * ((1 - tx) * psi[j0, i0] + tx * psi[j0, i0 + 1])
            + ty * ((1 - tx) * psi[j0 + 1, i0] + tx * psi[j0 + 1, i0 + 1]))


def search(psi, r, z, lim_mask, xpt_mask, lim_r, lim_z, s=1):
    """One O3 pass.  psi[nz, nr]; lim_mask/xpt_mask bool [nz, nr]; s = sign(I_p).
    Returns dict: status, axis (i, j, R, Z, psi), xpt (i, j, R, Z, psi) or i=j=-1, psi_b,
    limited, mask[nz, nr] (bool), psin[nz, nr] (clamped to [0,1] in the mask, 0 outside),
    axis_margin, xpt_margin, n_cand."""
    nz, nr = psi.shape
    dr, dz = r[1] - r[0], z[1] - z[0]
    out = dict(status=0, axis=(-1, -1, np.nan, np.nan, np.nan), xpt=(-1, -1, np.nan, np.nan, np.nan),
               psi_b=np.nan, limited=1, mask=np.zeros((nz, nr), bool), psin=np.zeros((nz, nr)),
               axis_margin=np.nan, xpt_margin=np.nan, n_cand=0, bnd_margin=np.inf, valid_margin=np.inf)
    if not np.all(np.isfinite(psi)):
        out["status"] = 2
        return out
    f = quad_fit(psi)
    # 1. axis node: arg-max of s*psi over lim_mask, tie -> smallest flat index (np.argmax)
    sp = np.where(lim_mask, s * psi, -np.inf)
    na = int(np.argmax(sp.ravel()))
    ja, ia = divmod(na, nr)
    spa_sorted = np.sort(sp.ravel())[::-1]
    fa = {k: v[ja - 1, ia - 1] for k, v in f.items()}
    if not (fa["det"] > 0.0) or max(abs(fa["xs"]), abs(fa["ys"])) > 1.0:
        out["status"] = 1
        return out
    Ra, Za, psia = r[ia] + fa["xs"] * dr, z[ja] + fa["ys"] * dz, fa["ps"]
    out["axis"] = (ia, ja, Ra, Za, psia)
    # 2. X candidates
    cand = (xpt_mask[1:-1, 1:-1] & (f["det"] < 0.0) & (np.abs(f["xs"]) <= 0.5)
            & (np.abs(f["ys"]) <= 0.5) & (s * f["ps"] < s * psia))
    cj, ci = np.nonzero(cand)          # row-major order => ascending flat index
    cR = r[ci + 1] + f["xs"][cj, ci] * dr
    cZ = z[cj + 1] + f["ys"][cj, ci] * dz
    cP = f["ps"][cj, ci]
    out["n_cand"] = len(ci)
    # 3. limiter vertices, valid iff not behind any candidate as seen from the axis
    pv = bilinear(psi, r, z, lim_r, lim_z)
    valid = np.ones(len(lim_r), bool)
    for c in range(len(ci)):
        valid &= ((lim_r - cR[c]) * (Ra - cR[c]) + (lim_z - cZ[c]) * (Za - cZ[c])) >= 0.0
    # 4. boundary flux
    best_lim = np.max(s * pv[valid]) if valid.any() else -np.inf
    if len(ci):
        kx = int(np.argmax(s * cP))     # tie -> first = smaller flat index
        best_x = s * cP[kx]
        out["xpt"] = (int(ci[kx]) + 1, int(cj[kx]) + 1, cR[kx], cZ[kx], cP[kx])
    else:
        best_x = -np.inf
    if best_x > best_lim:
        out["limited"] = 0
        spb = best_x
    else:
        spb = best_lim
    if not np.isfinite(spb):
        out["status"] = 1
        return out
    # decision margins (diagnostics only; the case generator rejects seeds whose decisions are fragile):
    # bnd_margin = gap between the best X-point and the best valid limiter vertex; valid_margin = how far the
    # half-plane test of a vertex that matters is from flipping (normalised dot product): vertices above the
    # boundary flux are all invalid -- the least firmly invalid one counts -- and so does the winning vertex.
    scale0 = abs(psia - s * spb)
    out["bnd_margin"] = abs(best_x - best_lim) / scale0 if (np.isfinite(best_x) and np.isfinite(best_lim) and scale0 > 0) else np.inf
    vm = np.inf
    if len(ci):
        dots = np.stack([((lim_r - cR[c]) * (Ra - cR[c]) + (lim_z - cZ[c]) * (Za - cZ[c]))
                         / (np.hypot(lim_r - cR[c], lim_z - cZ[c]) * np.hypot(Ra - cR[c], Za - cZ[c]) + 1e-300) for c in range(len(ci))])
        above = (~valid) & (s * pv > spb)
        if above.any():
            vm = min(vm, float(np.min(-np.min(dots[:, above], axis=0))))      # most negative dot of each such vertex
        if out["limited"] == 1 and valid.any():
            kw = int(np.argmax(np.where(valid, s * pv, -np.inf)))
            vm = min(vm, float(np.min(dots[:, kw])))
    out["valid_margin"] = vm
    psib = s * spb
    out["psi_b"] = psib
    # 5. plasma region
    R2, Z2 = np.meshgrid(r, z)
    mask = lim_mask & (s * (psi - psib) > 0.0)
    for c in range(len(ci)):
        mask &= ((R2 - cR[c]) * (Ra - cR[c]) + (Z2 - cZ[c]) * (Za - cZ[c])) > 0.0
    # 6. normalised flux
    if not mask.any() or psib == psia:
        out["status"] = 1
        return out
    psin = np.clip((psi - psia) / (psib - psia), 0.0, 1.0)
    out["mask"] = mask
    out["psin"] = np.where(mask, psin, 0.0)
    # margins (diagnostics for the near-tie clause)
    scale = abs(psia - psib)
    out["axis_margin"] = (spa_sorted[0] - spa_sorted[1]) / scale if len(spa_sorted) > 1 else np.inf
    if len(ci) > 1:
        o = np.sort(s * cP)[::-1]
        # neighbours claiming the same saddle have (nearly) equal fitted values; margin to the
        # next *distinct* saddle is what matters, reported as gap between best and 2nd best
        out["xpt_margin"] = (o[0] - o[1]) / scale
    return out


def cold_start(r, z, lim_mask, rc, zc, a, b):
    """O2 (paper silent; it only warm-starts): psin0 = min(1, ((R-Rc)/a)^2 +
    ((Z-Zc)/b)^2), mask0 = (psin0 < 1) & lim_mask."""
    R2, Z2 = np.meshgrid(r, z)
    x = np.minimum(1.0, ((R2 - rc) / a) ** 2 + ((Z2 - zc) / b) ** 2)
    mask = (x < 1.0) & lim_mask
    return np.where(mask, x, 0.0), mask
