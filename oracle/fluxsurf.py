"""Flux-surface post-processing (Sec. II.E, Eq. 12, Fig. 1): flux-surface vertices by
bisection along chords from the magnetic axis, Q_{mu,nu} = closed integral of |grad psi|^mu R^nu dl,
safety factor, LCFS geometry.

Oracle-side (test infrastructure).  Plain float64 loops over levels and chords.

What the paper fixes: bisection between the axis and a point of the reconstructed boundary, one chord
per thread, the flux outside the plasma region filtered with the boolean matrix of Sec. II.D so that it
is monotonic along the chord, linear interpolation of the grid flux at each new vertex, the boundary
points ordered (counter-)clockwise, "about 10 iterations".
Readings (O8; the paper gives no further detail):
  * chords: n_chord rays from the refined axis at angles 2 pi c / n_chord, counter-clockwise;
  * filtered field F = psi_N inside the mask and max(1, (psi - psi_a)/(psi_b - psi_a)) outside it (the flux
    outside the plasma is clipped from below at the boundary value, which keeps F monotonic along a chord
    and leaves the cell that holds the LCFS unsmeared), interpolated bilinearly;
  * boundary end of a chord: marching outwards in steps of h = min(dR, dZ)/2, the first point with
    F >= 1 (or outside the grid) closes the bracket;
  * level x: n_bisect halvings of the bracket [0, t_b] on F(t) - x, then one linear interpolation
    between the bracket ends gives the vertex;
  * |grad psi| at a vertex = gradient of the bilinear interpolant of psi in the vertex's cell;
  * the closed integral is the trapezoid rule on the polygon of the n_chord vertices;
  * levels x_p = (p + 1)/n_prof, p = 0..n_prof-1 (the last one is the LCFS);
  * safety factor: with psi per radian (COCOS 7) the poloidal field is |grad psi|/R and the paper's F is
    R B_phi / mu0 (Eq. 1, 10), so q = (mu0 F / 2 pi) Q_{-1,-1}.  The paper prints Q_{-1,-2}
    (PAPER.md:144), which matches only if |grad Psi| is read as B_p; both integrals are returned, q uses
    the dimensionally consistent one.  F(x)^2 = F_vac^2 - 2 (psi_b - psi_a) * integral_x^1 FF'(t) dt with
    FF'(t) = sum_j X_j (t^j - t^n_ff) (Eq. 9-10; polynomial terms only).
"""
import numpy as np

MU0 = 4.0e-7 * np.pi


def _cell(r, z, R, Z):
    dr, dz = r[1] - r[0], z[1] - z[0]
    fi, fj = (R - r[0]) / dr, (Z - z[0]) / dz
    i0 = int(min(max(np.floor(fi), 0), len(r) - 2))
    j0 = int(min(max(np.floor(fj), 0), len(z) - 2))
    return i0, j0, fi - i0, fj - j0


def bilinear_at(f, r, z, R, Z):
    i0, j0, tx, ty = _cell(r, z, R, Z)
    return ((1 - ty) * ((1 - tx) * f[j0, i0] + tx * f[j0, i0 + 1]) + ty * ((1 - tx) * f[j0 + 1, i0] + tx * f[j0 + 1, i0 + 1]))


def grad_at(f, r, z, R, Z):
    """Gradient of the bilinear interpolant in the cell containing (R, Z)."""
    i0, j0, tx, ty = _cell(r, z, R, Z)
    dr, dz = r[1] - r[0], z[1] - z[0]
    gR = ((1 - ty) * (f[j0, i0 + 1] - f[j0, i0]) + ty * (f[j0 + 1, i0 + 1] - f[j0 + 1, i0])) / dr
    gZ = ((1 - tx) * (f[j0 + 1, i0] - f[j0, i0]) + tx * (f[j0 + 1, i0 + 1] - f[j0, i0 + 1])) / dz
    return gR, gZ


def ffprime_integral(x, Xff, n_ff):
    """integral_x^1 sum_j X_j (t^j - t^n_ff) dt."""
    tot = 0.0
    for j in range(n_ff):
        tot += Xff[j] * ((1 - x ** (j + 1)) / (j + 1) - (1 - x ** (n_ff + 1)) / (n_ff + 1))
    return tot


def flux_surfaces(psi, psin, mask, r, z, axis_r, axis_z, psi_a, psi_b, n_prof=33, n_chord=128, n_bisect=10,
                  munu=((-1, -1), (-1, -2), (0, 0)), f_vac=0.0, Xff=None, n_ff=0):
    """Returns dict(vert[n_prof, n_chord, 2], Q[n_prof, len(munu)], q[n_prof], geom[6] = (R_min, R_max, Z_min,
    Z_max of the LCFS polygon, minor radius a, elongation kappa), status) ; status 1 = a chord found no
    boundary (axis outside the plasma)."""
    F = np.where(mask, psin, np.maximum((psi - psi_a) / (psi_b - psi_a), 1.0))
    dr, dz = r[1] - r[0], z[1] - z[0]
    h = 0.5 * min(dr, dz)
    vert = np.zeros((n_prof, n_chord, 2))
    status = 0
    for c in range(n_chord):
        th = 2.0 * np.pi * c / n_chord
        ct, st = np.cos(th), np.sin(th)
        # boundary end of the chord
        k = 1
        while True:
            R, Z = axis_r + k * h * ct, axis_z + k * h * st
            if R <= r[0] or R >= r[-1] or Z <= z[0] or Z >= z[-1] or bilinear_at(F, r, z, R, Z) >= 1.0:
                break
            k += 1
        tb = k * h
        if k == 1 and bilinear_at(F, r, z, axis_r, axis_z) >= 1.0:
            status = 1
        for p in range(n_prof):
            x = (p + 1.0) / n_prof
            lo, hi = 0.0, tb
            for _ in range(n_bisect):
                mid = 0.5 * (lo + hi)
                R, Z = axis_r + mid * ct, axis_z + mid * st
                inside = r[0] < R < r[-1] and z[0] < Z < z[-1]
                fm = bilinear_at(F, r, z, R, Z) if inside else 1.0
                if fm < x:
                    lo = mid
                else:
                    hi = mid
            Rl, Zl, Rh, Zh = axis_r + lo * ct, axis_z + lo * st, axis_r + hi * ct, axis_z + hi * st
            fl = bilinear_at(F, r, z, Rl, Zl)
            fh = bilinear_at(F, r, z, Rh, Zh) if (r[0] < Rh < r[-1] and z[0] < Zh < z[-1]) else 1.0
            w = (x - fl) / (fh - fl) if fh > fl else 0.5
            w = min(max(w, 0.0), 1.0)
            t = lo + w * (hi - lo)
            vert[p, c] = (axis_r + t * ct, axis_z + t * st)
    Q = np.zeros((n_prof, len(munu)))
    for p in range(n_prof):
        g = np.zeros((n_chord, len(munu)))
        for c in range(n_chord):
            R, Z = vert[p, c]
            gR, gZ = grad_at(psi, r, z, R, Z)
            gn = np.hypot(gR, gZ)
            for e, (mu, nu) in enumerate(munu):
                g[c, e] = gn ** mu * R ** nu
        for c in range(n_chord):
            c1 = (c + 1) % n_chord
            dl = np.hypot(vert[p, c1, 0] - vert[p, c, 0], vert[p, c1, 1] - vert[p, c, 1])
            Q[p] += 0.5 * (g[c] + g[c1]) * dl
    q = np.full(n_prof, np.nan)
    if (-1, -1) in tuple(map(tuple, munu)):
        e = list(map(tuple, munu)).index((-1, -1))
        for p in range(n_prof):
            x = (p + 1.0) / n_prof
            f2 = f_vac ** 2 - 2.0 * (psi_b - psi_a) * (ffprime_integral(x, Xff, n_ff) if Xff is not None else 0.0)
            q[p] = MU0 * np.sqrt(max(f2, 0.0)) / (2.0 * np.pi) * Q[p, e]
    lc = vert[-1]
    rmin, rmax, zmin, zmax = lc[:, 0].min(), lc[:, 0].max(), lc[:, 1].min(), lc[:, 1].max()
    geom = np.array([rmin, rmax, zmin, zmax, 0.5 * (rmax - rmin), (zmax - zmin) / (rmax - rmin)])
    return dict(vert=vert, Q=Q, q=q, geom=geom, status=status)
