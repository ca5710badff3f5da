"""Pins of the oracle's flux-surface post-processing (oracle/fluxsurf.py; Eq. 12) on
analytic flux maps whose surfaces, perimeters and integrals have closed forms."""
import numpy as np
import pytest
from scipy.integrate import quad

from oracle import fluxsurf as FS


def _ellipse_case(R0=0.8, Z0=0.05, kap=1.6, rho_b=0.35, c=1.0, n=129, rlo=0.15, rhi=1.6, zlo=-1.6, zhi=1.6):
    r = np.linspace(rlo, rhi, n); z = np.linspace(zlo, zhi, n)
    R2, Z2 = np.meshgrid(r, z)
    s = (R2 - R0) ** 2 + (Z2 - Z0) ** 2 / kap ** 2
    psi_a = 0.3
    psi = psi_a - c * s
    psi_b = psi_a - c * rho_b ** 2
    psin = s / rho_b ** 2
    mask = psin < 1.0
    return r, z, psi, np.where(mask, psin, 0.0), mask, psi_a, psi_b


def test_vertices_on_the_analytic_surfaces_and_counter_clockwise():
    R0, Z0, kap, rb = 0.8, 0.05, 1.6, 0.35
    r, z, psi, psin, mask, pa, pb = _ellipse_case(R0, Z0, kap, rb)
    o = FS.flux_surfaces(psi, psin, mask, r, z, R0, Z0, pa, pb, n_prof=8, n_chord=64, n_bisect=10)
    assert o["status"] == 0
    for p in range(8):
        x = (p + 1) / 8
        v = o["vert"][p]
        th = 2 * np.pi * np.arange(64) / 64
        rad_exact = np.sqrt(x) * rb / np.sqrt(np.cos(th) ** 2 + np.sin(th) ** 2 / kap ** 2)
        rad = np.hypot(v[:, 0] - R0, v[:, 1] - Z0)
        assert np.max(np.abs(rad - rad_exact)) < 1.2e-3            # ~1 mm after 10 bisections
        ang = np.arctan2(v[:, 1] - Z0, v[:, 0] - R0)
        assert np.max(np.abs(np.angle(np.exp(1j * (ang - th))))) < 1e-12   # the vertex stays on its chord
        area = 0.5 * np.sum(v[:, 0] * np.roll(v[:, 1], -1) - np.roll(v[:, 0], -1) * v[:, 1])
        assert area > 0 and abs(area / (np.pi * kap * x * rb ** 2) - 1) < 1.5e-2   # counter-clockwise polygon
    g = o["geom"]
    assert abs(g[4] / rb - 1) < 3e-3 and abs(g[5] / kap - 1) < 3e-3
    assert abs(g[0] - (R0 - rb)) < 1.5e-3 and abs(g[1] - (R0 + rb)) < 1.5e-3


def test_more_bisections_move_the_vertices_by_less_than_a_millimetre():
    r, z, psi, psin, mask, pa, pb = _ellipse_case()
    a = FS.flux_surfaces(psi, psin, mask, r, z, 0.8, 0.05, pa, pb, n_prof=4, n_chord=32, n_bisect=10)["vert"]
    b = FS.flux_surfaces(psi, psin, mask, r, z, 0.8, 0.05, pa, pb, n_prof=4, n_chord=32, n_bisect=24)["vert"]
    assert np.max(np.hypot(a[..., 0] - b[..., 0], a[..., 1] - b[..., 1])) < 1e-3


def test_integrals_on_circular_surfaces():
    """kappa = 1: |grad psi| = 2 c rho on the surface of radius rho, so
    Q_{0,0} = 2 pi rho, Q_{-1,-1} = pi / (c sqrt(R0^2 - rho^2)), Q_{-1,-2} = pi R0 / (c (R0^2 - rho^2)^{3/2})."""
    R0, rb, c = 0.8, 0.35, 1.3
    r, z, psi, psin, mask, pa, pb = _ellipse_case(R0, 0.0, 1.0, rb, c)
    o = FS.flux_surfaces(psi, psin, mask, r, z, R0, 0.0, pa, pb, n_prof=5, n_chord=128, munu=((-1, -1), (-1, -2), (0, 0)))
    for p in range(5):
        rho = np.sqrt((p + 1) / 5) * rb
        assert abs(o["Q"][p, 2] / (2 * np.pi * rho) - 1) < 5e-3     # 1 mm on a 15-35 cm radius
        assert abs(o["Q"][p, 0] / (np.pi / (c * np.sqrt(R0 ** 2 - rho ** 2))) - 1) < 1.5e-2
        assert abs(o["Q"][p, 1] / (np.pi * R0 / (c * (R0 ** 2 - rho ** 2) ** 1.5)) - 1) < 1.5e-2


def test_safety_factor_large_aspect_ratio_and_ffprime_integral():
    """q = (mu0 F / 2 pi) Q_{-1,-1} = mu0 F / (2 c sqrt(R0^2 - rho^2)) on circular surfaces (-> the cylinder's
    rho B_phi / (R0 B_theta) for rho << R0); F(x) from the FF' polynomial against numerical quadrature."""
    R0, rb, c = 10.0, 0.4, 0.7
    r, z, psi, psin, mask, pa, pb = _ellipse_case(R0, 0.0, 1.0, rb, c, n=129, rlo=9.4, rhi=10.6, zlo=-0.6, zhi=0.6)
    F = 2.0e6
    o = FS.flux_surfaces(psi, psin, mask, r, z, R0, 0.0, pa, pb, n_prof=4, n_chord=128, f_vac=F)
    for p in range(4):
        rho = np.sqrt((p + 1) / 4) * rb
        q_exact = FS.MU0 * F / (2 * c * np.sqrt(R0 ** 2 - rho ** 2))
        assert abs(o["q"][p] / q_exact - 1) < 1.5e-2
        b_phi, b_th = FS.MU0 * F / R0, 2 * c * rho / R0                # the paper's F is R B_phi / mu0
        assert abs(o["q"][p] / (rho * b_phi / (R0 * b_th)) - 1) < 2e-2      # cylinder limit
    Xff = np.array([3.0e5, -1.0e5, 2.0e5])
    for x in (0.0, 0.3, 0.9):
        num = quad(lambda t: sum(Xff[j] * (t ** j - t ** 3) for j in range(3)), x, 1.0)[0]
        assert abs(FS.ffprime_integral(x, Xff, 3) - num) < 1e-9 * abs(num)
    o2 = FS.flux_surfaces(psi, psin, mask, r, z, R0, 0.0, pa, pb, n_prof=4, n_chord=128, f_vac=F, Xff=Xff, n_ff=3)
    x = 0.25
    f2 = F ** 2 - 2 * (pb - pa) * FS.ffprime_integral(x, Xff, 3)
    assert abs(o2["q"][0] / o["q"][0] - np.sqrt(f2) / F) < 1e-12


def test_bilinear_helpers_are_exact_on_bilinear_fields():
    r = np.linspace(0.0, 1.0, 11); z = np.linspace(-1.0, 1.0, 21)
    R2, Z2 = np.meshgrid(r, z)
    f = 2.0 + 3.0 * R2 - 1.5 * Z2 + 0.7 * R2 * Z2
    for (R, Z) in ((0.234, -0.377), (0.91, 0.655)):
        assert abs(FS.bilinear_at(f, r, z, R, Z) - (2.0 + 3.0 * R - 1.5 * Z + 0.7 * R * Z)) < 1e-14
        gR, gZ = FS.grad_at(f, r, z, R, Z)
        assert abs(gR - (3.0 + 0.7 * Z)) < 1e-12 and abs(gZ - (-1.5 + 0.7 * R)) < 1e-12
