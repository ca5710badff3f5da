"""Pins for oracle/greens.py (Eq. 3-5)."""
import os

import numpy as np

from oracle import greens as G

HERE = os.path.dirname(__file__)


def _quad(f, n=4000):
    phi = (np.arange(n) + 0.5) * 2 * np.pi / n      # midpoint rule: spectrally accurate on a period
    return np.sum(f(phi)) * 2 * np.pi / n


def test_golden_values():
    for line in open(os.path.join(HERE, "golden", "greens_golden.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        v = [float(x) for x in t[1:]]
        if t[0] in "KE":
            K, E = G.ellip_ke(v[0])
            assert abs((K if t[0] == "K" else E) / v[1] - 1) < 1e-14
        elif t[0] == "G":
            psi = G.psi_filament(*v[:4])
            br, bz = G.b_filament(*v[:4])
            assert abs(psi / v[4] - 1) < 1e-13 and abs(br / v[5] - 1) < 1e-13 and abs(bz / v[6] - 1) < 1e-13
        else:
            assert abs(G.psi_filament(*v[:4]) / v[4] - 1) < 1e-12


def test_elliptic_against_library():
    from scipy.special import ellipk, ellipe
    m = np.concatenate([np.linspace(0, 0.999, 200), 1 - np.logspace(-12, -3, 20)])
    K, E = G.ellip_ke(m)
    assert np.max(np.abs(K / ellipk(m) - 1)) < 5e-15
    assert np.max(np.abs(E / ellipe(m) - 1)) < 5e-15


def test_psi_equals_eq5_quadrature():
    """Eq. 5 integrated directly: field point (r, z), source loop (r', z')."""
    rng = np.random.default_rng(1)
    for _ in range(10):
        rp, zp, r, z = rng.uniform(0.2, 1.6), rng.uniform(-1, 1), rng.uniform(0.2, 1.6), rng.uniform(-1, 1)
        if abs(rp - r) + abs(zp - z) < 0.2:
            continue
        q = _quad(lambda p: r * rp * np.cos(p) / np.sqrt((z - zp) ** 2 + (r - rp * np.cos(p)) ** 2 + (rp * np.sin(p)) ** 2))
        assert abs(G.MU0 / (4 * np.pi) * q / G.psi_filament(rp, zp, r, z) - 1) < 1e-10


def test_b_equals_biot_savart_quadrature():
    """Eq. 3-4 with the 3/2 power reading: B = mu0 I/(4 pi) int dl x d / |d|^3."""
    rng = np.random.default_rng(2)
    for _ in range(10):
        a, zs, r, z = rng.uniform(0.2, 1.6), rng.uniform(-1, 1), rng.uniform(0.2, 1.6), rng.uniform(-1, 1)
        if abs(a - r) + abs(zs - z) < 0.2:
            continue
        den = lambda p: ((z - zs) ** 2 + (r - a * np.cos(p)) ** 2 + (a * np.sin(p)) ** 2) ** 1.5
        br = G.MU0 / (4 * np.pi) * _quad(lambda p: a * (z - zs) * np.cos(p) / den(p))
        bz = G.MU0 / (4 * np.pi) * _quad(lambda p: (a * a - r * a * np.cos(p)) / den(p))
        obr, obz = G.b_filament(a, zs, r, z)
        assert abs(br - obr) < 1e-10 * abs(obz) + 1e-18 and abs(bz / obz - 1) < 1e-9


def test_reciprocity_and_cocos7():
    rng = np.random.default_rng(3)
    a, zs, r, z = rng.uniform(0.2, 1.6, 50), rng.uniform(-1, 1, 50), rng.uniform(0.2, 1.6, 50), rng.uniform(-1, 1, 50)
    assert np.max(np.abs(G.psi_filament(a, zs, r, z) / G.psi_filament(r, z, a, zs) - 1)) < 1e-14
    h = 1e-5   # COCOS 7: B_R = -psi_Z / R, B_Z = +psi_R / R
    br, bz = G.b_filament(a, zs, r, z)
    dpz = (G.psi_filament(a, zs, r, z + h) - G.psi_filament(a, zs, r, z - h)) / (2 * h)
    dpr = (G.psi_filament(a, zs, r + h, z) - G.psi_filament(a, zs, r - h, z)) / (2 * h)
    scale = np.hypot(br, bz)
    assert np.max(np.abs(br + dpz / r) / scale) < 1e-6
    assert np.max(np.abs(bz - dpr / r) / scale) < 1e-6


def test_synth_tables_agree_with_oracle_greens(dev_cfg1):
    """The generator tabulates with scipy.special; the oracle's AGM forms must reproduce it."""
    d, _ = dev_cfg1
    m, t, g = d["meta"], d["tables"], d["grid"]
    R2, Z2 = np.meshgrid(m["r"], m["z"])
    n = 5 * g["nr"] + 7
    npb = m["n_probe"]
    loops = G.psi_filament(R2.ravel()[n], Z2.ravel()[n], m["sen_r"][npb:], m["sen_z"][npb:])
    assert np.allclose(t["gp"][npb:, n], loops, rtol=1e-8, atol=0)
    br, bz = G.b_filament(R2.ravel()[n], Z2.ravel()[n], m["sen_r"][:npb], m["sen_z"][:npb])
    assert np.allclose(t["gp"][:npb, n], np.cos(m["alpha"]) * br + np.sin(m["alpha"]) * bz, rtol=1e-8, atol=1e-20)
    from oracle.gs_solve import boundary_nodes
    bn = boundary_nodes(g["nr"], g["nz"])
    k = 40
    assert np.allclose(t["gb"][k, n], G.psi_filament(R2.ravel()[n], Z2.ravel()[n], R2.ravel()[bn[k]], Z2.ravel()[bn[k]]), rtol=1e-8)
    assert np.all(t["gb"][:, bn] == 0) and np.all(t["gp"][:, bn] == 0)
    c = 3
    assert np.allclose(t["ggc"][:, c], m["src_w"][c] * G.psi_filament(m["src_r"][c], m["src_z"][c], R2.ravel(), Z2.ravel()), rtol=1e-8)
