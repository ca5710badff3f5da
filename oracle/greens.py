"""Green's functions of a toroidal current filament (Sec. II.A, Eq. 3-5).

Oracle-side (test infrastructure).  Closed forms in complete elliptic integrals, with our own
AGM evaluation of K and E; pinned in tests/test_oracle_greens.py against direct quadrature of
Eq. 5 and of Biot-Savart, golden values, and reciprocity.

Reading of the garbled Eq. 3-4: the printed denominators carry a square
root; Biot-Savart needs the power 3/2, and in the numerators r' is the SOURCE loop radius.
Eq. 5 (flux) is taken as printed: psi is flux per radian (no 2*pi), COCOS 7.
"""
import numpy as np

MU0 = 4.0e-7 * np.pi  # DESIGN.md reading O0: paper gives no value


def ellip_ke(m):
    """Complete elliptic integrals K(m), E(m), parameter m = k^2 in [0, 1), by the
    arithmetic-geometric mean (Abramowitz & Stegun 17.6): a0=1, b0=sqrt(1-m), c0=sqrt(m);
    K = pi/(2 a_N);  E = K * (1 - sum_n 2^(n-1) c_n^2)."""
    m = np.asarray(m, dtype=np.float64)
    a = np.ones_like(m)
    b = np.sqrt(1.0 - m)
    csum = 0.5 * m  # 2^(0-1) * c0^2
    pw = 0.5
    for _ in range(40):
        c = 0.5 * (a - b)
        a, b = 0.5 * (a + b), np.sqrt(a * b)
        pw *= 2.0
        csum = csum + pw * c * c
        if np.all(np.abs(c) <= 1e-17 * np.abs(a)):
            break
    K = np.pi / (2.0 * a)
    E = K * (1.0 - csum)
    return K, E


def psi_filament(a, zs, rho, zf):
    """Flux per radian at (rho, zf) from a unit-current filament of radius a at height zs.
    Equals Eq. 5: psi = mu0/(2 pi) * sqrt(a rho) * [(2-k^2) K - 2 E] / k,
    k^2 = 4 a rho / ((a+rho)^2 + z^2)."""
    a, zs, rho, zf = np.broadcast_arrays(*(np.asarray(v, dtype=np.float64) for v in (a, zs, rho, zf)))
    z = zf - zs
    k2 = 4.0 * a * rho / ((a + rho) ** 2 + z * z)
    K, E = ellip_ke(k2)
    k = np.sqrt(k2)
    return MU0 / (2.0 * np.pi) * np.sqrt(a * rho) * ((2.0 - k2) * K - 2.0 * E) / k


def b_filament(a, zs, rho, zf):
    """(B_R, B_Z) at (rho, zf) from a unit-current filament (Biot-Savart; Eq. 3-4 with the
    power 3/2 reading).  COCOS 7: B_R = -(1/R) dpsi/dZ, B_Z = +(1/R) dpsi/dR."""
    a, zs, rho, zf = np.broadcast_arrays(*(np.asarray(v, dtype=np.float64) for v in (a, zs, rho, zf)))
    z = zf - zs
    s2 = (a + rho) ** 2 + z * z
    d2 = (a - rho) ** 2 + z * z
    K, E = ellip_ke(4.0 * a * rho / s2)
    pref = MU0 / (2.0 * np.pi) / np.sqrt(s2)
    bz = pref * (K + (a * a - rho * rho - z * z) / d2 * E)
    br = pref * z / rho * (-K + (a * a + rho * rho + z * z) / d2 * E)
    return br, bz
