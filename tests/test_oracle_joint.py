"""Pins of the oracle's joint coil-current fit, Eq. 7 (oracle/lsq.py fit_joint).
The paper prints no worked example; the pins are limits and identities the mathematics fixes."""
import numpy as np
import pytest

from oracle import lsq as L


def _problem(seed=3, M=60, nb=4, nc=8):
    rng = np.random.default_rng(seed)
    resp = rng.normal(size=(M, nb)) * np.array([1.0, 3.0, 0.2, 5.0])[:nb]
    gc = rng.normal(size=(M, nc)) * 0.5
    sigma = rng.uniform(0.5, 2.0, M) * 1e-2
    xt = rng.uniform(0.5, 1.5, nb)
    ict = rng.uniform(-2.0, 2.0, nc)
    return rng, resp, gc, sigma, xt, ict


def test_tight_coil_rows_reduce_to_fixed_currents():
    """sigma_ic -> 0 pins I_C' to the measured currents: Eq. 7 becomes Eq. 6 with d = b - G_C I_C."""
    rng, resp, gc, sigma, xt, ict = _problem()
    b = resp @ xt + gc @ ict + sigma * rng.normal(size=len(sigma))
    X0, c0, st0 = L.fit(resp, b - gc @ ict, sigma, 0.01)
    X, icf, c, st = L.fit_joint(resp, gc, b, ict, sigma, np.full(len(ict), 1e-9), 0.01)
    assert st == st0 == 0
    assert np.max(np.abs(X / X0 - 1)) < 1e-7 and np.max(np.abs(icf - ict)) < 1e-9
    assert abs(c / c0 - 1) < 1e-6


def test_exact_data_recover_coefficients_and_currents():
    """Exact b from (X_t, I_C,t), measured currents off by 5 % with loose sigma_ic, lambda = 0: the joint
    fit returns the true currents, not the measured ones."""
    rng, resp, gc, sigma, xt, ict = _problem(seed=4)
    b = resp @ xt + gc @ ict
    meas = ict * (1 + 0.05 * rng.normal(size=len(ict)))
    X, icf, c, st = L.fit_joint(resp, gc, b, meas, sigma, np.full(len(ict), 1e4), 0.0)
    assert st == 0
    assert np.max(np.abs(X / xt - 1)) < 1e-8 and np.max(np.abs(icf - ict)) < 1e-8 and c < 1e-12


def test_stationarity_of_the_objective():
    """Gradient of |W(R X + G_C I' - b)|^2 + |(I' - I_C)/sigma_ic|^2 + lam^2 M sum (s_l X_l)^2 vanishes."""
    rng, resp, gc, sigma, xt, ict = _problem(seed=5)
    b = resp @ xt + gc @ ict + sigma * rng.normal(size=len(sigma))
    sic = rng.uniform(0.01, 0.2, len(ict))
    meas = ict + sic * rng.normal(size=len(ict))
    lam = 0.02
    X, icf, c, st = L.fit_joint(resp, gc, b, meas, sigma, sic, lam)
    A1, A2 = resp / sigma[:, None], gc / sigma[:, None]
    r = A1 @ X + A2 @ icf - b / sigma
    s = np.sqrt(np.sum(A1 * A1, axis=0))
    gX = A1.T @ r + lam ** 2 * len(sigma) * s ** 2 * X
    gI = A2.T @ r + (icf - meas) / sic ** 2
    scale = np.max(np.abs(A1.T @ (b / sigma)))
    assert np.max(np.abs(gX)) < 1e-9 * scale and np.max(np.abs(gI)) < 1e-9 * max(scale, np.max(np.abs(meas / sic ** 2)))
    assert abs(c - r @ r) < 1e-9 * c


def test_block_matrix_of_eq7_by_dense_lstsq():
    """lambda = 0: the solution equals the dense least squares of Eq. 7's block system
    [[R, G_C], [0, I]] [X; I'] = [b; I_C] with rows weighted 1/sigma and 1/sigma_ic."""
    rng, resp, gc, sigma, xt, ict = _problem(seed=6)
    b = resp @ xt + gc @ ict + sigma * rng.normal(size=len(sigma))
    sic = rng.uniform(0.01, 0.2, len(ict))
    meas = ict + sic * rng.normal(size=len(ict))
    nb, nc = resp.shape[1], gc.shape[1]
    blk = np.block([[resp / sigma[:, None], gc / sigma[:, None]], [np.zeros((nc, nb)), np.diag(1 / sic)]])
    sol = np.linalg.lstsq(blk, np.concatenate([b / sigma, meas / sic]), rcond=None)[0]
    X, icf, c, st = L.fit_joint(resp, gc, b, meas, sigma, sic, 0.0)
    assert np.max(np.abs(X - sol[:nb])) < 1e-9 * np.max(np.abs(sol[:nb])) and np.max(np.abs(icf - sol[nb:])) < 1e-9 * np.max(np.abs(sol[nb:]))


def test_status_codes():
    rng, resp, gc, sigma, xt, ict = _problem()
    b = resp @ xt
    assert L.fit_joint(resp * np.nan, gc, b, ict, sigma, np.ones(len(ict)), 0.0)[3] == 2
    assert L.fit_joint(resp * 0.0, gc, b, ict, sigma, np.ones(len(ict)), 0.0)[3] == 3


def test_picard_with_joint_fit_corrects_a_biased_coil_current(dev_cfg1):
    """Whole loop on config 1 with one measured PF current off by 10 %: the joint fit moves that current
    back towards the value the measurements were generated with, and fits better than Eq. 6."""
    from oracle.picard import Device, reconstruct
    d, s = dev_cfg1
    ic_true = s["ic"][0]
    meas = ic_true.copy()
    k = int(np.argmax(np.abs(ic_true)))
    meas[k] *= 1.10
    sic = np.full(len(ic_true), 0.05 * np.max(np.abs(ic_true)))
    dj = dict(d); dj["basis"] = dict(d["basis"], fit_coils=1, sigma_ic=sic)
    o0 = reconstruct(Device(d["grid"], d["geom"], d["tables"], d["basis"]), s["b"][0], meas, 10)
    oj = reconstruct(Device(dj["grid"], dj["geom"], dj["tables"], dj["basis"]), s["b"][0], meas, 10)
    assert oj["status"] == 0
    assert abs(oj["ic_fit"][k] - ic_true[k]) < 0.5 * abs(meas[k] - ic_true[k])
    assert oj["chi2"] < o0["chi2"]
