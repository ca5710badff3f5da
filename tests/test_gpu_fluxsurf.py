"""GPU parity of NEXT-2: flux-surface post-processing (ptefit_flux_surfaces) against
oracle/fluxsurf.py on the same flux map and search state (Eq. 12)."""
import numpy as np
import pytest

from oracle import fluxsurf as FS, search as OS
from oracle.picard import reconstruct
from tests.helpers import cached_case, oracle_device, round_inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,precision,ns", [("cfg1", "fp64", 2), ("cfg3", "fp32", 2), ("cfg4", "fp32", 6)])
def test_flux_surfaces_against_oracle(name, precision, ns):
    import torch
    import paper_2601_12378_b200 as P
    dev, sl = cached_case(name, ns)
    dv, b, ic = round_inputs(dev, sl, precision)
    od = oracle_device(dv)
    n_iter = dev["meta"]["cfg"]["n_iter"]
    rec = P.Reconstructor(dev, precision=precision, max_batch=ns)
    rec.reconstruct(torch.tensor(b, dtype=rec.dtype, device="cuda"), torch.tensor(ic, dtype=rec.dtype, device="cuda"), n_iter)
    n_prof, n_chord, munu, f_vac = 33, 128, ((-1, -1), (-1, -2), (0, 0), (1, 1)), 2.5e6
    out = rec.flux_surfaces(ns, n_prof=n_prof, n_chord=n_chord, n_bisect=10, munu=munu, f_vac=f_vac)
    torch.cuda.synchronize()
    psi = rec.psi.cpu().numpy().astype(np.float64)
    X = rec.coeffs.cpu().numpy().astype(np.float64)
    tol = 2e-5 if precision == "fp32" else 1e-9
    for q in range(ns):
        assert int(rec.status[q]) == 0 and int(out["status"][q]) == 0
        # the oracle post-processes the flux map the GPU returned, with the search state of that same map
        sr = OS.search(psi[q], od.r, od.z, od.lim_mask, od.xpt_mask, od.lim_r, od.lim_z, od.s)
        o = FS.flux_surfaces(psi[q], sr["psin"], sr["mask"], od.r, od.z, sr["axis"][2], sr["axis"][3], sr["axis"][4], sr["psi_b"],
                             n_prof=n_prof, n_chord=n_chord, n_bisect=10, munu=munu, f_vac=f_vac,
                             Xff=X[q][od.n_p:od.n_p + od.n_ff], n_ff=od.n_ff)
        v = out["vert"][q].cpu().numpy().astype(np.float64)
        dv_ = np.hypot(v[..., 0] - o["vert"][..., 0], v[..., 1] - o["vert"][..., 1])
        # vertices: same bisection on (nearly) the same field; FP32 psi_N differs by ~1e-7, i.e. << 1 mm
        assert np.max(dv_) <= (2e-5 if precision == "fp32" else 1e-10), (q, np.max(dv_))
        Q = out["Q"][q].cpu().numpy().astype(np.float64)
        assert np.max(np.abs(Q / o["Q"] - 1)) <= 50 * tol, (q, np.max(np.abs(Q / o["Q"] - 1)))
        qq = out["q"][q].cpu().numpy().astype(np.float64)
        assert np.max(np.abs(qq / o["q"] - 1)) <= 50 * tol
        g = out["geom"][q].cpu().numpy().astype(np.float64)
        assert np.max(np.abs(g - o["geom"])) <= 10 * tol
        assert np.all(np.isfinite(o["q"])) and o["geom"][5] > 1.0          # elongated plasmas in every config
    rec.close()
