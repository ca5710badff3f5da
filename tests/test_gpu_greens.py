"""GPU parity of NEXT-3: Green's tables computed by ptefit_greens_table against the
oracle's closed forms (oracle/greens.py, own AGM; pinned in tests/test_oracle_greens.py) and against
the scipy-tabulated input tables of a config."""
import numpy as np
import pytest

from oracle import greens as OG

pytestmark = pytest.mark.gpu


def _t(a):
    import torch
    return torch.tensor(np.ascontiguousarray(a, np.float64), dtype=torch.float64, device="cuda")


def test_greens_pairs_against_oracle():
    import torch
    import paper_2601_12378_b200 as P
    rng = np.random.default_rng(5)
    ns, nf = 301, 77                                     # ragged against the 256-thread blocks
    sr, sz = rng.uniform(0.05, 1.8, ns), rng.uniform(-1.7, 1.7, ns)
    fr, fz = rng.uniform(0.05, 1.8, nf), rng.uniform(-3.0, 3.0, nf)
    w = rng.integers(1, 33, ns).astype(np.float64)
    al = rng.uniform(0, 2 * np.pi, nf)
    out = torch.zeros(nf, ns, dtype=torch.float64, device="cuda")
    # flux rows
    P.ptefit_greens_table(_t(fr), _t(fz), _t(sr), _t(sz), out, d_src_w=_t(w))
    ref = OG.psi_filament(sr[None, :], sz[None, :], fr[:, None], fz[:, None]) * w[None, :]
    assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-13 * np.max(np.abs(ref))
    # probe rows, transposed store, no weights
    outT = torch.zeros(ns, nf, dtype=torch.float64, device="cuda")
    P.ptefit_greens_table(_t(fr), _t(fz), _t(sr), _t(sz), outT, d_fld_cos=_t(np.cos(al)), d_fld_sin=_t(np.sin(al)), transpose=True)
    br, bz = OG.b_filament(sr[None, :], sz[None, :], fr[:, None], fz[:, None])
    ref = np.cos(al)[:, None] * br + np.sin(al)[:, None] * bz
    assert np.max(np.abs(outT.cpu().numpy().T - ref)) <= 1e-13 * np.max(np.abs(ref))
    # the survey's golden values (tests/golden/greens_golden.txt): (a, z_s, rho, z_f) = (1, 0, 0.5, 0.2)
    one = torch.zeros(1, 1, dtype=torch.float64, device="cuda")
    P.ptefit_greens_table(_t([0.5]), _t([0.2]), _t([1.0]), _t([0.0]), one)
    assert abs(float(one[0, 0]) / 7.994041539299143e-08 - 1) < 1e-13
    P.ptefit_greens_table(_t([0.5]), _t([0.2]), _t([1.0]), _t([0.0]), one, d_fld_cos=_t([1.0]), d_fld_sin=_t([0.0]))
    assert abs(float(one[0, 0]) / 1.343142703162336e-07 - 1) < 1e-12
    P.ptefit_greens_table(_t([0.5]), _t([0.2]), _t([1.0]), _t([0.0]), one, d_fld_cos=_t([0.0]), d_fld_sin=_t([1.0]))
    assert abs(float(one[0, 0]) / 6.904221985351053e-07 - 1) < 1e-12
    # coincident points: 0, not Inf
    P.ptefit_greens_table(_t([0.7]), _t([0.1]), _t([0.7]), _t([0.1]), one)
    assert float(one[0, 0]) == 0.0


def test_config_tables_on_gpu():
    """All four input tables of config 2 (gp, gc, gb, ggc) regenerated on the GPU equal the scipy
    tabulation the configs use (synth.make_tables), interior-node columns."""
    import torch
    import synth
    import paper_2601_12378_b200 as P
    dev = synth.make_device("cfg2")
    m, g, tb = dev["meta"], dev["grid"], dev["tables"]
    nr, nz = g["nr"], g["nz"]
    R2, Z2 = np.meshgrid(m["r"], m["z"])
    rn, zn = R2.ravel(), Z2.ravel()
    npb = m["n_probe"]
    M = len(m["sen_r"])
    ca = np.concatenate([np.cos(m["alpha"]), np.zeros(M - npb)]); sa = np.concatenate([np.sin(m["alpha"]), np.zeros(M - npb)])
    interior = np.zeros((nz, nr), bool); interior[1:-1, 1:-1] = True
    interior = interior.ravel()
    gp = torch.zeros(M, nr * nz, dtype=torch.float64, device="cuda")
    P.ptefit_greens_table(_t(m["sen_r"]), _t(m["sen_z"]), _t(rn), _t(zn), gp, d_fld_cos=_t(ca), d_fld_sin=_t(sa))
    a = gp.cpu().numpy()[:, interior]; b = tb["gp"][:, interior]
    assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b))
    gc = torch.zeros(M, len(m["src_r"]), dtype=torch.float64, device="cuda")
    P.ptefit_greens_table(_t(m["sen_r"]), _t(m["sen_z"]), _t(m["src_r"]), _t(m["src_z"]), gc, d_fld_cos=_t(ca), d_fld_sin=_t(sa), d_src_w=_t(m["src_w"]))
    assert np.max(np.abs(gc.cpu().numpy() - tb["gc"])) <= 1e-12 * np.max(np.abs(tb["gc"]))
    from oracle.gs_solve import boundary_nodes
    bnd = boundary_nodes(nr, nz)
    gb = torch.zeros(len(bnd), nr * nz, dtype=torch.float64, device="cuda")
    P.ptefit_greens_table(_t(rn[bnd]), _t(zn[bnd]), _t(rn), _t(zn), gb)
    a = gb.cpu().numpy()[:, interior]; b = tb["gb"][:, interior]
    assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b))
    ggc = torch.zeros(nr * nz, len(m["src_r"]), dtype=torch.float64, device="cuda")
    P.ptefit_greens_table(_t(rn), _t(zn), _t(m["src_r"]), _t(m["src_z"]), ggc, d_src_w=_t(m["src_w"]))
    assert np.max(np.abs(ggc.cpu().numpy() - tb["ggc"])) <= 1e-12 * np.max(np.abs(tb["ggc"]))
