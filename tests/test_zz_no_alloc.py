"""GPU: ptefit_gs_solve_noalloc (include/ptefit.h) -- the Delta* solve whose workspace is the library's
file-scope static device array -- against the existing path (ptefit_debug_gs_solve, handle workspaces) on the
same inputs, two calls in a row that share the array, plus the size limit and the handle-kind checks.

Collected last on purpose (the name sorts after every other test file): the suite runs with pytest -x.
The test passes alone in a fresh process (the first call resolves the symbol address) and after the other tests.
"""
import numpy as np
import pytest

from tests.helpers import PSI_TOL, oracle_device, psi_rel_err

pytestmark = pytest.mark.gpu


def _inputs(od, B, seed):
    rng = np.random.default_rng(seed)
    N = od.nr * od.nz
    I = rng.uniform(0.0, 40.0, (B, N)) * od.lim_mask.ravel()[None, :]
    pbd = rng.uniform(-0.05, 0.05, (B, len(od.bnd)))
    return I, pbd


@pytest.mark.parametrize("name,B1,B2", [("cfg2", 8, 3), ("cfg3", 4, 2)])
def test_gs_solve_noalloc_matches_existing_path_two_calls(name, B1, B2):
    """Two calls in a row with different inputs and different batch sizes (the second, smaller call runs on an
    array still holding the first call's values): each equals the existing path within the FP64 flux tolerance
    of the parity tests, edge nodes bit-exact, and both satisfy the oracle's discrete operator."""
    import torch
    import synth
    import paper_2601_12378_b200 as P
    from oracle.gs_solve import MU0
    dev = synth.make_device(name)
    synth.make_slices(dev, 1)                        # fills sigma
    od = oracle_device(dev)
    rec = P.Reconstructor(dev, precision="fp64", max_batch=max(B1, B2))
    a_inf = 2.0 * (2.0 / od.op.dr ** 2 + 2.0 / od.op.dz ** 2)
    for call, (B, seed) in enumerate(((B1, 5), (B2, 6))):
        I, pbd = _inputs(od, B, seed)
        dI, dp = torch.tensor(I, device="cuda"), torch.tensor(pbd, device="cuda")
        ref = torch.zeros(B, od.nz, od.nr, dtype=torch.float64, device="cuda")
        out = torch.full((B, od.nz, od.nr), float("nan"), dtype=torch.float64, device="cuda")
        rec.debug_gs_solve(dI, dp, ref)
        rec.gs_solve_noalloc(dI, dp, out)
        torch.cuda.synchronize()
        r, o = ref.cpu().numpy(), out.cpu().numpy()
        assert np.all(np.isfinite(o)), (name, call)
        for q in range(B):
            assert psi_rel_err(o[q], r[q]) <= PSI_TOL["fp64"], (name, call, q, psi_rel_err(o[q], r[q]))
            assert np.array_equal(o[q].ravel()[od.bnd], pbd[q])
            rhs = -MU0 * od.r[None, 1:-1] * I[q].reshape(od.nz, od.nr)[1:-1, 1:-1] / od.dA
            res = od.op.apply(o[q]) - rhs
            assert np.max(np.abs(res)) <= a_inf * 2e-13 * np.max(np.abs(o[q])), (name, call, q)
    rec.close()


def test_gs_solve_noalloc_limits():
    """Sizes beyond the static array and handles of the wrong kind are rejected with a clear error, and a call
    after a rejected one still works."""
    import torch
    import synth
    import paper_2601_12378_b200 as P
    from paper_2601_12378_b200.binding import NOALLOC_SCRATCH_BYTES
    dev = synth.make_device("cfg2")
    synth.make_slices(dev, 1)
    od = oracle_device(dev)
    nri, nzi = od.nr - 2, od.nz - 2
    per_slice = nri * (3 * ((nzi + 1) & ~1) + nzi) * 8
    Bmax = NOALLOC_SCRATCH_BYTES // per_slice
    rec = P.Reconstructor(dev, precision="fp64", max_batch=Bmax + 1)
    I, pbd = _inputs(od, Bmax + 1, 9)
    dI, dp = torch.tensor(I, device="cuda"), torch.tensor(pbd, device="cuda")
    out = torch.zeros(Bmax + 1, od.nz, od.nr, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PtefitError, match="scratch"):
        rec.gs_solve_noalloc(dI, dp, out)
    # the largest batch that fits, against the existing path
    ref = torch.zeros(Bmax, od.nz, od.nr, dtype=torch.float64, device="cuda")
    rec.debug_gs_solve(dI[:Bmax], dp[:Bmax], ref)
    rec.gs_solve_noalloc(dI[:Bmax], dp[:Bmax], out[:Bmax])
    torch.cuda.synchronize()
    r, o = ref.cpu().numpy(), out[:Bmax].cpu().numpy()
    assert max(psi_rel_err(o[q], r[q]) for q in range(Bmax)) <= PSI_TOL["fp64"]
    rec.close()
    rec32 = P.Reconstructor(dev, precision="fp32", max_batch=2)
    with pytest.raises(P.PtefitError, match="FP64"):
        rec32.gs_solve_noalloc(dI[:2].float(), dp[:2].float(), out[:2])
    rec32.close()
