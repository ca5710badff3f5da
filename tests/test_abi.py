"""CPU: the C-ABI library loads and exports every symbol include/ptefit.h declares, and the
product path fails loudly without a GPU (no fallback)."""
import os
import re

import pytest

import paper_2601_12378_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    P.build if hasattr(P, "build") else None
    from paper_2601_12378_b200 import build as B
    B.build()
    hdr = open(os.path.join(ROOT, "include", "ptefit.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(ptefit_[a-z0-9_]+)\s*\(", hdr)))
    assert "ptefit_create" in declared and "ptefit_reconstruct" in declared and "ptefit_destroy" in declared
    lib = P.load_library()
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(P.EXPORTED_SYMBOLS) == declared


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import synth
    d = synth.make_device("cfg1")
    synth.make_slices(d, 1)
    with pytest.raises(P.PtefitError):
        P.Reconstructor(d)
    # the raw C entry point also refuses
    with pytest.raises(P.PtefitError):
        P.ptefit_create(d["grid"], d["geom"], d["tables"], P.poly_terms(2, 2, True), 0.01, 0.6, 1, 0, 1)


def test_product_does_not_import_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2601_12378_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inc", ".h")):
                src = open(os.path.join(root, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "synth")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "synth", f)).read()
            assert "import oracle" not in src and "from oracle" not in src and "paper_2601_12378_b200" not in src.replace('``paper_2601_12378_b200``', ''), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2601_12378_b200" not in src and "from paper_2601_12378_b200" not in src, f


def _create_status(d, terms=None, **over):
    """Call the raw C entry point with overrides; returns (status, error string).  Validation happens
    before any device is touched, so this runs without a GPU."""
    import ctypes as C
    import numpy as np
    from paper_2601_12378_b200 import binding as Bd
    lib = P.load_library()
    grid = dict(d["grid"], **{k: v for k, v in over.items() if k in d["grid"]})
    geom = dict(d["geom"], **{k: v for k, v in over.items() if k in ("ip_sign", "cold_a", "n_coil")})
    keep = dict(sigma=np.ascontiguousarray(over.get("sigma", geom["sigma"]), np.float64),
                lim_r=np.ascontiguousarray(geom["lim_r"], np.float64), lim_z=np.ascontiguousarray(geom["lim_z"], np.float64),
                lim_mask=np.ascontiguousarray(over.get("lim_mask", geom["lim_mask"]), np.uint8).ravel(),
                gp=np.ascontiguousarray(d["tables"]["gp"]), gc=np.ascontiguousarray(d["tables"]["gc"]),
                gb=np.ascontiguousarray(d["tables"]["gb"]), ggc=np.ascontiguousarray(d["tables"]["ggc"]))
    g = Bd._Grid(int(grid["nr"]), int(grid["nz"]), grid["rmin"], grid["rmax"], grid["zmin"], grid["zmax"])
    ge = Bd._Geometry(int(geom["n_meas"]), int(geom["n_coil"]), Bd._ptr(keep["sigma"]), len(keep["lim_r"]), Bd._ptr(keep["lim_r"]),
                      Bd._ptr(keep["lim_z"]), Bd._ptr(keep["lim_mask"]), None, int(geom.get("ip_sign", 1)), geom["cold_rc"],
                      geom["cold_zc"], geom["cold_a"], geom["cold_b"])
    tb = Bd._Tables(Bd._ptr(keep["gp"]), Bd._ptr(keep["gc"]), Bd._ptr(keep["gb"]), Bd._ptr(keep["ggc"]))
    terms = terms if terms is not None else P.poly_terms(2, 2, True)
    kk = []
    tarr = (Bd._Term * len(terms))(*[Bd._term_struct(t, kk) for t in terms])
    ba = Bd._Basis(len(terms), tarr, float(over.get("lambda_reg", 0.01)), float(over.get("relax", 0.6)),
                   int(over.get("lsq_method", 0)), int(over.get("fit_coils", 0)), None)
    op = Bd._Options(int(over.get("precision", 1)), int(over.get("gemm", 0)), int(over.get("max_batch", 1)),
                     int(over.get("flags", 0)), 0)
    h = C.c_void_p()
    st = lib.ptefit_create(C.byref(g), C.byref(ge), C.byref(tb), C.byref(ba), C.byref(op), C.byref(h))
    msg = lib.ptefit_global_error().decode()
    if st == 0:
        lib.ptefit_destroy(h)
    return st, msg


def test_create_validates_arguments_on_the_host():
    """include/ptefit.h error behaviour: argument errors are reported as PTEFIT_ERR_INVALID_ARG (1) /
    PTEFIT_ERR_UNSUPPORTED (2) with a message, before any CUDA call."""
    import numpy as np
    import synth
    d = synth.make_device("cfg1")
    synth.make_slices(d, 1)
    INVALID, UNSUPPORTED = 1, 2
    assert _create_status(d, nz=34)[0] == INVALID                       # nz-1 not a power of two
    assert _create_status(d, rmin=0.0)[0] == INVALID                    # R must be > 0
    assert _create_status(d, ip_sign=0)[0] == INVALID
    assert _create_status(d, cold_a=0.0)[0] == INVALID
    assert _create_status(d, relax=0.0)[0] == INVALID and _create_status(d, relax=1.5)[0] == INVALID
    assert _create_status(d, lambda_reg=-1.0)[0] == INVALID
    assert _create_status(d, max_batch=0)[0] == INVALID
    bad_sigma = np.array(d["geom"]["sigma"], np.float64).copy(); bad_sigma[3] = 0.0
    assert _create_status(d, sigma=bad_sigma)[0] == INVALID
    edge_mask = np.array(d["geom"]["lim_mask"], np.uint8).copy(); edge_mask[0, 5] = 1
    st, msg = _create_status(d, lim_mask=edge_mask)
    assert st == INVALID and "edge" in msg
    assert _create_status(d, terms=[(0, 0, 2), (2, 0, 0), (1, 0, 2)])[0] == INVALID     # delz term must be last
    assert _create_status(d, terms=[(0, 2, 2)])[0] == INVALID                           # needs i < N
    assert _create_status(d, terms=[(5, 0, 2)])[0] == UNSUPPORTED                       # unknown kind
    assert _create_status(d, terms=[(2, 0, 0)])[0] == INVALID                           # no P'/FF' term at all
    kn = np.linspace(0.7, 1.0, 7)
    assert _create_status(d, terms=[(0, 0, 1), (1, 9, 0, 1, kn, 10.0)])[0] == INVALID     # cardinal index out of range
    assert _create_status(d, terms=[(0, 0, 1), (1, 2, 0, 1, kn[::-1], 10.0)])[0] == INVALID   # knots must increase
    assert _create_status(d, terms=[(0, 0, 1), (1, 2, 0, 1, kn, 0.0)])[0] == INVALID      # tension > 0
    assert _create_status(d, terms=[(0, 0, 1), (1, 2, 0, 1, kn, 10.0), (1, 3, 0, 1, kn, 5.0)])[0] == UNSUPPORTED   # one tension only
    assert _create_status(d, gemm=1)[0] == INVALID                                       # reserved single-pass TF32 mode
    assert _create_status(d, flags=64)[0] == INVALID
    assert _create_status(d, lsq_method=2)[0] == INVALID
    assert _create_status(d, fit_coils=1)[0] == INVALID                                  # needs sigma_ic
