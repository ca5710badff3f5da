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
