"""CPU-side checks of the product boundary: the C-ABI library builds, loads, exports every
symbol include/tnlm.h declares, validates arguments, and fails loudly without a CUDA device.
No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tn():
    from paper_1009_1351_b200 import build
    build.build()
    import paper_1009_1351_b200 as tn
    return tn


def test_every_declared_symbol_is_exported(tn):
    header = open(os.path.join(ROOT, "include", "tnlm.h")).read()
    declared = sorted(set(re.findall(r"\b(tnlm_[a-z_]+)\s*\(", header)))
    assert len(declared) >= 12
    lib = C.CDLL(tn.lib_path())
    for name in declared:
        assert hasattr(lib, name), name
    from paper_1009_1351_b200 import binding
    assert sorted(binding.EXPORTS) == declared
    assert "sm_100a" in tn.version()


def test_argument_validation_happens_before_any_device_work(tn):
    import numpy as np
    bad = [dict(nx=0), dict(window=4), dict(patch=2), dict(h=0.0), dict(h=float("nan")), dict(h=1e-20), dict(mu=-0.1),
           dict(n_phase=0)]
    base = dict(nx=8, ny=8, n_phase=3, window=5, patch=3, h=0.01, mu=0.1)
    for b in bad:
        kw = dict(base, **b)
        with pytest.raises(tn.TnlmError) as ei:
            tn.create(None, kw["nx"], kw["ny"], kw["n_phase"], kw["window"], kw["patch"], kw["h"], kw["mu"])
        assert ei.value.code == 1, b
    with pytest.raises(tn.TnlmError) as ei:
        tn.create(None, 8, 8, 3, 33, 3, 0.01, 0.1)
    assert ei.value.code == 4
    ang = np.zeros((3, 4))
    for g in (tn.Geometry(4, 8, 50.0, 40.0, 1.0, ang),            # sid >= sdd
              tn.Geometry(4, 8, 5.0, 40.0, 1.0, ang),             # image corner outside source circle
              tn.Geometry(0, 8, 50.0, 90.0, 1.0, np.zeros((3, 0)))):
        with pytest.raises(tn.TnlmError) as ei:
            tn.create(g, 8, 8, 3, 5, 3, 0.01, 0.1)
        assert ei.value.code == 1
    with pytest.raises(tn.TnlmError) as ei:
        tn.create(tn.Geometry(4, 8, 50.0, 90.0, 1.0, ang, detector_arc=0), 8, 8, 3, 5, 3, 0.01, 0.1)
    assert ei.value.code == 4


def test_no_cpu_fallback_without_a_device(tn):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(tn.TnlmError) as ei:
        tn.create(None, 8, 8, 3, 5, 3, 0.01, 0.1)
    assert ei.value.code == 2          # TNLM_CUDA_ERROR, not a silent CPU path


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1009_1351_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), os.path.join(dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1009_1351_b200" not in src and "libtnlm" not in src
