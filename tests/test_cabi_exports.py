"""CPU: the C-ABI library builds for sm_100a, loads without a GPU, and exports every symbol
include/sldg.h declares (no compute calls here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "sldg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sldg_[a-z_0-9A-Z]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = _declared_functions()
    for required in ("sldg_create", "sldg_set_initial", "sldg_advect", "sldg_compute_rho",
                     "sldg_poisson_E", "sldg_step", "sldg_diagnostics", "sldg_translate"):
        assert required in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1907_08316_b200 import build
    lib = ctypes.CDLL(build.build())
    for name in _declared_functions():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_names():
    from paper_1907_08316_b200 import sldg
    assert sorted(sldg.EXPORTS) == _declared_functions()


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1907_08316_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src, fn
                assert "sldg_oracle" not in src, fn


def test_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        return
    import pytest
    from paper_1907_08316_b200.sldg import Sldg, SldgError
    with pytest.raises(SldgError):
        Sldg(1, 1, (4, 4), 2, (0.0, 0.0), (1.0, 1.0))
