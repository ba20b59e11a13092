"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/nf.h declares (no compute calls without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2405_14903_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "nf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nf_[a-z_A-Z0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for must in ("nf_grid_create", "nf_set_solid", "nf_project", "nf_project_adjoint", "nf_advect"):
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_binding_covers_every_declared_symbol(lib_path):
    from paper_2405_14903_b200 import api
    assert sorted(api.EXPORTED_SYMBOLS) == _declared_symbols()
    lib = api.load_library()
    assert lib.nf_version().decode().startswith("nf-b200")


def test_null_handle_is_rejected_without_a_gpu(lib_path):
    from paper_2405_14903_b200 import api
    lib = api.load_library()
    assert lib.nf_set_dt_rho(None, 1.0) == api.NF_ERR_INVALID
    assert lib.nf_project(None, None, None, None, None, 1e-6, 10) == api.NF_ERR_INVALID
    assert lib.nf_launch_count(None) == 0
    assert lib.nf_geom_sdf(None, None, 1, 4, 8, 0, None) == api.NF_ERR_INVALID
    assert lib.nf_geom_csg(None, 0, None, None, None) == api.NF_ERR_INVALID
    assert lib.nf_geom_velocity_adjoint(None, None, 1, 4, 8, 1.0, None, None, None, None) == api.NF_ERR_INVALID


def test_no_cpu_fallback_in_binding():
    import torch
    from paper_2405_14903_b200 import api
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        api.Grid(8, 8, 8, 0.125)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2405_14903_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
