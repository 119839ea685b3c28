"""CPU-side checks of the boundary: the shared library builds, loads, and exports every symbol include/imager.h
declares; the binding's struct matches the header; no compute call is made (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2206_15117_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "imager.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(imager_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_functions()
    assert {"imager_plan_create", "imager_grid", "imager_degrid", "imager_plan_destroy"} <= set(names)
    for name in names:
        assert getattr(lib, name) is not None, name
    from paper_2206_15117_b200 import EXPORTS
    assert sorted(EXPORTS) == names


def test_params_struct_matches_header(lib):
    from paper_2206_15117_b200.binding import ImagerParams
    text = open(os.path.join(ROOT, "include", "imager.h")).read()
    body = re.search(r"typedef struct imager_params \{(.*?)\} imager_params;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [re.sub(r"\[\d+\]", "", d.split()[-1].lstrip("*")) for d in body.split(";") if d.strip()]
    assert fields == [f[0] for f in ImagerParams._fields_]
    assert ctypes.sizeof(ImagerParams) == 40 + 9 * 8 + 4 * 8 + 8


def test_calls_fail_loudly_without_gpu(lib):
    """No CPU fallback: on a box without CUDA, plan creation must fail with IMAGER_ERR_CUDA, not compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2206_15117_b200.binding import ImagerParams
    p = ImagerParams(grid_size=64, n_corr=1, n_pol=1, n_wplanes=1, support_min=1, support_max=1, oversample=1,
                     n_aplanes=1, kernel_mode=0, cell_size_rad=1e-3, max_nvis=16)
    h = ctypes.c_void_p()
    rc = lib.imager_plan_create(ctypes.byref(p), None, ctypes.byref(h))
    assert rc == -4 and b"no CUDA device" in lib.imager_last_error()
    bad = ImagerParams(grid_size=63)
    assert lib.imager_plan_create(ctypes.byref(bad), None, ctypes.byref(h)) == -1
    assert lib.imager_plan_destroy(None) == 0
