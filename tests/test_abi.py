"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/idg_b200.h declares (no compute calls without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_1909_07226_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "idg_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(idg_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for required in ("idg_plan_create", "idg_grid", "idg_degrid", "idg_gridder", "idg_subgrid_fft",
                     "idg_adder", "idg_splitter", "idg_degridder", "idg_grid_host", "idg_degrid_host"):
        assert required in names


def test_library_exports_every_declared_symbol(built_lib):
    lib = ctypes.CDLL(built_lib)
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_symbols(built_lib):
    from paper_1909_07226_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()
    lib = binding.lib()
    assert lib.idg_strerror(0) == b"ok"
    assert b"16, 24, 32 or 48" in lib.idg_strerror(-5)
    assert binding.META_DTYPE.itemsize == 48 and ctypes.sizeof(binding.PlanParams) == 48


def test_argument_errors_without_a_device(built_lib):
    """NULL / bad-parameter paths return error codes before touching CUDA."""
    from paper_1909_07226_b200 import binding
    lib = binding.lib()
    h = ctypes.c_void_p()
    assert lib.idg_plan_create(ctypes.byref(h), None, None, None, None, 1, 1, 1, 1, None) == -1
    assert lib.idg_plan_size(None, None, None, None) == -1
    assert lib.idg_grid(None, None, None, None, None, None, None) == -1
    assert lib.idg_subgrid_fft(None, None, 1, None) == -1
    lib.idg_plan_destroy(None)                                  # must be a no-op


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1909_07226_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "idg_oracle" not in src and "from oracle" not in src and "import oracle" not in src, f


def test_binding_constants_match_the_header():
    """Limits and flags that the Python binding repeats are the header's."""
    from paper_1909_07226_b200 import binding, synth
    text = open(os.path.join(ROOT, "include", "idg_b200.h")).read()
    defs = dict(re.findall(r"#define\s+(IDG_[A-Z_0-9]+)\s+(\d+)", text))
    assert int(defs["IDG_IMAGE_TAPER_STATIC_MAX_LN"]) == binding.IMAGE_TAPER_STATIC_MAX_LN
    assert int(defs["IDG_PLAN_FORCE_BLOCKS"]) == synth.FLAG_FORCE_BLOCKS
    assert int(defs["IDG_PLAN_SPAN_ATERMS"]) == synth.FLAG_SPAN_ATERMS
    assert int(defs["IDG_PLAN_FP32_GRIDDER"]) == synth.FLAG_FP32_GRIDDER
