"""CPU-side checks of the boundary: the library builds for sm_100a, loads, and exports every symbol the
header declares (no compute call is made here - there is no GPU on the build box)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mwa_grid.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mwa_(?:grid|image)_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_0902_0915_b200 import _build
    lib_path = _build.build()
    assert os.path.exists(lib_path)
    lib = ctypes.CDLL(lib_path)
    names = _declared_symbols()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), n


def test_binding_names_match_header():
    import paper_0902_0915_b200 as m
    assert sorted(m.EXPORTS) == _declared_symbols()
    for n in m.EXPORTS:
        assert callable(getattr(m, n)), n


def test_plan_create_reports_errors_without_a_gpu_or_with_bad_arguments():
    import pytest
    import paper_0902_0915_b200 as m
    from gen import make_kernel_table
    with pytest.raises(m.MwaGridError) as e:
        m.mwa_grid_plan_create(63, 1.0, 7, 8, make_kernel_table(7, 8))     # odd grid: rejected before any CUDA call
    assert "grid_n" in str(e.value)
    assert m.mwa_grid_last_error() != ""


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_0902_0915_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src, f


def test_noalloc_limits_in_the_binding_match_the_header():
    import paper_0902_0915_b200 as m
    text = open(os.path.join(ROOT, "include", "mwa_grid.h")).read()
    lim = {k: int(v) for k, v in re.findall(r"#define\s+MWA_GRID_NOALLOC_(MAX_[A-Z_]+)\s+(\d+)", text)}
    assert lim == {"MAX_VIS": m.NOALLOC_MAX_VIS, "MAX_CHAN": m.NOALLOC_MAX_CHAN, "MAX_GRID_N": m.NOALLOC_MAX_GRID_N}
