"""The C-ABI library loads and exports every symbol include/rick.h declares (no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "rick.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rick_[a-z_]+)\s*\(", src)))


def test_header_declares_north_star_calls():
    names = _declared()
    for n in ["rick_plan", "rick_grid", "rick_fft_wplanes", "rick_wcorrect_accumulate",
              "rick_gridcorrect", "rick_image"]:
        assert n in names


def test_library_exports_every_declared_symbol():
    from paper_2601_19714_b200 import build, rick
    build.build()
    lib = ctypes.CDLL(rick.LIB_PATH)
    for n in _declared():
        assert hasattr(lib, n), n
    assert sorted(rick.EXPORTS) == _declared()
    lib.rick_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.rick_version()


def test_binding_has_same_names():
    from paper_2601_19714_b200 import rick
    for n in ["rick_grid", "rick_fft_wplanes", "rick_wcorrect_accumulate", "rick_gridcorrect",
              "rick_image", "rick_image_host", "rick_image_stream_host", "rick_get_image", "rick_get_stats"]:
        assert hasattr(rick.Plan, n)


def test_no_cpu_fallback():
    """Without a CUDA device the product fails loudly instead of computing on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2601_19714_b200 import rick
    with pytest.raises(RuntimeError):
        rick.Plan(256, 8, 7, 1e-4)
    # and the raw ABI refuses too
    lib = rick.load_library()
    h = ctypes.c_void_p()
    d = rick.PlanDesc(256, 8, 7, 1e-4, 0.0, 0, 0, 0, 0, 0, float("nan"), float("nan"))
    assert lib.rick_plan(ctypes.byref(h), ctypes.byref(d), None) == rick.RICK_ERR_CUDA
    assert not h.value


def test_product_does_not_import_oracle():
    """Product and oracle share no code and neither imports / links the other."""
    imp = re.compile(r"^\s*(import|from)\s+oracle\b|dlopen|CDLL\([^)]*oracle|#include\s+\".*oracle", re.M)
    pkg = os.path.join(ROOT, "paper_2601_19714_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not imp.search(open(os.path.join(dirpath, f)).read()), f
    imp2 = re.compile(r"^\s*(import|from)\s+paper_2601_19714_b200\b|CDLL\([^)]*librick_b200|#include\s+\".*(rick\.h|\.cuh)", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            assert not imp2.search(open(os.path.join(ROOT, "oracle", f)).read()), f
