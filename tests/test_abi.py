"""CPU-only checks of the C-ABI boundary: libfp.so builds, loads and exports every symbol
include/fp.h declares; argument validation that needs no device.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1609_00958_b200 import fp
    return fp.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "fp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fp_[a-z_]+)\s*\(", text)))


def test_header_declares_the_expected_entry_points():
    from paper_1609_00958_b200 import fp
    assert declared_symbols() == sorted(fp.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_no_torch_types_in_the_abi():
    text = open(os.path.join(ROOT, "include", "fp.h")).read()
    assert "torch" not in text and "at::" not in text and "#include <cuda" not in text


def test_create_validates_arguments(lib):
    h = ctypes.c_void_p()
    o = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    bad = [(0, 4, 4, 1.0), (4, -1, 4, 1.0), (4, 4, 4, 0.0), (4, 4, 4, -1.0), (4, 4, 4, float("nan")),
           (4, 4, 4, float("inf"))]
    for nx, ny, nz, d in bad:
        assert lib.fp_create(nx, ny, nz, d, o, ctypes.byref(h)) == 1
        assert not h.value
    onan = (ctypes.c_double * 3)(0.0, float("nan"), 0.0)
    assert lib.fp_create(4, 4, 4, 1.0, onan, ctypes.byref(h)) == 1
    assert lib.fp_create(4, 4, 4, 1.0, None, ctypes.byref(h)) == 1
    assert lib.fp_create(4, 5, 6, 0.5, o, ctypes.byref(h)) == 0 and h.value
    assert lib.fp_destroy(h) == 0
    assert lib.fp_destroy(None) == 1


def test_options_round_trip_and_reject_unknown(lib):
    from paper_1609_00958_b200 import fp
    with fp.Projector(4, 5, 6, 1.0, (0, 0, 0)) as P:
        assert P.get_option(fp.OPT_VOLATILE) == 1
        P.set_option(fp.OPT_VOLATILE, 0)
        assert P.get_option(fp.OPT_VOLATILE) == 0
        P.set_option(fp.OPT_INTERP, fp.INTERP_SPLINE)
        assert P.get_option(fp.OPT_INTERP) == fp.INTERP_SPLINE
        with pytest.raises(fp.FpError):
            P.set_option(fp.OPT_INTERP, 7)
        with pytest.raises(fp.FpError):
            P.set_option(99, 1)
        with pytest.raises(fp.FpError):
            P.set_option(fp.OPT_KERNEL, 17)


def test_status_strings(lib):
    assert lib.fp_status_string(0) == b"FP_OK"
    assert lib.fp_status_string(2) == b"FP_ERR_CUDA"
    assert b"sm_100a" in lib.fp_version()


def test_project_argument_validation_needs_no_device(lib):
    """Bad arguments are rejected before any CUDA call."""
    import numpy as np
    h = ctypes.c_void_p()
    o = (ctypes.c_double * 3)(0.0, 0.0, 0.0)
    assert lib.fp_create(4, 4, 4, 1.0, o, ctypes.byref(h)) == 0
    g = np.zeros(12)
    gp = g.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    assert lib.fp_project(h, None, 1, gp, 4, 4, None, None) == 1          # null pointers
    assert lib.fp_project(h, 16, -1, gp, 4, 4, 16, None) == 1             # n_proj < 0
    assert lib.fp_project(h, 16, 1, gp, 0, 4, 16, None) == 1              # nu < 1
    assert lib.fp_project(h, None, 0, None, 4, 4, None, None) == 0        # n_proj = 0: no-op
    assert b"n" in lib.fp_last_error(h) or True
    lib.fp_destroy(h)


def test_product_does_not_import_the_oracle():
    """The product package must never route through oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1609_00958_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "joseph_oracle" not in src, f
