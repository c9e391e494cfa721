"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/fdd.h declares; argument validation that needs no GPU; no compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2110_03482_b200 import build as fbuild
    fbuild.build()
    from paper_2110_03482_b200 import binding
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "fdd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fdd_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = _declared_symbols()
    assert "fdd_plan_create" in names and "fdd_execute" in names and "fdd_plan_destroy" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/fdd.h but not exported"
    from paper_2110_03482_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_error_strings(lib):
    from paper_2110_03482_b200 import binding
    assert binding.error_string(0) == "ok"
    assert "argument" in binding.error_string(-1)
    assert binding.error_string(-99) == "unknown status"


def test_argument_validation_without_gpu(lib):
    h = ctypes.c_void_p()
    dms = (ctypes.c_double * 2)(0.0, 1.0)
    bad = [
        (0, 128, 64e-6, 1200.0, 1500.0, 2),     # nchans
        (4, 1, 64e-6, 1200.0, 1500.0, 2),       # nsamps
        (4, 128, 0.0, 1200.0, 1500.0, 2),       # tsamp
        (4, 128, 64e-6, 0.0, 1500.0, 2),        # f_lo
        (4, 128, 64e-6, 1500.0, 1200.0, 2),     # f_lo > f_hi
        (4, 128, 64e-6, 1200.0, 1500.0, 0),     # ndm
    ]
    for nch, ns, ts, flo, fhi, ndm in bad:
        rc = lib.fdd_plan_create(ctypes.byref(h), nch, ns, ts, flo, fhi, dms, ndm)
        assert rc == -1 and not h.value
    nan = (ctypes.c_double * 2)(0.0, float("nan"))
    assert lib.fdd_plan_create(ctypes.byref(h), 4, 128, 64e-6, 1200.0, 1500.0, nan, 2) == -1
    assert lib.fdd_plan_create(None, 4, 128, 64e-6, 1200.0, 1500.0, dms, 2) == -1
    assert lib.fdd_plan_destroy(None) == 0
    assert lib.fdd_execute(None, None, None, 0, None) == -1
    assert lib.fdd_plan_get_info(None, None, None, None, None, None, None) == -1


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or synth) -- check the sources."""
    pkg = os.path.join(ROOT, "paper_2110_03482_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), (f, "mentions oracle")
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2110_03482_b200" not in src and "from paper_2110_03482_b200" not in src
