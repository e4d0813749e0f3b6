"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports
every symbol include/qcd.h declares.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2502_03249_b200 import build, load_library
    build.build()
    return load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "qcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qcd_[a-zA-Z_]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    import paper_2502_03249_b200 as pkg
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/qcd.h but not exported"
    assert sorted(pkg.SYMBOLS) == declared, "binding symbol list out of sync with include/qcd.h"


def test_library_is_sm100a_only(lib):
    import subprocess
    from paper_2502_03249_b200.build import LIB_PATH
    out = subprocess.run(["cuobjdump", "-lelf", LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def test_strerror_and_argument_errors_without_gpu(lib):
    assert lib.qcd_strerror(0) == b"ok"
    assert b"converge" in lib.qcd_strerror(4)
    h = ctypes.c_void_p()
    bad = (ctypes.c_int * 4)(4, 4, 3, 4)                    # odd extent: rejected before any CUDA call
    assert lib.qcd_init(ctypes.byref(h), bad, 64, None) == 1
    assert b"even" in lib.qcd_last_error(None)
    ok = (ctypes.c_int * 4)(4, 4, 4, 4)
    assert lib.qcd_init(ctypes.byref(h), ok, 16, None) == 1   # bad precision
    bad0 = (ctypes.c_int * 4)(6, 4, 4, 4)
    assert lib.qcd_init(ctypes.byref(h), bad0, 64, None) == 1  # N0 % 4
    assert lib.qcd_field_bytes(None, 0) == 0


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p()
    ok = (ctypes.c_int * 4)(4, 4, 4, 4)
    assert lib.qcd_init(ctypes.byref(h), ok, 64, None) == 3          # QCD_ECUDA
    assert b"no CPU fallback" in lib.qcd_last_error(None)
    import paper_2502_03249_b200 as pkg
    with pytest.raises(RuntimeError):
        pkg.Context((4, 4, 4, 4), 64)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2502_03249_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), (d, f)
                assert "liboracle" not in src and "staggered_oracle" not in src, (d, f)
