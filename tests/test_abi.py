"""Host-side checks that need no GPU: the C-ABI library builds/loads and exports every symbol that
include/rtcc.h declares; argument validation that happens before any CUDA call."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2301_04249_b200 import build, rtcc
    build.build()
    return rtcc.load()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "rtcc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(rtcc_[a-z0-9_]+)\s*\(", hdr))
    assert len(names) >= 20
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in include/rtcc.h but not exported"
    from paper_2301_04249_b200 import rtcc
    assert set(rtcc.SYMBOLS) == names


def test_strerror_and_invalid_arguments(lib):
    assert lib.rtcc_strerror(0) == b"ok"
    assert b"converge" in lib.rtcc_strerror(-4)
    h = ctypes.c_void_p()
    buf = (ctypes.c_double * 8)()
    # validation precedes any CUDA call, so these run without a GPU
    assert lib.rtcc_create(ctypes.byref(h), 1, 1, 2, 3, 4, buf, buf, 1, None) == -1      # oa+va != ob+vb
    assert lib.rtcc_create(ctypes.byref(h), 1, 1, 0, 0, 4, buf, buf, 1, None) == -1      # no virtuals
    assert lib.rtcc_create(ctypes.byref(h), 0, 0, 2, 2, 4, buf, buf, 1, None) == -1      # no electrons
    assert lib.rtcc_create(ctypes.byref(h), 1, 1, 2, 2, 0, buf, buf, 1, None) == -1      # no Cholesky vectors
    assert lib.rtcc_create(ctypes.byref(h), 1, 1, 2, 2, 4, None, buf, 1, None) == -1     # null L
    assert lib.rtcc_create(None, 1, 1, 2, 2, 4, buf, buf, 1, None) == -1
    assert lib.rtcc_step(None, 0.1) == -1
    assert lib.rtcc_cumulant(None, buf) == -1
    assert lib.rtcc_residual(None, buf, buf, buf, buf) == -1


def test_product_has_no_oracle_dependency():
    """The product path must not import / call the oracle (nor any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2301_04249_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|from\s+\.+\s*oracle|oracle[/.]|librtcc_oracle|orc_", src), f
