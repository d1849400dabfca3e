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


def test_problem_sizes_reproduce_table_2(lib):
    """The library's own size accounting (rtcc_problem_sizes, no GPU needed) against the T2 column of Table 2:
    three unpacked spin blocks, complex128, GiB -- values in tests/golden/table2_t2_sizes.txt are the paper's."""
    from paper_2301_04249_b200 import rtcc
    rows = [l.split() for l in open(os.path.join(ROOT, "tests", "golden", "table2_t2_sizes.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for name, oa, ob, va, vb, gib in rows:
        oa, ob, va, vb = int(oa), int(ob), int(va), int(vb)
        ps = rtcc.problem_sizes(oa, ob, va, vb, 100)
        assert abs(16 * ps["t2_unpacked_elements"] / 2 ** 30 - float(gib)) < 0.07, name        # 5.74 computed vs 5.8 printed
        P = lambda x: x * (x - 1) // 2
        assert ps["n_t2"] == P(oa) * P(va) + P(ob) * P(vb) + oa * ob * va * vb and ps["n_t1"] == oa * va + ob * vb


def test_memory_budget_of_the_baseline_configs(lib):
    """Closed-form device-memory budget.  Configs 1-4 fit one 180 GB B200 with everything resident; config 5
    needs the low-memory layout, which must stay under 175 GB (the card reports 183 359 MiB = 192 GB) and is bounded below by the paper's own count: the
    Adams-Moulton history (three amplitude-sized tensors) plus the residual and the Cholesky vectors."""
    from paper_2301_04249_b200 import inputs, rtcc
    GB = 1e9
    for name, cfg in inputs.CONFIGS.items():
        oa, ob, va, vb = cfg.dims
        ps = rtcc.problem_sizes(oa, ob, va, vb, cfg.K)
        floor = 4 * 16 * (ps["n_t1"] + ps["n_t2"]) + 8 * ps["cholesky_doubles"]
        assert floor < ps["bytes_lean"] and floor < ps["bytes_standard"]
        if name == "largest":
            assert ps["bytes_standard"] > 300 * GB and ps["bytes_lean"] < 175 * GB
        else:
            assert ps["bytes_standard"] < 160 * GB            # Large: 150 GB incl. the 18 GB of the three-multiplication ring operands
    with pytest.raises(rtcc.RtccError):
        rtcc.problem_sizes(1, 1, 2, 3, 4)
