"""CPU-side checks of the C ABI: the library builds, loads and exports every symbol
include/qcd.h declares; argument validation that needs no device; and the product path
fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def qcd():
    from paper_2001_05706_b200 import build
    build.build()
    from paper_2001_05706_b200 import qcd as q
    q.lib()
    return q


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "qcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qcd_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound(qcd):
    names = declared_symbols()
    assert len(names) >= 30
    L = C.CDLL(qcd.LIB_PATH)
    for n in names:
        assert hasattr(L, n), "libqcd_b200.so does not export %s" % n
        assert n in qcd.SIGNATURES, "python binding has no signature for %s" % n
    assert sorted(qcd.SIGNATURES) == names


def test_size_queries(qcd):
    L = qcd.lib()
    d = qcd._dims((16, 16, 16, 32))
    V = 16 * 16 * 16 * 32
    assert L.qcd_gauge_bytes(d, 4, 18) == 37748736
    assert L.qcd_gauge_bytes(d, 4, 12) == 25165824
    assert L.qcd_spinor_bytes(d, 4) == V * 24 * 4
    assert L.qcd_clover_bytes(qcd._dims((24, 24, 24, 64)), 8) == 2 * 509607936
    # odd or too small extents, bad precision
    assert L.qcd_gauge_bytes(qcd._dims((3, 4, 4, 4)), 4, 12) == 0
    assert L.qcd_gauge_bytes(qcd._dims((4, 4, 4, 0)), 4, 12) == 0
    assert L.qcd_gauge_bytes(d, 3, 12) == 0
    # 16-bit storage (reading H1): 24 B per link, 148 B per clover site and block, 52 B per spinor site
    assert L.qcd_gauge_bytes(d, 2, 12) == 8 * (V // 2) * 24
    assert L.qcd_gauge_bytes(d, 2, 18) == 0
    assert L.qcd_clover_bytes(d, 2) == 4 * (V // 2) * 148
    assert L.qcd_half_spinor_bytes(d) == V * 52
    assert L.qcd_gauge_bytes(d, 4, 8) == 0


def test_no_device_means_error_not_fallback(qcd):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    rc = qcd.lib().qcd_init(0, None, C.byref(h))
    assert rc == qcd.ECUDA
    assert b"no CPU fallback" in qcd.lib().qcd_last_error()
    with pytest.raises(RuntimeError):
        qcd.Context(0)


def test_null_arguments_are_rejected(qcd):
    L = qcd.lib()
    assert L.qcd_cg_solve(None, None, 1e-10, 10) == qcd.EINVAL
    assert L.qcd_hop(None, None, None, 0, 0, qcd._dims((4, 4, 4, 4)), 4) == qcd.EINVAL
    assert L.qcd_set_operator(None, None, None, None, None, 0.1, 0.0, 2, 0.1) == qcd.EINVAL
    assert L.qcd_norm2(None, None, 4, 4, None) == qcd.EINVAL


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2001_05706_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "qcd_oracle" not in src and "liboracle" not in src, f
