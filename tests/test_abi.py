"""The C-ABI library loads and exports every symbol include/*.h declares; host-side
argument checks (no compute calls, no GPU)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2602_05255_b200 import build, lrux

    build.build()
    return lrux.load_library()


def _declared():
    names = []
    for h in ("lrux.h", "lrux_harness.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names += re.findall(r"(?:lrux_status_t|const char\*)\s+(lruxh?_\w+)\s*\(", src)
    return sorted(set(names))


def test_exports_every_declared_symbol(lib):
    from paper_2602_05255_b200 import lrux

    names = _declared()
    assert len(names) >= 20
    for name in names:
        assert hasattr(lib, name), name
        assert name in lrux.SIGNATURES, "binding lacks %s" % name
    assert sorted(lrux.SIGNATURES) == names


def test_state_bytes_and_arg_checks(lib):
    from paper_2602_05255_b200 import lrux

    out = C.c_size_t(0)
    assert lib.lrux_det_state_bytes(4, 32, 1, 0, lrux.F64, C.byref(out)) == lrux.OK
    base = out.value
    assert base >= 4 * 32 * 32 * 8
    assert lib.lrux_det_state_bytes(4, 32, 1, 0, lrux.C128, C.byref(out)) == lrux.OK
    assert out.value >= 2 * 4 * 32 * 32 * 8
    assert lib.lrux_det_state_bytes(4, 32, 2, 16, lrux.F64, C.byref(out)) == lrux.OK
    assert out.value >= base + 2 * 4 * 32 * 32 * 8          # two delay buffers of K*k*n
    assert lib.lrux_pf_state_bytes(4, 32, 1, 0, lrux.F64, C.byref(out)) == lrux.OK
    # misuse -> LRUX_EINVAL, nothing done
    assert lib.lrux_pf_state_bytes(4, 33, 1, 0, lrux.F64, C.byref(out)) == lrux.EINVAL   # odd n
    assert lib.lrux_det_state_bytes(0, 32, 1, 0, lrux.F64, C.byref(out)) == lrux.EINVAL
    assert lib.lrux_det_state_bytes(4, 128, 65, 0, lrux.F64, C.byref(out)) == lrux.EINVAL  # k > MAX_K
    # ranks above 8: float64 determinants, K = 0, even n only
    assert lib.lrux_det_state_bytes(4, 128, 9, 0, lrux.F64, C.byref(out)) == lrux.OK
    assert lib.lrux_det_state_bytes(4, 128, 64, 0, lrux.F64, C.byref(out)) == lrux.OK
    assert lib.lrux_det_state_bytes(4, 128, 9, 0, lrux.C128, C.byref(out)) == lrux.EUNSUPPORTED
    assert lib.lrux_det_state_bytes(4, 128, 9, 4, lrux.F64, C.byref(out)) == lrux.EUNSUPPORTED
    assert lib.lrux_det_state_bytes(4, 127, 9, 0, lrux.F64, C.byref(out)) == lrux.EUNSUPPORTED
    assert lib.lrux_pf_state_bytes(4, 128, 9, 0, lrux.F64, C.byref(out)) == lrux.EUNSUPPORTED
    assert lib.lrux_det_state_bytes(4, 32, 1, -1, lrux.F64, C.byref(out)) == lrux.EINVAL
    assert lib.lrux_det_state_bytes(4, 32, 1, 0, 7, C.byref(out)) == lrux.EINVAL
    assert lib.lrux_det_state_bytes(4, 32, 1, 0, lrux.F64, None) == lrux.EINVAL
    assert lib.lrux_destroy(None) == lrux.EINVAL
    assert lib.lrux_det_ratio(None, 1, None, None, None, None) == lrux.EINVAL
    assert lib.lrux_det_init(None, 4, 32, 1, 0, lrux.F64, None, None, 0, None, None) == lrux.EINVAL
    assert b"LRUX_OK" in lib.lrux_status_string(0)
    assert b"EINVAL" in lib.lrux_status_string(1)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2602_05255_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|#include.*oracle|oracle[/.]lrux_oracle",
                                     src, flags=re.M), os.path.join(dirpath, f)
    osrc = open(os.path.join(ROOT, "oracle", "lrux_oracle.py")).read()
    assert "import paper_2602_05255_b200" not in osrc and "from paper_2602_05255_b200" not in osrc
