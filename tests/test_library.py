"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/whp.h declares; argument errors are reported without a GPU; the product package never
touches the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def so_path():
    from paper_2110_13693_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "whp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(whp_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(so_path):
    lib = C.CDLL(so_path)
    declared = _declared_symbols()
    assert len(declared) >= 13
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/whp.h but not exported"
    from paper_2110_13693_b200 import whp
    assert sorted(whp.SYMBOLS) == declared


def test_version_and_null_handling(so_path):
    from paper_2110_13693_b200 import whp
    L = whp.lib()
    assert b"sm_100a" in L.whp_version()
    assert L.whp_last_error(None) == b"null context"
    assert L.whp_launch_count(None) == 0
    L.whp_destroy(None)  # no-op
    assert L.whp_load_orders(None, 1, None, None, 1) == whp.ERR_INVALID_ARG
    assert L.whp_set_penalty(None, None, None, None) == whp.ERR_INVALID_ARG
    assert L.whp_argmin(None, None, 1, None, None, None) == whp.ERR_INVALID_ARG


def test_create_layout_argument_errors(so_path):
    """Validation happens before any CUDA call, so these are decidable on a CPU-only box."""
    from paper_2110_13693_b200 import whp
    L = whp.lib()
    loc = np.array([0, 5, 79], np.int32)
    cls = np.array([0, 1, 3], np.int32)
    h = C.c_void_p()

    def create(na=4, s=10, pitch=1, sp=3, depot=0, n=3, loc=loc, cls=cls, k=4, out=h):
        return L.whp_create_layout(na, s, pitch, sp, depot, n, loc.ctypes.data if loc is not None
                                   else None, cls.ctypes.data if cls is not None else None, k, 0,
                                   C.byref(out) if out is not None else None)
    assert create(out=None) == whp.ERR_INVALID_ARG
    assert create(loc=None) == whp.ERR_INVALID_ARG
    assert create(na=0) == whp.ERR_INVALID_ARG
    assert create(k=0) == whp.ERR_INVALID_ARG
    assert create(na=1025) == whp.ERR_OUT_OF_RANGE
    assert create(s=4096) == whp.ERR_OUT_OF_RANGE
    assert create(k=257) == whp.ERR_OUT_OF_RANGE
    assert create(depot=4) == whp.ERR_OUT_OF_RANGE
    assert create(loc=np.array([0, 5, 80], np.int32)) == whp.ERR_OUT_OF_RANGE
    assert create(cls=np.array([0, 1, 4], np.int32)) == whp.ERR_OUT_OF_RANGE
    assert h.value is None


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2110_13693_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "whp_oracle" not in text, f
    orc = open(os.path.join(ROOT, "oracle", "whp_oracle.c")).read()
    assert "csrc" not in orc.split("*/")[1] and "#include \"" not in orc


def test_missing_library_fails_loudly(monkeypatch):
    from paper_2110_13693_b200 import whp
    monkeypatch.setattr(whp, "_lib", None)
    monkeypatch.setattr(whp, "_SO", os.path.join(ROOT, "does_not_exist.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        whp.lib()
