"""The C-ABI library loads on a machine without a GPU and exports every symbol include/frost.h
declares; argument errors are reported as status codes (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2011_14984_b200 import build as b
    b.build()
    import paper_2011_14984_b200 as frost
    return frost.load_library()


def _declared():
    names = set()
    inc = os.path.join(ROOT, "include")
    for h in sorted(os.listdir(inc)):
        if h.endswith(".h"):
            src = open(os.path.join(inc, h)).read()
            src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
            names |= set(re.findall(r"\b(frost_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_every_declared_symbol_is_exported(lib):
    import paper_2011_14984_b200 as frost
    names = _declared()
    assert len(names) >= 15
    assert sorted(frost.exported_symbols) == names
    for nm in names:
        assert hasattr(lib, nm), nm


def test_status_codes_and_strings(lib):
    assert lib.frost_strerror(0) == b"ok"
    assert b"invalid" in lib.frost_strerror(-1)
    assert lib.frost_version().startswith(b"frost-b200")
    assert lib.frost_create(None, 0, None) == -1          # FROST_EINVAL: NULL out pointer
    assert lib.frost_destroy(None) == -1
    assert lib.frost_forces(None, 1, 1, None, None, None, None, 0, None, 0, None, None, 1) == -1


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    import paper_2011_14984_b200 as frost
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    assert lib.frost_create(C.byref(h), 0, None) == -2    # FROST_ECUDA: fails loudly
    with pytest.raises(frost.FrostError):
        frost.Frost()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2011_14984_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "frost_oracle" not in txt, f
