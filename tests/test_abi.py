"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/pct.h declares; argument errors that need no GPU are reported, not crashed on."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pct():
    import paper_1707_05014_b200 as p

    p.build()
    return p


def test_header_symbols_are_exported(pct):
    hdr = open(os.path.join(ROOT, "include", "pct.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pct_[a-z_]+)\s*\(", hdr))
    assert {"pct_create", "pct_set_histories", "pct_iterate", "pct_get_image"} <= declared
    L = pct.lib()
    for name in declared:
        assert hasattr(L, name), "libpct.so does not export %s" % name
    assert declared == set(pct.EXPORTS)


def test_library_is_sm100a_and_has_no_torch_dependency(pct):
    import subprocess

    from paper_1707_05014_b200 import _build

    out = subprocess.run(["cuobjdump", "-lelf", _build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    deps = subprocess.run(["ldd", _build.LIB], capture_output=True, text=True).stdout
    assert "torch" not in deps and "libc10" not in deps


def test_version_and_null_safety(pct):
    assert "sm_100a" in pct.pct_version()
    pct.pct_destroy(None)  # NULL-safe
    assert pct.lib().pct_iterate(None, 0.1, 10, 1) == -1
    assert pct.lib().pct_get_image(None, None, 0) == -1


def test_create_rejects_bad_arguments_without_a_gpu(pct):
    L = pct.lib()
    h = C.c_void_p()
    assert L.pct_create(None, 8, 8, 8, 1.0, -8.0, 8.0, None) == -1
    for args in [(0, 8, 8, 1.0, -8.0, 8.0), (8, 8, 8, 0.0, -8.0, 8.0), (8, 8, 8, -1.0, -8.0, 8.0),
                 (8, 8, 8, 1.0, -3.0, 8.0), (8, 8, 8, 1.0, -8.0, 3.9), (8, 8, 8, float("nan"), -8.0, 8.0),
                 (2048, 2048, 1024, 1.0, -2000.0, 2000.0)]:
        assert L.pct_create(C.byref(h), *args, None) == -1
        assert h.value is None
        assert len(L.pct_last_error(None)) > 0


def test_product_never_touches_the_oracle():
    """The product path must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1707_05014_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower(), f
