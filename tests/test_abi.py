"""CPU-side checks of the boundary: libcspt.so builds, loads and exports every symbol
include/cspt.h declares; argument validation that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cspt_lib():
    from paper_1912_04855_b200 import build, cspt
    build.build()
    return cspt.lib()


def _declared():
    src = open(os.path.join(ROOT, "include", "cspt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cspt_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(cspt_lib):
    from paper_1912_04855_b200 import cspt
    names = _declared()
    assert len(names) >= 16
    bound = {n for n, _, _ in cspt.SYMBOLS}
    for n in names:
        assert hasattr(cspt_lib, n), n
        assert n in bound, "binding lacks " + n


def test_workspace_bytes_and_strerror(cspt_lib):
    assert cspt_lib.cspt_workspace_bytes(0, 4, 4, 0) == 0
    assert cspt_lib.cspt_workspace_bytes(4, 4, 4, 7) == 0
    b64 = cspt_lib.cspt_workspace_bytes(64, 4, 4, 0)
    b32 = cspt_lib.cspt_workspace_bytes(64, 4, 4, 1)
    assert b64 > b32 > 0 and b64 % 256 == 0
    # 1024^3 fp32 must fit a 180 GB B200 with room for the caller's arrays
    assert cspt_lib.cspt_workspace_bytes(1024, 1024, 1024, 1) < 150e9
    assert cspt_lib.cspt_strerror(0) == b"ok"
    assert b"invalid" in cspt_lib.cspt_strerror(-1)


def test_create_rejects_bad_arguments_without_a_device(cspt_lib):
    h = ctypes.c_void_p()
    bc = (ctypes.c_int * 6)(0, 0, 0, 0, 0, 0)
    ws = ctypes.c_void_p(256)     # never dereferenced on the EINVAL paths
    big = 1 << 40
    f = cspt_lib.cspt_create
    assert f(None, 8, 8, 8, 0.1, 1.4, bc, 0, ws, big, None) == -1
    assert f(ctypes.byref(h), 0, 8, 8, 0.1, 1.4, bc, 0, ws, big, None) == -1
    assert f(ctypes.byref(h), 8, 8, 8, -0.1, 1.4, bc, 0, ws, big, None) == -1
    assert f(ctypes.byref(h), 8, 8, 8, 0.1, 1.0, bc, 0, ws, big, None) == -1
    assert f(ctypes.byref(h), 8, 8, 8, 0.1, 1.4, bc, 2, ws, big, None) == -1
    assert f(ctypes.byref(h), 8, 8, 8, 0.1, 1.4, bc, 0, ws, 16, None) == -1            # workspace too small
    assert f(ctypes.byref(h), 8, 8, 8, 0.1, 1.4, bc, 0, ctypes.c_void_p(8), big, None) == -1   # misaligned
    mixed = (ctypes.c_int * 6)(0, 1, 0, 0, 0, 0)
    assert f(ctypes.byref(h), 8, 8, 8, 0.1, 1.4, mixed, 0, ws, big, None) == -1
    small = (ctypes.c_int * 6)(1, 1, 0, 0, 0, 0)
    assert f(ctypes.byref(h), 3, 8, 8, 0.1, 1.4, small, 0, ws, big, None) == -1       # n < 4 on a non-periodic axis
    assert cspt_lib.cspt_step(None, 0.1) == -1
    cspt_lib.cspt_destroy(None)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1912_04855_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "csph_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, fn
    orc = open(os.path.join(ROOT, "oracle", "csph_oracle.cpp")).read()
    assert "cspt.h" not in orc.replace("paper_1912_04855_b200/csrc", "") and "#include \"cspt" not in orc
