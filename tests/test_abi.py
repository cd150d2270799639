"""The boundary without a GPU: libgx.so builds (nvcc cross-compiles sm_100a), loads, and exports every function
include/gx.h declares; the ctypes binding lists the same names; the product and the oracle do not touch each other."""
from __future__ import annotations

import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gx_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2306_07552_b200 import binding, build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert {"gx_create_scene", "gx_render_batch", "gx_destroy", "gx_last_error"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names
    # no compute without a GPU, but argument errors are reported without one
    lib.gx_last_error.restype = ctypes.c_char_p
    assert lib.gx_render_batch(None, None, 0, 0, None, None, None, None, None, None, None, None) == -1
    assert b"NULL" in lib.gx_last_error() or b"depth_out" in lib.gx_last_error()


def test_product_and_oracle_are_independent():
    pkg = os.path.join(ROOT, "paper_2306_07552_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert not re.search(r'#include\s+"[^"]*oracle', text), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2306_07552_b200" not in re.sub(r'""".*?"""', "", text, flags=re.S).replace("paper_2306_07552_b200/csrc", ""), f
            assert not re.search(r'#include\s+"[^"]*(gx\.h|csrc)', text), f
    hdr = open(os.path.join(ROOT, "include", "gx.h")).read()
    assert "oracle" not in hdr.lower() or "#include" not in "".join(l for l in hdr.splitlines() if "oracle" in l.lower())
