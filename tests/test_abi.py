"""The C-ABI library loads here (no GPU) and exports every symbol include/tmd.h declares; host-side argument checks."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "tmd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tmd_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    names = declared_functions()
    for must in ("tmd_create", "tmd_decode", "tmd_destroy", "tmd_workspace_bytes", "tmd_decode_host", "tmd_status_string"):
        assert must in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2411_02206_b200 import build, tmd
    path = build.build()
    assert os.path.exists(path)
    L = C.CDLL(path)
    for name in declared_functions():
        assert hasattr(L, name), name
    assert tmd.tmd_status_string(0) == "ok" and tmd.tmd_status_string(-5) == "inconsistent compressed input"


def test_binding_struct_layout_matches_header_sizes():
    # x86-64 SysV layout of the structs the binding marshals (pointers 8 bytes, natural alignment)
    from paper_2411_02206_b200 import tmd
    assert C.sizeof(tmd.tmd_geometry) == 4 * 4 + 2 * 4 + 4 * 8
    assert C.sizeof(tmd.tmd_compressed) == 8 + 8 + 8 + 23 * 8
    assert C.sizeof(tmd.tmd_output) == 3 * 8 + 8 + 8 + 8
    assert len(tmd.COMPRESSED_ARRAYS) == 23


def test_sources_are_sm100a_only_and_do_not_touch_the_oracle():
    from paper_2411_02206_b200 import build
    assert "arch=compute_100a,code=sm_100a" in " ".join(build.FLAGS) and "--fmad=false" in build.FLAGS
    pkg = os.path.join(ROOT, "paper_2411_02206_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "tmd_oracle" not in text, f
