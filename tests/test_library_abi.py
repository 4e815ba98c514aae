"""Host-side checks that need no GPU: libmred.so builds for sm_100a, loads, and exports every symbol that
include/mred.h declares; the product path holds no route into the oracle; generator/oracle independence."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2008_11486_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "mred.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mred_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported(libpath):
    names = _declared()
    assert len(names) >= 12 and "mred_calibrate" in names
    lib = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(lib, n), "libmred.so does not export %s" % n
    from paper_2008_11486_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_host_only_calls(libpath):
    from paper_2008_11486_b200 import binding as m
    assert m.lib().mred_version().startswith(b"mred")
    assert m.lib().mred_strerror(-3) == b"workspace missing or too small"
    g = (1074, 1024, 0, 50, 50, 0, 1024, 1024)
    assert m.workspace_bytes(m.CALL_CALIBRATE, g, 10) == 10 * 4 * 8      # 4 block partials of the overscan sum per frame
    need = m.workspace_bytes(m.CALL_REDUCE, g, 10)
    assert need >= 2 * 10 * 1024 * 1024 * 4
    assert m.reduce_host_workspace_bytes(g, 10) >= need + 10 * 1074 * 1024 * 2
    assert m.workspace_bytes(m.CALL_COADD, g, 10) == 0
    assert m.workspace_bytes(m.CALL_RESAMPLE, g, 10) == 0      # 16-byte-aligned rows, >= 256 x 64: the tiled kernel, no scratch
    assert m.workspace_bytes(m.CALL_RESAMPLE, (4128, 4096, 0, 32, 32, 0, 4096, 4096), 100) == 0
    assert m.workspace_bytes(m.CALL_RESAMPLE, (0, 0, 0, 0, 0, 0, 192, 136), 12) == 12 * 192 * 136 * 4   # small planes: x kernel + y kernel


def test_sass_is_sm100a(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_product_path_never_touches_oracle():
    pkg = os.path.join(ROOT, "paper_2008_11486_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle's", "").replace("float64 oracle", "").lower() or \
                    not re.search(r"^\s*(import|from)\s+oracle|#include.*oracle", txt, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2008_11486_b200|#include.*csrc", txt, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "synth")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "synth", f)).read()
            assert not re.search(r"^\s*(import|from)\s+(oracle|paper_2008_11486_b200)", txt, flags=re.M), f
