"""The C-ABI library builds for sm_100a here (no GPU needed) and exports every symbol include/sgs.h
declares; the binding refuses to run without a device (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2506_00970_b200 import build
    return build.build()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sgs.h")).read()
    return sorted(set(re.findall(r"SGS_API\s+[\w\s\*]+?\b(sgs_\w+)\s*\(", src)))


def test_exports_every_declared_symbol(libpath):
    names = declared_symbols()
    assert len(names) >= 14
    lib = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(lib, n), n
    import paper_2506_00970_b200 as m
    assert sorted(m.EXPORTS) == names


def test_status_strings(libpath):
    lib = ctypes.CDLL(libpath)
    lib.sgs_status_string.restype = ctypes.c_char_p
    seen = {lib.sgs_status_string(i) for i in range(6)}
    assert len(seen) == 6 and lib.sgs_status_string(99) == b"unknown status"


def test_sass_is_sm100a(libpath):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback():
    import torch
    import paper_2506_00970_b200 as m
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        m.Renderer()
