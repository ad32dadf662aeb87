"""No-GPU checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/fdgs.h declares; host-side argument checks that need no device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2412_20720_b200 import build, fdgs
    build.build()
    return fdgs.load()


def _declared():
    text = open(os.path.join(ROOT, "include", "fdgs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fdgs_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2412_20720_b200 import fdgs
    names = _declared()
    assert len(names) >= 10
    assert set(names) == set(fdgs.EXPORTED_SYMBOLS)
    for n in names:
        assert getattr(lib, n) is not None


def test_library_is_sm100a_only():
    import subprocess
    from paper_2412_20720_b200 import fdgs
    out = subprocess.run(["cuobjdump", "-lelf", fdgs.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out


def test_host_side_calls_without_a_device(lib):
    from paper_2412_20720_b200 import fdgs
    cfg = fdgs.default_config()
    assert abs(cfg.marginal_min - 0.05) < 1e-9 and abs(cfg.alpha_min - 1 / 255) < 1e-9 and abs(cfg.alpha_max - 0.99) < 1e-7
    assert lib.fdgs_default_config(None) == fdgs.ERR_INVALID
    n1 = fdgs.workspace_bytes(1000, 48, 1352, 1014, 1 << 20)
    n2 = fdgs.workspace_bytes(2000, 48, 1352, 1014, 1 << 20)
    n3 = fdgs.workspace_bytes(1000, 48, 1352, 1014, 1 << 21)
    assert n2 > n1 and n3 > n1 and n3 - n1 >= 4 * (1 << 20)      # 4 B per pair of capacity: ids only, no key array
    with pytest.raises(fdgs.FdgsError):
        fdgs.workspace_bytes(-1, 48, 64, 64, 100)
    with pytest.raises(fdgs.FdgsError):
        fdgs.workspace_bytes(10, 48, 64, 64, 1 << 31)
    assert fdgs.strerror(fdgs.ERR_PAIR_OVERFLOW).startswith("number of")
    assert fdgs.strerror(0) == "ok"


def test_struct_layouts_match_the_header():
    from paper_2412_20720_b200 import fdgs
    assert C.sizeof(fdgs.CScene) == 64           # 3 x int32 (+pad) + 6 pointers
    assert C.sizeof(fdgs.CView) == 64 + 16 + 8 + 8 + 12
    assert C.sizeof(fdgs.CConfig) == 32
    assert C.sizeof(fdgs.CGrads) == 64
    assert C.sizeof(fdgs.CViewBuffers) == 64


def test_product_fails_loudly_without_the_library(monkeypatch):
    from paper_2412_20720_b200 import fdgs
    monkeypatch.setattr(fdgs, "_lib", None)
    monkeypatch.setattr(fdgs, "LIB_PATH", "/nonexistent/libfdgs.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        fdgs.load()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_20720_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "fdgs_oracle" not in src, f
