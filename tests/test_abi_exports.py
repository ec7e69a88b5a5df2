"""CPU checks of the boundary: the C-ABI library builds, loads, and exports every function
include/cbmf.h declares; the binding declares the same names; no compute calls (no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "cbmf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cbmf_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    from paper_1006_4644_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in cbmf.h but not exported"


def test_binding_matches_header():
    from paper_1006_4644_b200 import cbmf
    assert sorted(cbmf.EXPORTS) == _declared()
    cbmf.lib()                                   # declares argtypes for every name or raises
    assert cbmf.version().startswith("cbmf")
    assert cbmf.lib().cbmf_strerror(cbmf.ESTATE).decode().startswith("call order")


def test_argument_errors_need_no_gpu():
    """EINVAL paths that return before any CUDA call."""
    from paper_1006_4644_b200 import cbmf
    L = cbmf.lib()
    h = ctypes.c_void_p()
    assert L.cbmf_create(None, 0, 1 << 16, 2048.0, 40.0, None) == cbmf.EINVAL
    assert L.cbmf_create(ctypes.byref(h), 0, 1000, 2048.0, 40.0, None) == cbmf.EINVAL
    assert L.cbmf_create(ctypes.byref(h), 0, 1 << 25, 2048.0, 40.0, None) == cbmf.EINVAL
    assert L.cbmf_create(ctypes.byref(h), 0, 1 << 16, -1.0, 40.0, None) == cbmf.EINVAL
    assert L.cbmf_create(ctypes.byref(h), 0, 1 << 16, 2048.0, 1024.0, None) == cbmf.EINVAL
    assert L.cbmf_destroy(None) == cbmf.EINVAL
    assert L.cbmf_set_psd(None, None, 0) == cbmf.EINVAL
    assert L.cbmf_launch_count(None) == -1


def test_product_does_not_import_oracle():
    """The product path never routes through the oracle (③): no import of oracle/ anywhere
    in the package, and no CPU fallback module."""
    pkg = os.path.join(ROOT, "paper_1006_4644_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "mf_oracle" not in txt and "liboracle" not in txt, f
