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
    """The product path never routes through the oracle (③): no import of oracle/ or of the test-support
    generators anywhere in the package, no CPU fallback module, no library FFT (north_star: cuFFT is never
    on the product path), no environment variables read behind the C ABI, and the method's arithmetic only
    in csrc/ (the Python side holds marshalling and index bookkeeping)."""
    pkg = os.path.join(ROOT, "paper_1006_4644_b200")
    py_files = []
    for dirpath, dirs, files in os.walk(pkg):
        dirs[:] = [d for d in dirs if d != "__pycache__"]
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+(oracle|testsupport)\b", txt, flags=re.M), f
                assert "mf_oracle" not in txt and "liboracle" not in txt, f
                assert not re.search(r"torch\.fft|cufft|numpy\.fft|np\.fft|scipy\.fft", txt, flags=re.I), f
                assert "getenv" not in txt, f
                if f.endswith(".py"):
                    py_files.append(f)
                    # the 2PN phase coefficients (3715/756, 15293365/508032) belong to csrc/ only
                    assert "3715" not in txt and "15293365" not in txt and "4.925490947641267e-6" not in txt, f
    assert sorted(py_files) == ["__init__.py", "build.py", "cbmf.py", "sharding.py"], py_files
    assert sorted(os.listdir(os.path.join(pkg, "csrc"))) == ["cbmf.cu", "cluster.h", "fft_regs.cuh", "kernels.cuh", "probe.cuh", "td.cuh"]


def test_binding_rejects_wrong_dtypes():
    """cbmf.py checks dtype / size of every array it hands to the C ABI (a float32 PSD tensor would be
    read as float64 by the kernel).  Pure host checks: they raise before any library call."""
    import numpy as np
    import pytest
    import torch
    from paper_1006_4644_b200 import cbmf
    with pytest.raises(ValueError):
        cbmf._ptr(torch.zeros(9, dtype=torch.float32), "float64")
    with pytest.raises(ValueError):
        cbmf._ptr(torch.zeros(8, dtype=torch.float64), "float32")
    with pytest.raises(ValueError):
        cbmf._ptr(np.zeros(8, dtype=np.float32), "float64")
    with pytest.raises(ValueError):
        cbmf._ptr(torch.zeros(24, dtype=torch.uint8), "peak records", itemsize=16)     # not a multiple of 16 bytes
    with pytest.raises(ValueError):
        cbmf._ptr(torch.zeros((4, 4), dtype=torch.float64).t(), "float64")               # not contiguous
    assert cbmf._ptr(torch.zeros(32, dtype=torch.uint8), "peak records", itemsize=16)[1] is False
    assert cbmf._ptr(np.zeros(2, dtype=cbmf.PEAK_DTYPE), "peak records", itemsize=16)[1] is False
    assert cbmf._ptr(torch.zeros(8, dtype=torch.float64), "float64")[1] is False


def test_binding_keeps_stream_ordered_inputs_alive(monkeypatch):
    """cbmf_set_psd_dev / cbmf_load_segment_dev return before the device has read their input: the binding holds
    the tensors until a call that waits for the context's stream has returned (no GPU: stubbed library, fake tensors)."""
    from paper_1006_4644_b200 import cbmf

    class Stub:
        def __getattr__(self, name):
            if name == "cbmf_strerror":
                return lambda rc: b"stub"
            return lambda *a: 0

    class FakeTensor:
        is_cuda = True
        dtype = "torch.float64"

        class device:
            index = 0

        def __init__(self, n, dtype):
            self._n, self.dtype = n, dtype

        def data_ptr(self):
            return 4096

        def is_contiguous(self):
            return True

        def numel(self):
            return self._n

    monkeypatch.setattr(cbmf, "lib", lambda: Stub())
    g = cbmf.Context(1 << 12, 4096.0, 40.0)
    psd, seg = FakeTensor((1 << 11) + 1, "torch.float64"), FakeTensor(1 << 12, "torch.float32")
    g.set_psd(psd)
    g.load_segment(seg)
    assert g._held == [psd, seg]
    g.set_profiling(0); g.get_split()                  # calls that do not wait keep them
    assert g._held == [psd, seg]
    g.filter_bank([[1.4, 1.4]], 6.0)                   # a call that waits releases them
    assert g._held == []
    g.load_segment(seg)
    assert g._held == [seg]
    g.close()
    assert g._held == []
