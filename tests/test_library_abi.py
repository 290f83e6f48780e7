"""-m "not gpu": libcdh.so builds, loads without a GPU and exports every symbol include/*.h declares;
host-side argument validation returns error codes (no compute calls here)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1808_01478_b200 import binding
from paper_1808_01478_b200 import build as cdh_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    names = set()
    for h in ("cdh.h", "cdh_bench.h"):
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names.update(re.findall(r"\b(cdh_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


@pytest.fixture(scope="module")
def lib():
    cdh_build.build()
    return binding.load()


def test_headers_declare_the_boundary():
    names = declared_symbols()
    for required in ("cdh_create", "cdh_histograms", "cdh_destroy"):
        assert required in names
    assert sorted(binding.EXPORTS) == names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert getattr(lib, name) is not None


def test_strerror_texts(lib):
    assert binding.cdh_strerror(0) == "ok"
    assert "invalid" in binding.cdh_strerror(binding.ERR_INVALID_ARG)
    assert "unsupported" in binding.cdh_strerror(binding.ERR_UNSUPPORTED)
    assert "unknown" in binding.cdh_strerror(-99)


def test_null_arguments_are_rejected_without_a_device(lib):
    assert lib.cdh_create(None, 0, 0) == binding.ERR_INVALID_ARG
    off = np.array([0, 4], dtype=np.int32)
    rc = lib.cdh_histograms(None, 1, 1, off.ctypes.data, 1, 0, None, 0, 1.0, 8, 0, None, 1)
    assert rc == binding.ERR_INVALID_ARG
    assert lib.cdh_destroy(None) == binding.OK
    info = (ctypes.c_int64 * 8)()
    assert lib.cdh_last_call_info(None, info) == binding.ERR_INVALID_ARG
    # the entry point without a context checks its arguments, and its size limits, before it touches a device
    assert lib.cdh_histograms_noalloc(0, None, 1, off.ctypes.data, 1, 0, None, 0, 1.0, 8, None, 1) == binding.ERR_INVALID_ARG
    assert b"null pointer" in lib.cdh_noalloc_last_error()
    big = np.array([0, 131073], dtype=np.int32)
    assert lib.cdh_histograms_noalloc(0, 1, 1, big.ctypes.data, 1, 0, None, 0, 1.0, 8, None, 1) == binding.ERR_UNSUPPORTED
    assert b"131072 padded particles" in lib.cdh_noalloc_last_error()
    assert lib.cdh_histograms_noalloc(0, 1, 1, off.ctypes.data, 1, 0, None, 0, 1.0, 32769, None, 1) == binding.ERR_UNSUPPORTED
    assert b"n_bins" in lib.cdh_noalloc_last_error()


def test_no_cpu_fallback_when_library_is_missing(tmp_path):
    with pytest.raises(OSError):
        binding.load(str(tmp_path / "libcdh_missing.so"))


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1808_01478_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert not re.search(r"#include\s+[\"<][^\">]*oracle", text), f
                assert "libcdh_oracle" not in text, f


def test_binding_rejects_tensors_the_c_call_would_misread():
    """Context.cdh_histograms takes data_ptr() of torch tensors: a CPU, non-contiguous, wrongly typed or undersized tensor
    must be refused by the binding (the C ABI sees plain pointers and cannot tell)."""
    torch = pytest.importorskip("torch")
    from paper_1808_01478_b200 import binding
    with pytest.raises(ValueError, match="CUDA tensor"):
        binding._check_device_tensor(torch.zeros(30), "coords", 0, "float32", 30)
    binding._check_device_tensor(123456, "coords", 0, "float32", 30)          # raw pointers pass through
    binding._check_device_tensor(None, "coords", 0, "float32", 30)

    class Fake:                                                                # stands in for a CUDA tensor on a CPU-only box
        is_cuda = True
        dtype = torch.float64
        class device:
            index = 0
        def __init__(self, n, contiguous=True): self._n, self._c = n, contiguous
        def data_ptr(self): return 1
        def is_contiguous(self): return self._c
        def numel(self): return self._n
    with pytest.raises(ValueError, match="dtype"):
        binding._check_device_tensor(Fake(30), "coords", 0, "float32", 30)
    with pytest.raises(ValueError, match="contiguous"):
        binding._check_device_tensor(Fake(30, False), "coords", 0, "float64", 30)
    with pytest.raises(ValueError, match="elements"):
        binding._check_device_tensor(Fake(29), "coords", 0, "float64", 30)
    with pytest.raises(ValueError, match="cuda:0"):
        binding._check_device_tensor(Fake(30), "coords", 1, "float64", 30)
    binding._check_device_tensor(Fake(30), "coords", 0, "float64", 30)
