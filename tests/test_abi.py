"""The C-ABI shared library builds here (nvcc cross-compiles sm_100a without a GPU), loads, and exports
every symbol include/nnp.h declares.  No compute call is made (no GPU in this container)."""
import ctypes
import os
import re

import pytest

from paper_2201_08110_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_functions():
    src = open(os.path.join(ROOT, "include", "nnp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nnp_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    build.build_cuda()
    return ctypes.CDLL(binding.LIB_PATH)


def test_header_declares_the_boundary():
    names = _header_functions()
    for required in ("nnp_create", "nnp_compute", "nnp_status", "nnp_destroy", "nnp_error_string"):
        assert required in names
    assert sorted(binding.SYMBOLS) == names  # the binding wraps exactly what the header declares


def test_library_exports_every_declared_symbol(lib):
    for name in _header_functions():
        assert hasattr(lib, name), f"libnnp_b200.so does not export {name}"


def test_error_strings_and_null_handles(lib):
    lib.nnp_error_string.restype = ctypes.c_char_p
    assert lib.nnp_error_string(0) == b"ok"
    assert b"capacity" in lib.nnp_error_string(-4)
    # argument validation happens before any CUDA call
    assert lib.nnp_create(None, None, 0, None, 1, None) == -1
    assert lib.nnp_status(None) == -1
    assert lib.nnp_launches_per_compute(None) == 0
    lib.nnp_destroy(None)


def test_no_signature_mentions_torch_or_cxx_types():
    src = open(os.path.join(ROOT, "include", "nnp.h")).read()
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)  # declarations only: comments may say "PyTorch"
    for token in ("torch", "at::", "c10::", "std::", "Tensor", "cudaStream_t", "template", "class "):
        assert token not in code, f"include/nnp.h declares something with {token!r}"
    assert 'extern "C"' in src


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "missing.so"))
    monkeypatch.setattr(binding, "_lib", None)
    with pytest.raises(FileNotFoundError):
        binding.load_library()
