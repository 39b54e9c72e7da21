"""CPU-only checks of the C-ABI boundary: libmkv.so loads without a GPU, exports every symbol
include/mkv.h declares, and fails loudly (no CPU fallback) when no device is present."""
import ctypes
import os
import re

import pytest

import __graft_entry__  # noqa: F401  (builds the library if needed)

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mkv.h")


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"MKV_API\s+[\w\s\*]+?\b(mkv_\w+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    syms = declared_symbols()
    for name in ("mkv_cache_create", "mkv_cache_free", "mkv_compress_segment", "mkv_select",
                 "mkv_packed_attention"):
        assert name in syms
    assert len(syms) >= 16


def test_library_exports_every_declared_symbol():
    __graft_entry__.build()
    from paper_2607_00760_b200 import binding
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(lib, name), f"libmkv.so does not export {name}"
    assert sorted(binding.SYMBOLS) == declared_symbols()
    assert binding.mkv_version() == 2


def test_no_torch_types_in_the_boundary():
    text = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    assert "torch" not in text.lower() and "at::" not in text and "#include <cuda" not in text


def test_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2607_00760_b200 import binding
    with pytest.raises(binding.MkvError):
        binding.mkv_cache_create(1, 1, 2, 8, 128, 4096, 64)
    assert binding.mkv_last_error() != ""


def test_create_rejects_a_nonzero_reserved_field():
    """mkv_cache_desc.reserved must be 0 (include/mkv.h): checked on the host before any CUDA call"""
    from paper_2607_00760_b200 import binding
    desc = binding.mkv_cache_desc(1, 1, 2, 8, 128, 4096, 64, 0, 0, 8, 1)
    h = ctypes.c_void_p()
    assert binding._lib.mkv_cache_create(ctypes.byref(desc), ctypes.byref(h)) == binding.MKV_E_ARG
    assert "reserved" in binding.mkv_last_error() and not h.value


def test_trace_build_is_a_separate_library():
    """-DMKV_TRACE (paper_2607_00760_b200/trace.py) goes into libmkv_trace.so: the product library carries neither the
    stamps' reader nor anything else the header does not declare"""
    from paper_2607_00760_b200 import build as mkv_build
    lib = ctypes.CDLL(mkv_build.build())
    assert not hasattr(lib, "mkv_trace_read")
    trace = ctypes.CDLL(mkv_build.build(trace=True))
    assert hasattr(trace, "mkv_trace_read")
    for name in declared_symbols():
        assert hasattr(trace, name), name


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_00760_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "mkv_oracle" not in src, f
    orc_dir = os.path.join(ROOT, "oracle")
    for f in os.listdir(orc_dir):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(orc_dir, f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2607", src, flags=re.M), f
            assert '#include "mkv.h"' not in src and "mkv_internal" not in src, f
