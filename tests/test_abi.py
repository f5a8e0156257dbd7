"""The C-ABI boundary without a GPU: libfp8attn.so builds, loads and exports every symbol that
include/fp8attn.h declares; argument checks run before any CUDA call; without a
compute-capability-10 device a well-formed call fails loudly (there is no CPU path)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "fp8attn.h")


@pytest.fixture(scope="module")
def fa():
    from paper_2606_06521_b200 import fp8attn
    return fp8attn


def _declared_symbols():
    text = open(HEADER).read()
    return sorted(set(re.findall(r"FP8ATTN_API\s+[\w\s\*]+?\b(fp8attn_\w+)\s*\(", text)))


def test_header_declares_the_expected_calls():
    syms = _declared_symbols()
    for s in ("fp8attn_fwd", "fp8attn_fwd_host", "fp8attn_quantize_e4m3", "fp8attn_strerror", "fp8attn_version"):
        assert s in syms


def test_library_exports_every_declared_symbol(fa):
    lib = C.CDLL(fa.LIB_PATH)
    for s in _declared_symbols():
        assert hasattr(lib, s), s


def test_no_torch_types_in_the_header():
    text = open(HEADER).read()
    assert "torch" not in text.lower() and "at::" not in text


def test_stats_struct_layout_matches_header(fa):
    # the library rejects a struct_size that differs from its own sizeof(fp8attn_stats)
    st = fa.Stats()
    st.struct_size = C.sizeof(fa.Stats) + 4
    one = C.c_void_p(16)
    rc = fa.fp8attn_fwd(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, 1.0, 0, 1, C.byref(st))
    assert rc == -8
    assert "struct_size" in fa.fp8attn_strerror(rc)


def test_argument_checks_precede_any_cuda_call(fa):
    one = C.c_void_p(16)
    f = fa.fp8attn_fwd
    assert f(None, one, one, one, 1, 1, 1, 1, 1, 64, 0, 1.0, 0, 1, None) == -1
    assert f(one, one, one, one, 1, 3, 2, 1, 1, 64, 0, 1.0, 0, 1, None) == -2       # Hq % Hkv
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 96, 0, 1.0, 0, 1, None) == -2       # d
    assert f(one, one, one, one, 1, 1, 1, 0, 1, 64, 0, 1.0, 0, 1, None) == -2       # Lq
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, 0.0, 0, 1, None) == -3       # S
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, float("inf"), 0, 1, None) == -3
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, float("nan"), 0, 1, None) == -3
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, 1.0, 3, 1, None) == -4       # kv_order (0, 1, 2 exist)
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, 1.0, 0, 3, None) == -4       # mode
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, 1.0, 0, 2, None) == -4       # FP8 mode, FP32 dtype
    assert f(one, one, one, one, 1, 1, 1, 1, 1, 128, 0, 1.0, 0, 2 | (2 << 8), None) == -1   # no scales
    for code in range(-8, 1):
        assert fa.fp8attn_strerror(code) != "unknown error code"
    assert fa.fp8attn_version() >= 100


def test_no_cpu_fallback(fa):
    """Without a CC-10 device a valid call returns FP8ATTN_E_DEVICE: nothing is computed on the host."""
    import torch
    if torch.cuda.is_available() and torch.cuda.get_device_capability()[0] == 10:
        pytest.skip("a B200 is present")
    one = C.c_void_p(16)
    assert fa.fp8attn_fwd(one, one, one, one, 1, 1, 1, 1, 1, 64, 0, 1.0, 0, 1, None) == -6
    assert fa.fp8attn_quantize_e4m3(one, one, one, 1, 1, 1, 1, None) == -6


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_06521_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), f
                assert "fp8attn_oracle" not in src, f
    orc = os.path.join(ROOT, "oracle")
    for f in os.listdir(orc):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(orc, f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_06521_b200\b", src, re.M), f
