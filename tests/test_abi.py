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
    for code in range(-9, 1):
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


def test_stats_struct_fields_follow_the_header(fa):
    """The ctypes mirror of fp8attn_stats lists the header's fields in the header's order (a field added on one side
    only would shift every later field)."""
    text = open(HEADER).read()
    body = text[text.index("typedef struct fp8attn_stats {") + len("typedef struct fp8attn_stats {"):text.index("} fp8attn_stats;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl or decl.startswith("typedef"):
            continue
        for part in decl.split(","):
            m = re.search(r"(\w+)\s*(\[[^\]]*\])?\s*$", part.strip())
            names.append(m.group(1))
    assert names == [n for n, _ in fa.Stats._fields_], (names, [n for n, _ in fa.Stats._fields_])


def test_new_options_are_validated_before_any_cuda_call(fa):
    one = C.c_void_p(16)
    st = fa.Stats()
    st.struct_size = C.sizeof(fa.Stats)
    call = lambda: fa.fp8attn_fwd(one, one, one, one, 1, 1, 1, 8, 8, 64, 0, 1.0, 0, 1 | fa.DTYPE_BF16, C.byref(st))
    st.scale_mode = 2
    assert call() == -4
    st.scale_mode, st.o_dtype = 0, 3
    assert call() == -4
    st.o_dtype = 0
    bad = (C.c_int32 * 2)(5, 3)                     # not ascending
    st.sink_pos, st.n_sink = C.cast(bad, C.c_void_p), 2
    assert call() == -2
    ok = (C.c_int32 * 2)(3, 9)                      # past the last key
    st.sink_pos = C.cast(ok, C.c_void_p)
    assert call() == -2
    st.sink_pos, st.n_sink = None, 4
    st.block_table, st.page_size, st.max_pages, st.num_pages = 16, 4, 1, 1      # table does not reach Lk = 8
    assert call() == -2
    st.block_table = None
    st.scale_mode = 1                               # the dynamic scale needs a cast: not in the no-cast mode
    assert fa.fp8attn_fwd(one, one, one, one, 1, 1, 1, 8, 8, 64, 0, 1.0, 0, 0 | fa.DTYPE_BF16, C.byref(st)) == -4
