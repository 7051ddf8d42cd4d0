"""CPU-only checks of the C-ABI boundary: the library builds, loads, exports every symbol the
header declares, and its host-side helpers / argument validation behave (no kernel runs)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "fourtune.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2607_05711_b200 import build
    path = build.build()
    return C.CDLL(path)


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ft_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_four_entry_points():
    syms = declared_symbols()
    for name in ("ft_quantize_blockwise", "ft_linear_fwd", "ft_linear_bwd_dgrad", "ft_lora_wgrad"):
        assert name in syms


def test_every_declared_symbol_is_exported(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_sf_bytes_and_workspace(lib):
    lib.ft_sf_bytes.restype = C.c_size_t
    lib.ft_sf_bytes.argtypes = [C.c_int64, C.c_int64, C.c_int32, C.c_int32]
    # row-major: one byte per block
    assert lib.ft_sf_bytes(256, 3072, 1, 0) == 256 * 192
    assert lib.ft_sf_bytes(3072, 3072, 16, 0) == 192 * 192
    # tiled: rows padded to 128, blocks to 4, 512 bytes per tile
    assert lib.ft_sf_bytes(256, 3072, 1, 1) == 2 * 48 * 512
    assert lib.ft_sf_bytes(130, 64, 1, 1) == 2 * 1 * 512
    assert lib.ft_sf_bytes(4608, 9216, 1, 1) == 36 * 144 * 512
    lib.ft_workspace_bytes.restype = C.c_size_t
    lib.ft_workspace_bytes.argtypes = [C.c_int64, C.c_int64, C.c_int64, C.c_int32]
    assert lib.ft_workspace_bytes(4608, 3072, 9216, 64) >= 256 + 4608 * 64 * 2


def test_error_strings(lib):
    lib.ft_error_string.restype = C.c_char_p
    seen = {lib.ft_error_string(c) for c in (0, -1, -2, -3, -4, -5)}
    assert len(seen) == 6 and lib.ft_error_string(0) == b"ok"
    assert lib.ft_version() >= 100


def test_argument_validation_needs_no_gpu(lib):
    # NULL pointers are rejected on the host before any CUDA call
    vp = C.c_void_p
    lib.ft_tensor_amax.argtypes = [vp, C.c_int64, vp, vp]
    assert lib.ft_tensor_amax(None, 16, None, None) == -1
    lib.ft_quantize_blockwise.argtypes = [vp, C.c_int64, C.c_int64, vp, vp, vp, C.c_int32, C.c_uint64, C.c_uint64, vp,
                                          C.c_size_t, vp]
    assert lib.ft_quantize_blockwise(None, 128, 64, None, None, None, 0, 0, 0, None, 0, None) == -1
    lib.ft_linear_fwd.argtypes = [vp, vp, C.c_int64, vp, vp, vp, vp, C.c_size_t, vp]
    assert lib.ft_linear_fwd(None, None, 1, None, None, None, None, 0, None) == -1
    assert lib.ft_debug_set_gemm_tile_n(100) == -1 and lib.ft_debug_set_gemm_tile_n(0) == 0


def test_binding_fails_loudly_without_library(monkeypatch):
    from paper_2607_05711_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libfourtune.so")
    with pytest.raises(binding.FtError):
        binding.lib()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2607_05711_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
