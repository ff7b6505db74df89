"""CPU-side checks of the boundary: the shared library builds/loads, exports every symbol that
include/nvfp4.h declares, and validates arguments before touching CUDA (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_13233_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "nvfp4.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:nvfp4|reset_sampler)_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 11
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/nvfp4.h but not exported"


def test_binding_lists_every_symbol():
    from paper_2606_13233_b200 import binding
    assert sorted(binding.SYMBOLS) == declared_symbols()


def test_version_and_sizes(lib):
    assert lib.nvfp4_version() == 2
    lib.nvfp4_repacked_bytes.restype = ctypes.c_size_t
    # exactly the information of the canonical pair (+ the 128-byte versioned header) when N % 32 == 0 and K % 256 == 0
    for N, K in [(2048, 2048), (10240, 5120), (5120, 8192), (51200, 5120), (5120, 25600)]:
        assert lib.nvfp4_repacked_bytes(N, K) == 128 + N * K // 2 + N * K // 16
    # ragged shapes: whole 4608-byte cells, never less than the canonical information, bounded padding
    for N, K in [(33, 144), (100, 208), (1, 16), (1000, 2576)]:
        b = lib.nvfp4_repacked_bytes(N, K)
        assert (b - 128) % 4608 == 0 and b - 128 >= N * K * 9 // 16
        assert b - 128 <= (N + 31) * ((K + 255) // 256 * 256 * 1.04) * 9 / 16 + 4608
    assert lib.nvfp4_repacked_bytes(0, 128) == 0
    assert lib.nvfp4_repacked_bytes(32, 24) == 0          # K % 16 != 0


def test_argument_validation_without_gpu(lib):
    vp = ctypes.c_void_p
    lib.nvfp4_quantize_act.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int64, vp, vp, vp, ctypes.c_int,
                                       vp, ctypes.c_size_t, vp]
    assert lib.nvfp4_quantize_act(None, 1, 64, 64, None, None, None, 0, None, 0, None) == -1
    fake = vp(0x1000)                                       # never dereferenced: validation fails first
    assert lib.nvfp4_quantize_act(fake, 9, 64, 64, fake, fake, fake, 0, None, 0, None) == -2   # M > 8
    assert lib.nvfp4_quantize_act(fake, 1, 40, 40, fake, fake, fake, 0, None, 0, None) == -2   # K % 16
    assert lib.nvfp4_quantize_act(fake, 1, 64, 64, fake, fake, fake, 7, None, 0, None) == -1   # bad mode
    assert lib.nvfp4_quantize_act(vp(0x1008), 1, 64, 64, fake, fake, fake, 0, None, 0, None) == -3
    lib.nvfp4_gemv.argtypes = [ctypes.c_int, vp, vp, ctypes.c_int, ctypes.c_int, vp, vp, vp, ctypes.c_int,
                               ctypes.c_int64, vp, ctypes.c_int, ctypes.c_int64, vp, ctypes.c_size_t, vp]
    assert lib.nvfp4_gemv(5, fake, fake, 32, 128, fake, fake, fake, 1, 64, fake, 0, 32, None, 0, None) == -1
    assert lib.nvfp4_gemv(0, fake, fake, 32, 128, fake, None, fake, 1, 64, fake, 0, 32, None, 0, None) == -1
    assert lib.nvfp4_gemv(0, fake, fake, 32, 128, fake, fake, fake, 0, 64, fake, 0, 32, None, 0, None) == -2
    assert lib.nvfp4_gemv(0, fake, fake, 32, 128, fake, fake, fake, 1, 64, fake, 0, 16, None, 0, None) == -2  # ldy < N


def test_config_table_is_sane(lib):
    ip = ctypes.POINTER(ctypes.c_int)
    lib.nvfp4_gemv_get_config.argtypes = [ctypes.c_int] * 4 + [ip] * 6
    lib.nvfp4_gemv_workspace_bytes.restype = ctypes.c_size_t
    for N, K in [(2048, 2048), (10240, 5120), (5120, 8192), (51200, 5120), (5120, 25600), (1, 16), (100, 208)]:
        for M in range(1, 9):
            for mode in (0, 1):
                v = [ctypes.c_int(0) for _ in range(6)]
                assert lib.nvfp4_gemv_get_config(mode, M, N, K, *[ctypes.byref(a) for a in v]) == 0
                ks, warps, rows, stages, cps, bal = [a.value for a in v]
                assert 1 <= ks <= (K + 255) // 256 and 1 <= warps <= 20 and rows in (1, 2) and 1 <= stages <= 16 and 1 <= cps <= 3 and bal in (1, 2)
            assert lib.nvfp4_gemv_workspace_bytes(M, N, K) > 0
    assert lib.nvfp4_gemv_set_config(0, 0, 3, 0, 0, 0) == -1
    assert lib.nvfp4_gemv_set_config(0, 0, 4, 0, 0, 0) == -1 and lib.nvfp4_gemv_set_config(0, 0, 0, 0, 4, 0) == -1
    assert lib.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 3) == -1
    assert lib.nvfp4_set_layout_kparts(3) == -1 and lib.nvfp4_set_layout_kparts(64) == -1
    assert lib.nvfp4_set_layout_kparts(4) == 0 and lib.nvfp4_get_layout_kparts(5120, 5120) == 4
    assert lib.nvfp4_set_layout_kparts(0) == 0 and lib.nvfp4_get_layout_kparts(5120, 25600) == 4
    assert lib.nvfp4_get_layout_kparts(51200, 5120) == 1
    assert lib.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0) == 0


def test_gemm_sizes_and_validation_without_gpu(lib):
    vp, ci, cs = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
    lib.nvfp4_gemm_repacked_bytes.restype = cs
    lib.nvfp4_gemm_workspace_bytes.restype = cs
    lib.nvfp4_gemm_packed_act_bytes.restype = cs
    lib.nvfp4_gemm_packed_workspace_bytes.restype = cs
    # 128-row tiles x 256-k stages of 18432 B behind the 128-byte header: the canonical information when N % 128 == 0
    for N, K in [(10240, 5120), (5120, 8192), (51200, 5120), (5120, 25600), (2048, 2048)]:
        assert lib.nvfp4_gemm_repacked_bytes(N, K) == 128 + N * K // 2 + N * K // 16
    assert lib.nvfp4_gemm_repacked_bytes(130, 512) == 128 + 2 * 2 * 18432
    assert lib.nvfp4_gemm_repacked_bytes(128, 384) == 0 and lib.nvfp4_gemm_repacked_bytes(0, 256) == 0
    # packed activations: per 256 k one record of MT*128 code bytes + 2048 scale bytes, MT = 8, 16, 32, 64, 128 >= M
    for M, MT in [(1, 8), (8, 8), (9, 16), (17, 32), (33, 64), (65, 128), (128, 128)]:
        assert lib.nvfp4_gemm_packed_act_bytes(M, 5120) == 20 * (MT * 128 + 2048)
    assert lib.nvfp4_gemm_packed_act_bytes(129, 5120) == 0 and lib.nvfp4_gemm_packed_act_bytes(1, 100) == 0
    assert lib.nvfp4_gemm_workspace_bytes(300, 5120, 8192) >= lib.nvfp4_gemm_packed_workspace_bytes(128, 5120, 8192)
    fake = vp(0x1000)
    lib.nvfp4_gemm.argtypes = [vp, vp, ci, ci, vp, vp, vp, ci, ci, ctypes.c_int64, vp, ci, ctypes.c_int64, vp, cs, vp]
    assert lib.nvfp4_gemm(None, fake, 128, 256, fake, fake, fake, 0, 1, 128, fake, 0, 128, fake, 1 << 30, None) == -1
    assert lib.nvfp4_gemm(fake, fake, 128, 384, fake, fake, fake, 0, 1, 192, fake, 0, 128, fake, 1 << 30, None) == -2
    assert lib.nvfp4_gemm(fake, fake, 128, 256, fake, fake, fake, 0, 1, 128, fake, 0, 64, fake, 1 << 30, None) == -2   # ldy < N
    assert lib.nvfp4_gemm(fake, fake, 128, 256, fake, fake, fake, 0, 1, 128, fake, 0, 128, fake, 16, None) == -1       # workspace
    assert lib.nvfp4_gemm(vp(0x1004), fake, 128, 256, fake, fake, fake, 0, 1, 128, fake, 0, 128, fake, 1 << 30, None) == -3
    lib.nvfp4_gemm_set_config.argtypes = [ci, ci]
    assert lib.nvfp4_gemm_set_config(99, 0) == -1 and lib.nvfp4_gemm_set_config(0, 0) == 0
