"""ctypes binding of the C ABI in include/nvfp4.h -- argument marshalling only.

Every function takes torch CUDA tensors (device memory + the current stream are all PyTorch
is used for), checks nothing the library does not check itself, and raises `Nvfp4Error` on a
non-zero status.  There is NO fallback: if the shared library is missing, importing this module
raises, and if no CUDA device is usable every compute call fails with NVFP4_ERR_CUDA.
"""
from __future__ import annotations

import ctypes
import os

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libnvfp4_b200.so")

MODE_W4A4, MODE_W4A16 = 0, 1
DTYPE_F32, DTYPE_BF16 = 0, 1
GSCALE_DYNAMIC, GSCALE_STATIC, GSCALE_DYNAMIC_PER_ROW = 0, 1, 2
ERR_NAMES = {0: "NVFP4_OK", -1: "NVFP4_ERR_INVALID_ARG", -2: "NVFP4_ERR_UNSUPPORTED_SHAPE",
             -3: "NVFP4_ERR_ALIGNMENT", -4: "NVFP4_ERR_CUDA"}

# every symbol include/nvfp4.h declares (tests check that the library exports all of them)
SYMBOLS = ("nvfp4_version", "nvfp4_last_cuda_error", "nvfp4_quantize_act", "nvfp4_repacked_bytes",
           "nvfp4_repack_weight", "nvfp4_unpack_weight", "nvfp4_gemv_workspace_bytes", "nvfp4_gemv",
           "nvfp4_gemv_set_config", "nvfp4_gemv_get_config", "nvfp4_silu_mul", "nvfp4_gemv_fused_quant",
           "nvfp4_gemv_rowscale", "nvfp4_set_layout_kparts", "nvfp4_get_layout_kparts", "nvfp4_silu_mul_quantize",
           "reset_sampler_state_bytes", "reset_sampler_step", "nvfp4_linear", "nvfp4_linear_workspace_bytes",
           "nvfp4_gemm_repacked_bytes", "nvfp4_gemm_repack_weight", "nvfp4_gemm_unpack_weight",
           "nvfp4_gemm_workspace_bytes", "nvfp4_gemm", "nvfp4_gemm_packed_act_bytes", "nvfp4_gemm_pack_act",
           "nvfp4_quantize_act_packed", "nvfp4_silu_mul_quantize_packed", "nvfp4_gemm_packed_workspace_bytes",
           "nvfp4_gemm_packed", "nvfp4_gemm_set_config", "nvfp4_gemv_noalloc", "nvfp4_gemm_packed_quant_out",
           "nvfp4_gemm_w4a16", "nvfp4_gemm_w4a16_workspace_bytes", "nvfp4_gemm_repack_weight_gate_up",
           "nvfp4_gemm_unpack_weight_gate_up", "nvfp4_gemm_packed_silu_quant_out", "nvfp4_gemv_xrecord_bytes",
           "nvfp4_quantize_act_records", "nvfp4_gemv_records", "nvfp4_silu_mul_quantize_records")


class Nvfp4Error(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = status
        super().__init__(f"{ERR_NAMES.get(status, status)} {detail}".strip())


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2606_13233_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    c_int, c_i64, c_sz, vp = ctypes.c_int, ctypes.c_int64, ctypes.c_size_t, ctypes.c_void_p
    lib.nvfp4_version.restype = c_int
    lib.nvfp4_version.argtypes = []
    lib.nvfp4_last_cuda_error.restype = ctypes.c_char_p
    lib.nvfp4_last_cuda_error.argtypes = []
    lib.nvfp4_quantize_act.restype = c_int
    lib.nvfp4_quantize_act.argtypes = [vp, c_int, c_int, c_i64, vp, vp, vp, c_int, vp, c_sz, vp]
    lib.nvfp4_repacked_bytes.restype = c_sz
    lib.nvfp4_repacked_bytes.argtypes = [c_int, c_int]
    lib.nvfp4_repack_weight.restype = c_int
    lib.nvfp4_repack_weight.argtypes = [vp, vp, c_int, c_int, vp, vp]
    lib.nvfp4_unpack_weight.restype = c_int
    lib.nvfp4_unpack_weight.argtypes = [vp, c_int, c_int, vp, vp, vp]
    lib.nvfp4_gemv_workspace_bytes.restype = c_sz
    lib.nvfp4_gemv_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.nvfp4_gemv.restype = c_int
    lib.nvfp4_gemv.argtypes = [c_int, vp, vp, c_int, c_int, vp, vp, vp, c_int, c_i64, vp, c_int, c_i64,
                               vp, c_sz, vp]
    lib.nvfp4_linear_workspace_bytes.restype = c_sz
    lib.nvfp4_linear_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.nvfp4_linear.restype = c_int
    lib.nvfp4_linear.argtypes = [c_int, vp, vp, c_int, c_int, vp, vp, vp, c_int, c_i64, vp, c_int, c_i64, vp, c_sz, vp]
    lib.nvfp4_gemv_rowscale.restype = c_int
    lib.nvfp4_gemv_rowscale.argtypes = [vp, vp, c_int, c_int, vp, vp, vp, c_int, c_i64, vp, c_int, c_i64, vp, c_sz, vp]
    lib.nvfp4_set_layout_kparts.restype = c_int
    lib.nvfp4_set_layout_kparts.argtypes = [c_int]
    lib.nvfp4_get_layout_kparts.restype = c_int
    lib.nvfp4_get_layout_kparts.argtypes = [c_int, c_int]
    lib.nvfp4_gemv_xrecord_bytes.restype = c_sz
    lib.nvfp4_gemv_xrecord_bytes.argtypes = [c_int, c_int]
    lib.nvfp4_quantize_act_records.restype = c_int
    lib.nvfp4_quantize_act_records.argtypes = [vp, c_int, c_int, c_i64, vp, vp, c_int, vp]
    lib.nvfp4_silu_mul_quantize_records.restype = c_int
    lib.nvfp4_silu_mul_quantize_records.argtypes = [vp, c_int, c_int, vp, vp, c_int, vp, vp]
    lib.nvfp4_gemv_records.restype = c_int
    lib.nvfp4_gemv_records.argtypes = [vp, vp, c_int, c_int, vp, vp, c_int, vp, c_int, c_i64, vp, c_sz, vp]
    lib.nvfp4_gemv_fused_quant.restype = c_int
    lib.nvfp4_gemv_fused_quant.argtypes = [vp, vp, c_int, c_int, vp, c_int, c_i64, vp, vp, c_int, c_i64, vp, c_sz, vp]
    lib.nvfp4_gemv_set_config.restype = c_int
    lib.nvfp4_gemv_set_config.argtypes = [c_int, c_int, c_int, c_int, c_int, c_int]
    lib.nvfp4_gemv_get_config.restype = c_int
    lib.nvfp4_gemv_get_config.argtypes = [c_int, c_int, c_int, c_int] + [ctypes.POINTER(c_int)] * 6
    lib.nvfp4_silu_mul_quantize.restype = c_int
    lib.nvfp4_silu_mul_quantize.argtypes = [vp, c_int, c_int, vp, vp, vp, c_int, vp, vp]
    lib.reset_sampler_state_bytes.restype = c_sz
    lib.reset_sampler_state_bytes.argtypes = []
    lib.reset_sampler_step.restype = c_int
    lib.reset_sampler_step.argtypes = [vp, c_int, c_int, c_int, c_i64, vp, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                       ctypes.c_float, c_int, c_int, ctypes.c_uint64, vp, vp, vp]
    lib.nvfp4_silu_mul.restype = c_int
    lib.nvfp4_silu_mul.argtypes = [vp, c_int, c_int, vp, vp]
    lib.nvfp4_gemm_repacked_bytes.restype = c_sz
    lib.nvfp4_gemm_repacked_bytes.argtypes = [c_int, c_int]
    lib.nvfp4_gemm_repack_weight.restype = c_int
    lib.nvfp4_gemm_repack_weight.argtypes = [vp, vp, c_int, c_int, vp, vp]
    lib.nvfp4_gemm_unpack_weight.restype = c_int
    lib.nvfp4_gemm_unpack_weight.argtypes = [vp, c_int, c_int, vp, vp, vp]
    lib.nvfp4_gemm_workspace_bytes.restype = c_sz
    lib.nvfp4_gemm_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.nvfp4_gemm.restype = c_int
    lib.nvfp4_gemm.argtypes = [vp, vp, c_int, c_int, vp, vp, vp, c_int, c_int, c_i64, vp, c_int, c_i64, vp, c_sz, vp]
    lib.nvfp4_gemm_packed_act_bytes.restype = c_sz
    lib.nvfp4_gemm_packed_act_bytes.argtypes = [c_int, c_int]
    lib.nvfp4_gemm_pack_act.restype = c_int
    lib.nvfp4_gemm_pack_act.argtypes = [vp, vp, c_int, c_int, c_i64, vp, vp]
    lib.nvfp4_quantize_act_packed.restype = c_int
    lib.nvfp4_quantize_act_packed.argtypes = [vp, c_int, c_int, c_i64, vp, vp, c_int, vp]
    lib.nvfp4_silu_mul_quantize_packed.restype = c_int
    lib.nvfp4_silu_mul_quantize_packed.argtypes = [vp, c_int, c_int, vp, vp, c_int, vp, vp]
    lib.nvfp4_gemm_packed_workspace_bytes.restype = c_sz
    lib.nvfp4_gemm_packed_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.nvfp4_gemm_packed_quant_out.restype = c_int
    lib.nvfp4_gemm_packed_quant_out.argtypes = [vp, vp, c_int, c_int, vp, vp, c_int, c_int, vp, c_int, c_i64, vp, vp, c_int,
                                                vp, c_sz, vp]
    lib.nvfp4_gemm_w4a16_workspace_bytes.restype = c_sz
    lib.nvfp4_gemm_w4a16_workspace_bytes.argtypes = [c_int, c_int, c_int]
    lib.nvfp4_gemm_w4a16.restype = c_int
    lib.nvfp4_gemm_w4a16.argtypes = [vp, vp, c_int, c_int, vp, c_int, c_i64, vp, c_int, c_i64, vp, c_sz, vp]
    lib.nvfp4_gemm_repack_weight_gate_up.restype = c_int
    lib.nvfp4_gemm_repack_weight_gate_up.argtypes = [vp, vp, c_int, c_int, vp, vp]
    lib.nvfp4_gemm_unpack_weight_gate_up.restype = c_int
    lib.nvfp4_gemm_unpack_weight_gate_up.argtypes = [vp, c_int, c_int, vp, vp, vp]
    lib.nvfp4_gemm_packed_silu_quant_out.restype = c_int
    lib.nvfp4_gemm_packed_silu_quant_out.argtypes = [vp, vp, c_int, c_int, vp, vp, c_int, c_int, vp, c_int, c_i64, vp, vp, vp, c_sz, vp]
    lib.nvfp4_gemv_noalloc.restype = c_int
    lib.nvfp4_gemv_noalloc.argtypes = [c_int, vp, vp, c_int, c_int, vp, vp, vp, c_int, c_i64, vp, c_int, c_i64, vp]
    lib.nvfp4_gemm_set_config.restype = c_int
    lib.nvfp4_gemm_set_config.argtypes = [c_int, c_int]
    lib.nvfp4_gemm_packed.restype = c_int
    lib.nvfp4_gemm_packed.argtypes = [vp, vp, c_int, c_int, vp, vp, c_int, c_int, vp, c_int, c_i64, vp, c_sz, vp]
    return lib


lib = _load()


def _check(status):
    if status != 0:
        raise Nvfp4Error(status, lib.nvfp4_last_cuda_error().decode())


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


def nvfp4_version() -> int:
    return lib.nvfp4_version()


def nvfp4_quantize_act(x_bf16, codes=None, scales=None, gscale=None, gscale_mode=GSCALE_DYNAMIC):
    """x_bf16 [M,K] torch.bfloat16 (row stride = x.stride(0)) -> (codes u8 [M,K/2], scales u8 [M,K/16], g f32 [1])."""
    M, K = x_bf16.shape
    dev = x_bf16.device
    if codes is None:
        codes = torch.empty((M, K // 2), dtype=torch.uint8, device=dev)
    if scales is None:
        scales = torch.empty((M, K // 16), dtype=torch.uint8, device=dev)
    if gscale is None:
        gscale = torch.zeros(M if gscale_mode == GSCALE_DYNAMIC_PER_ROW else 1, dtype=torch.float32, device=dev)
    _check(lib.nvfp4_quantize_act(_ptr(x_bf16), M, K, x_bf16.stride(0), _ptr(codes), _ptr(scales), _ptr(gscale),
                                  gscale_mode, None, 0, _stream()))
    return codes, scales, gscale


def nvfp4_repacked_bytes(N, K) -> int:
    return lib.nvfp4_repacked_bytes(N, K)


def nvfp4_repack_weight(codes, scales, blob=None):
    N, K = codes.shape[0], codes.shape[1] * 2
    if blob is None:
        blob = torch.empty(nvfp4_repacked_bytes(N, K), dtype=torch.uint8, device=codes.device)
    _check(lib.nvfp4_repack_weight(_ptr(codes), _ptr(scales), N, K, _ptr(blob), _stream()))
    return blob


def nvfp4_unpack_weight(blob, N, K):
    codes = torch.empty((N, K // 2), dtype=torch.uint8, device=blob.device)
    scales = torch.empty((N, K // 16), dtype=torch.uint8, device=blob.device)
    _check(lib.nvfp4_unpack_weight(_ptr(blob), N, K, _ptr(codes), _ptr(scales), _stream()))
    return codes, scales


def nvfp4_gemv_workspace_bytes(M, N, K) -> int:
    return lib.nvfp4_gemv_workspace_bytes(M, N, K)


def new_workspace(M, N, K, device="cuda"):
    """zero-filled workspace (the ABI requires zero fill before first use)."""
    return torch.zeros(max(16, nvfp4_gemv_workspace_bytes(M, N, K)), dtype=torch.uint8, device=device)


def nvfp4_gemv(mode, w_blob, w_gscale, N, K, x, x_scales=None, x_gscale=None, y=None, y_dtype=DTYPE_BF16,
               workspace=None):
    """W4A4: x = codes u8 [M,K/2]; W4A16: x = bf16 [M,K].  Returns y [M,N] (f32 or bf16)."""
    M = x.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x.device)
    if workspace is None:
        workspace = new_workspace(M, N, K, x.device)
    _check(lib.nvfp4_gemv(mode, _ptr(w_blob), _ptr(w_gscale), N, K, _ptr(x), _ptr(x_scales), _ptr(x_gscale), M,
                          x.stride(0), _ptr(y), y_dtype, y.stride(0), _ptr(workspace), workspace.numel(), _stream()))
    return y


def nvfp4_linear(mode, w_blob, w_gscale, N, K, x, x_scales=None, x_gscale=None, y=None, y_dtype=DTYPE_BF16, workspace=None):
    """any M: ceil(M/8) GEMV passes over 8-row chunks (see include/nvfp4.h)."""
    M = x.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x.device)
    if workspace is None:
        workspace = torch.zeros(max(16, lib.nvfp4_linear_workspace_bytes(M, N, K)), dtype=torch.uint8, device=x.device)
    _check(lib.nvfp4_linear(mode, _ptr(w_blob), _ptr(w_gscale), N, K, _ptr(x), _ptr(x_scales), _ptr(x_gscale), M,
                            x.stride(0), _ptr(y), y_dtype, y.stride(0), _ptr(workspace), workspace.numel(), _stream()))
    return y


def nvfp4_gemm_repack_weight(codes, scales):
    """canonical codes u8 [N,K/2] + scales u8 [N,K/16] (device) -> tensor-core blob (u8, device)."""
    N, K = codes.shape[0], codes.shape[1] * 2
    nbytes = lib.nvfp4_gemm_repacked_bytes(N, K)
    if nbytes == 0:
        raise Nvfp4Error(-2, f"tensor-core GEMM needs K % 256 == 0 (N={N}, K={K})")
    blob = torch.empty(nbytes, dtype=torch.uint8, device=codes.device)
    _check(lib.nvfp4_gemm_repack_weight(_ptr(codes), _ptr(scales), N, K, _ptr(blob), _stream()))
    return blob


def nvfp4_gemm_unpack_weight(blob, N, K):
    codes = torch.zeros((N, K // 2), dtype=torch.uint8, device=blob.device)
    scales = torch.zeros((N, K // 16), dtype=torch.uint8, device=blob.device)
    _check(lib.nvfp4_gemm_unpack_weight(_ptr(blob), N, K, _ptr(codes), _ptr(scales), _stream()))
    return codes, scales


def nvfp4_gemm_new_workspace(M, N, K, device):
    return torch.zeros(max(16, lib.nvfp4_gemm_workspace_bytes(M, N, K)), dtype=torch.uint8, device=device)


def nvfp4_gemm(w_blob_tc, w_gscale, N, K, x_codes, x_scales, x_gscale, y=None, y_dtype=DTYPE_BF16, workspace=None,
               gscale_per_row=False):
    """tensor-core W4A4 GEMM, any M >= 1: Y[M,N] = X . W^T (see include/nvfp4.h)."""
    M = x_codes.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x_codes.device)
    if workspace is None:
        workspace = nvfp4_gemm_new_workspace(M, N, K, x_codes.device)
    _check(lib.nvfp4_gemm(_ptr(w_blob_tc), _ptr(w_gscale), N, K, _ptr(x_codes), _ptr(x_scales), _ptr(x_gscale),
                          1 if gscale_per_row else 0, M, x_codes.stride(0), _ptr(y), y_dtype, y.stride(0), _ptr(workspace),
                          workspace.numel(), _stream()))
    return y


def nvfp4_gemm_set_config(stages=0, ctas=0):
    _check(lib.nvfp4_gemm_set_config(stages, ctas))


def nvfp4_gemm_pack_act(x_codes, x_scales, xpack=None):
    """canonical activation codes [M,K/2] / scales [M,K/16] (M <= 128) -> the GEMM's packed records."""
    M, K = x_codes.shape[0], x_codes.shape[1] * 2
    if xpack is None:
        xpack = torch.empty(lib.nvfp4_gemm_packed_act_bytes(M, K), dtype=torch.uint8, device=x_codes.device)
    _check(lib.nvfp4_gemm_pack_act(_ptr(x_codes), _ptr(x_scales), M, K, x_codes.stride(0), _ptr(xpack), _stream()))
    return xpack


def nvfp4_quantize_act_packed(x_bf16, xpack=None, gscale=None, gscale_mode=GSCALE_DYNAMIC):
    """BF16 [M,K] (M <= 128) -> (packed activation records, g f32 [1] or [M])."""
    M, K = x_bf16.shape
    if xpack is None:
        xpack = torch.empty(lib.nvfp4_gemm_packed_act_bytes(M, K), dtype=torch.uint8, device=x_bf16.device)
    if gscale is None:
        gscale = torch.zeros(M if gscale_mode == GSCALE_DYNAMIC_PER_ROW else 1, dtype=torch.float32, device=x_bf16.device)
    _check(lib.nvfp4_quantize_act_packed(_ptr(x_bf16), M, K, x_bf16.stride(0), _ptr(xpack), _ptr(gscale), gscale_mode,
                                         _stream()))
    return xpack, gscale


def nvfp4_silu_mul_quantize_packed(gu_bf16, xpack=None, gscale=None, gscale_mode=GSCALE_DYNAMIC, h_out=None):
    M, I = gu_bf16.shape[0], gu_bf16.shape[1] // 2
    if xpack is None:
        xpack = torch.empty(lib.nvfp4_gemm_packed_act_bytes(M, I), dtype=torch.uint8, device=gu_bf16.device)
    if gscale is None:
        gscale = torch.zeros(M if gscale_mode == GSCALE_DYNAMIC_PER_ROW else 1, dtype=torch.float32, device=gu_bf16.device)
    _check(lib.nvfp4_silu_mul_quantize_packed(_ptr(gu_bf16), M, I, _ptr(xpack), _ptr(gscale), gscale_mode, _ptr(h_out),
                                              _stream()))
    return xpack, gscale


def nvfp4_gemm_packed_new_workspace(M, N, K, device):
    return torch.zeros(max(16, lib.nvfp4_gemm_packed_workspace_bytes(M, N, K)), dtype=torch.uint8, device=device)


def nvfp4_gemm_packed(w_blob_tc, w_gscale, N, K, xpack, x_gscale, M, y=None, y_dtype=DTYPE_BF16, workspace=None,
                      gscale_per_row=False):
    """tensor-core W4A4 GEMM on packed activations (M <= 128)."""
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=xpack.device)
    if workspace is None:
        workspace = nvfp4_gemm_packed_new_workspace(M, N, K, xpack.device)
    _check(lib.nvfp4_gemm_packed(_ptr(w_blob_tc), _ptr(w_gscale), N, K, _ptr(xpack), _ptr(x_gscale),
                                 1 if gscale_per_row else 0, M, _ptr(y), y_dtype, y.stride(0), _ptr(workspace),
                                 workspace.numel(), _stream()))
    return y


def nvfp4_gemm_packed_quant_out(w_blob_tc, w_gscale, N, K, xpack, x_gscale, M, out_gscale, n_quant=None, xpack_out=None, y=None,
                                y_dtype=DTYPE_BF16, workspace=None, gscale_per_row=False):
    """nvfp4_gemm_packed whose epilogue also quantises the first n_quant output columns with the STATIC global scale
    out_gscale into packed records for the next GEMM.  `y` optional (None: only the records are written).
    Returns (xpack_out, y)."""
    n_quant = N if n_quant is None else n_quant
    if xpack_out is None:
        xpack_out = torch.empty(lib.nvfp4_gemm_packed_act_bytes(M, n_quant), dtype=torch.uint8, device=xpack.device)
    if workspace is None:
        workspace = nvfp4_gemm_packed_new_workspace(M, N, K, xpack.device)
    _check(lib.nvfp4_gemm_packed_quant_out(_ptr(w_blob_tc), _ptr(w_gscale), N, K, _ptr(xpack), _ptr(x_gscale),
                                           1 if gscale_per_row else 0, M, _ptr(y), y_dtype, y.stride(0) if y is not None else N,
                                           _ptr(xpack_out), _ptr(out_gscale), n_quant, _ptr(workspace), workspace.numel(),
                                           _stream()))
    return xpack_out, y


def nvfp4_gemm_w4a16(w_blob_tc, w_gscale, N, K, x_bf16, y=None, y_dtype=DTYPE_BF16, workspace=None):
    """tensor-core W4A16 GEMM: NVFP4 weights (tensor-core blob) x BF16 activations [M,K], any M."""
    M = x_bf16.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x_bf16.device)
    if workspace is None:
        workspace = torch.zeros(max(16, lib.nvfp4_gemm_w4a16_workspace_bytes(M, N, K)), dtype=torch.uint8, device=x_bf16.device)
    _check(lib.nvfp4_gemm_w4a16(_ptr(w_blob_tc), _ptr(w_gscale), N, K, _ptr(x_bf16), M, x_bf16.stride(0), _ptr(y), y_dtype,
                                y.stride(0), _ptr(workspace), workspace.numel(), _stream()))
    return y


def nvfp4_gemm_repack_weight_gate_up(codes, scales):
    """fused gate_up weight [2I, K] -> tensor-core blob with gate / up rows interleaved per tile (see include/nvfp4.h)."""
    N, K = codes.shape[0], codes.shape[1] * 2
    blob = torch.empty(lib.nvfp4_gemm_repacked_bytes(N, K), dtype=torch.uint8, device=codes.device)
    _check(lib.nvfp4_gemm_repack_weight_gate_up(_ptr(codes), _ptr(scales), N, K, _ptr(blob), _stream()))
    return blob


def nvfp4_gemm_unpack_weight_gate_up(blob, N, K):
    codes = torch.zeros((N, K // 2), dtype=torch.uint8, device=blob.device)
    scales = torch.zeros((N, K // 16), dtype=torch.uint8, device=blob.device)
    _check(lib.nvfp4_gemm_unpack_weight_gate_up(_ptr(blob), N, K, _ptr(codes), _ptr(scales), _stream()))
    return codes, scales


def nvfp4_gemm_packed_silu_quant_out(w_blob_gate_up, w_gscale, N, K, xpack, x_gscale, M, out_gscale, xpack_out=None, h=None,
                                     h_dtype=DTYPE_BF16, workspace=None, gscale_per_row=False):
    """gate_up GEMM + SiLU*mul + STATIC-scale quantizer in one launch: packed records of h [M, N/2] for the down GEMM."""
    if xpack_out is None:
        xpack_out = torch.empty(lib.nvfp4_gemm_packed_act_bytes(M, N // 2), dtype=torch.uint8, device=xpack.device)
    if workspace is None:
        workspace = nvfp4_gemm_packed_new_workspace(M, N, K, xpack.device)
    _check(lib.nvfp4_gemm_packed_silu_quant_out(_ptr(w_blob_gate_up), _ptr(w_gscale), N, K, _ptr(xpack), _ptr(x_gscale),
                                                1 if gscale_per_row else 0, M, _ptr(h), h_dtype, h.stride(0) if h is not None else N // 2,
                                                _ptr(xpack_out), _ptr(out_gscale), _ptr(workspace), workspace.numel(), _stream()))
    return xpack_out, h


NOALLOC_SCRATCH_BYTES = 4 << 20


def nvfp4_gemv_noalloc(mode, w_blob, w_gscale, N, K, x, x_scales=None, x_gscale=None, y=None, y_dtype=DTYPE_BF16):
    """nvfp4_gemv on the library's built-in scratch array (no workspace argument, nothing allocated by the call; `y` is
    the caller's, pass it in when the caller must not allocate either)."""
    M = x.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x.device)
    _check(lib.nvfp4_gemv_noalloc(mode, _ptr(w_blob), _ptr(w_gscale), N, K, _ptr(x), _ptr(x_scales), _ptr(x_gscale), M,
                                  x.stride(0), _ptr(y), y_dtype, y.stride(0), _stream()))
    return y


def nvfp4_gemv_rowscale(w_blob, w_gscale, N, K, x_codes, x_scales, x_gscales, y=None, y_dtype=DTYPE_BF16, workspace=None):
    """W4A4 GEMV with per-row (per-token) activation global scales x_gscales f32 [M]."""
    M = x_codes.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x_codes.device)
    if workspace is None:
        workspace = new_workspace(M, N, K, x_codes.device)
    _check(lib.nvfp4_gemv_rowscale(_ptr(w_blob), _ptr(w_gscale), N, K, _ptr(x_codes), _ptr(x_scales), _ptr(x_gscales), M,
                                   x_codes.stride(0), _ptr(y), y_dtype, y.stride(0), _ptr(workspace), workspace.numel(),
                                   _stream()))
    return y


def nvfp4_gemv_fused_quant(w_blob, w_gscale, N, K, x_bf16, x_gscale_out=None, y=None, y_dtype=DTYPE_BF16,
                           workspace=None):
    """quantize_act + W4A4 gemv in ONE launch; x_bf16 [M,K] torch.bfloat16.  Returns y [M,N]."""
    M = x_bf16.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=x_bf16.device)
    if workspace is None:
        workspace = new_workspace(M, N, K, x_bf16.device)
    _check(lib.nvfp4_gemv_fused_quant(_ptr(w_blob), _ptr(w_gscale), N, K, _ptr(x_bf16), M, x_bf16.stride(0),
                                      _ptr(x_gscale_out), _ptr(y), y_dtype, y.stride(0), _ptr(workspace),
                                      workspace.numel(), _stream()))
    return y


def nvfp4_new_xrecords(N, K, device):
    """zero-filled record buffer for nvfp4_quantize_act_records / nvfp4_gemv_records on a weight of shape [N, K]."""
    return torch.zeros(lib.nvfp4_gemv_xrecord_bytes(N, K), dtype=torch.uint8, device=device)


def nvfp4_quantize_act_records(x_bf16, xrec, gscale=None, gscale_mode=GSCALE_DYNAMIC):
    """BF16 [1,K] -> the CUDA-core GEMV's activation records (xrec from nvfp4_new_xrecords) and g f32 [1]."""
    M, K = x_bf16.shape
    if gscale is None:
        gscale = torch.zeros(1, dtype=torch.float32, device=xrec.device)
    _check(lib.nvfp4_quantize_act_records(_ptr(x_bf16), M, K, x_bf16.stride(0), _ptr(xrec), _ptr(gscale), gscale_mode, _stream()))
    return xrec, gscale


def nvfp4_silu_mul_quantize_records(gu_bf16, xrec, gscale=None, gscale_mode=GSCALE_DYNAMIC, h=None):
    """BF16 gate_up [1, 2I] -> records of h = silu(gate) * up for nvfp4_gemv_records (and optionally h itself)."""
    M, I = gu_bf16.shape[0], gu_bf16.shape[1] // 2
    if gscale is None:
        gscale = torch.zeros(1, dtype=torch.float32, device=xrec.device)
    _check(lib.nvfp4_silu_mul_quantize_records(_ptr(gu_bf16), M, I, _ptr(xrec), _ptr(gscale), gscale_mode, _ptr(h), _stream()))
    return xrec, gscale


def nvfp4_gemv_records(w_blob, w_gscale, N, K, xrec, x_gscale, M=1, y=None, y_dtype=DTYPE_BF16, workspace=None):
    """W4A4 GEMV at M = 1 on activation records (one bulk copy instead of the load / decode / store staging)."""
    if y is None:
        y = torch.empty((M, N), dtype=torch.float32 if y_dtype == DTYPE_F32 else torch.bfloat16, device=xrec.device)
    if workspace is None:
        workspace = new_workspace(M, N, K, xrec.device)
    _check(lib.nvfp4_gemv_records(_ptr(w_blob), _ptr(w_gscale), N, K, _ptr(xrec), _ptr(x_gscale), M, _ptr(y), y_dtype,
                                  y.stride(0), _ptr(workspace), workspace.numel(), _stream()))
    return y


def nvfp4_gemv_set_config(ksplit=0, warps=0, rows=0, stages=0, ctas_per_sm=0, balance=0):
    _check(lib.nvfp4_gemv_set_config(ksplit, warps, rows, stages, ctas_per_sm, balance))


def nvfp4_gemv_get_config(mode, M, N, K):
    v = [ctypes.c_int(0) for _ in range(6)]
    _check(lib.nvfp4_gemv_get_config(mode, M, N, K, *[ctypes.byref(a) for a in v]))
    return dict(ksplit=v[0].value, warps=v[1].value, rows=v[2].value, stages=v[3].value, ctas_per_sm=v[4].value, balance=v[5].value)


def nvfp4_set_layout_kparts(kparts=0):
    _check(lib.nvfp4_set_layout_kparts(kparts))


def nvfp4_get_layout_kparts(N, K) -> int:
    return lib.nvfp4_get_layout_kparts(N, K)


def nvfp4_silu_mul_quantize(gu_bf16, codes=None, scales=None, gscale=None, gscale_mode=GSCALE_DYNAMIC, h=None):
    """gu_bf16 [M,2I] -> NVFP4 of h = RN_bf16(silu(gate) * up) in one launch: (codes [M,I/2], scales [M,I/16], g)."""
    M, I2 = gu_bf16.shape
    I = I2 // 2
    dev = gu_bf16.device
    if codes is None:
        codes = torch.empty((M, I // 2), dtype=torch.uint8, device=dev)
    if scales is None:
        scales = torch.empty((M, I // 16), dtype=torch.uint8, device=dev)
    if gscale is None:
        gscale = torch.zeros(M if gscale_mode == GSCALE_DYNAMIC_PER_ROW else 1, dtype=torch.float32, device=dev)
    _check(lib.nvfp4_silu_mul_quantize(_ptr(gu_bf16), M, I, _ptr(codes), _ptr(scales), _ptr(gscale), gscale_mode, _ptr(h),
                                       _stream()))
    return codes, scales, gscale


def nvfp4_silu_mul(gu_bf16, h=None):
    M, I2 = gu_bf16.shape
    I = I2 // 2
    if h is None:
        h = torch.empty((M, I), dtype=torch.bfloat16, device=gu_bf16.device)
    _check(lib.nvfp4_silu_mul(_ptr(gu_bf16), M, I, _ptr(h), _stream()))
    return h


def reset_sampler_new_state(B=1, device="cuda"):
    """zero-filled ReSET state for B sequences."""
    return torch.zeros(B * lib.reset_sampler_state_bytes(), dtype=torch.uint8, device=device)


def reset_sampler_step(logits, state, tau0, t_low, t_high, top_p=0.95, w=32, delimiter_token=-1, seed=0,
                       token_out=None, diag_out=None):
    """one ReSET decoding step for every row of logits [B, V] (float32 or bfloat16).  Returns (tokens int32 [B], diag)."""
    Bn, V = logits.shape
    if token_out is None:
        token_out = torch.empty(Bn, dtype=torch.int32, device=logits.device)
    dt = DTYPE_F32 if logits.dtype == torch.float32 else DTYPE_BF16
    _check(lib.reset_sampler_step(_ptr(logits), dt, Bn, V, logits.stride(0), _ptr(state), tau0, t_low, t_high, top_p, w,
                                  delimiter_token, seed, _ptr(token_out), _ptr(diag_out), _stream()))
    return token_out, diag_out
