"""Helpers for the `-m gpu` parity tests: move oracle-side NumPy arrays to the device and back.
No method arithmetic lives here."""
import numpy as np
import torch

from oracle import nvfp4_oracle as orc
from paper_2606_13233_b200 import inputs


def dev_u8(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.uint8)).cuda()


def dev_bf16_from_bits(bits):
    """uint16 BF16 bit patterns [M,K] -> torch.bfloat16 CUDA tensor (bit-identical)."""
    t = torch.from_numpy(np.ascontiguousarray(bits, dtype=np.uint16).view(np.int16)).cuda()
    return t.view(torch.bfloat16)


def dev_f32(v):
    return torch.tensor([float(v)], dtype=torch.float32, device="cuda")


def host_u8(t):
    return t.cpu().numpy()


def host_bf16_bits(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def host_y_f64(y):
    """GPU output (f32 or bf16) -> float64 ndarray (exact)."""
    return y.float().cpu().numpy().astype(np.float64)


def oracle_weight(N, K, seed=0, shape_id=0):
    """config recipe: W ~ N(0, 0.02) -> BF16 -> oracle NVFP4.  Returns (codes, scales, g)."""
    w = inputs.bf16_bits_as_f32(inputs.make_weight_bits(N, K, seed, shape_id))
    return orc.quantize(w)


def check_gemv(y_gpu_f64, Y, A, what="", bf16_slack=False):
    """north_star tolerance, as written.  `bf16_slack` adds the BF16 output rounding itself
    (half an ulp <= 2^-9 |Y|) for small-K cases with no cancellation, where |Y|/A > 0.26 and NO
    BF16 value can be within 1e-3*A of Y (R9); the BF16 epilogue is pinned bit-exactly
    against the kernel's own FP32 output in those tests."""
    tol = orc.tolerance(A)
    if bf16_slack:
        tol = tol + np.abs(Y) * 2.0 ** -9
    err = np.abs(y_gpu_f64 - Y)
    worst = float(np.max(err / tol)) if err.size else 0.0
    assert np.all(err <= tol), f"{what}: max err/tol = {worst:.3g} at {np.unravel_index(np.argmax(err / tol), err.shape)}"
    return worst
