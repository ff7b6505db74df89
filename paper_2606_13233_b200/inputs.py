"""Seeded synthetic input generators shared by the tests, the oracle legs and bench.py.

This module holds NONE of the method's arithmetic (no quantisation, no codecs, no
GEMV): it only draws random numbers with NumPy and stores them as BF16 bit
patterns.  Recipe (BASELINE.json configs[0..3]):

* weights      W[N,K] ~ N(0, 0.02)            -> BF16
* activations  X[M,K] ~ N(0, 1), then a Bernoulli(0.005) mask over the K channels
               multiplies those columns by 20 -> BF16

They stand in for the Qwen3-32B layer shapes of PAPER.md:231-234 (Table 4); no
checkpoint or dataset is involved.
"""
from __future__ import annotations

import numpy as np

# (name, N, K) -- BASELINE.json configs[1]; shape_id = index in this tuple + 1
QWEN3_32B_SHAPES = (
    ("qkv", 10240, 5120),
    ("o", 5120, 8192),
    ("gate_up", 51200, 5120),
    ("down", 5120, 25600),
)
CONFIG0_SHAPE = ("cfg0", 2048, 2048)

TENSOR_W, TENSOR_X = 0, 1


def _rng(seed: int, shape_id: int, tensor_id: int) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([int(seed), int(shape_id), int(tensor_id)]))


def to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> BF16 bit patterns (uint16), round to nearest even.  Storage
    conversion of the synthetic inputs only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))
    return (r >> np.uint32(16)).astype(np.uint16)


def bf16_bits_as_f32(bits: np.ndarray) -> np.ndarray:
    return (np.asarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def make_weight_bits(N: int, K: int, seed: int = 0, shape_id: int = 0, rows=None) -> np.ndarray:
    """W[N,K] ~ N(0, 0.02) as BF16 bits.  Rows are drawn in chunks of 1024 from
    per-chunk streams so that any subset of rows can be regenerated cheaply
    (`rows` = iterable of row indices -> only those rows, in that order)."""
    chunk = 1024
    def chunk_bits(ci):
        rng = np.random.default_rng(np.random.SeedSequence([int(seed), int(shape_id), TENSOR_W, int(ci)]))
        n = min(chunk, N - ci * chunk)
        return to_bf16_bits(rng.standard_normal((n, K), dtype=np.float32) * np.float32(0.02))
    if rows is None:
        out = np.empty((N, K), dtype=np.uint16)
        for ci in range((N + chunk - 1) // chunk):
            out[ci * chunk: ci * chunk + chunk] = chunk_bits(ci)
        return out
    rows = [int(r) for r in rows]
    out = np.empty((len(rows), K), dtype=np.uint16)
    cache = {}
    for i, r in enumerate(rows):
        ci = r // chunk
        if ci not in cache:
            cache = {ci: chunk_bits(ci)}
        out[i] = cache[ci][r - ci * chunk]
    return out


def make_activation_bits(M: int, K: int, seed: int = 0, shape_id: int = 0) -> np.ndarray:
    """X[M,K] ~ N(0,1) with 0.5% of the K channels scaled x20, as BF16 bits."""
    rng = _rng(seed, shape_id, TENSOR_X)
    x = rng.standard_normal((M, K), dtype=np.float32)
    outlier = rng.random(K) < 0.005
    x[:, outlier] *= np.float32(20.0)
    return to_bf16_bits(x)


def make_nvfp4_weight_device(N: int, K: int, seed: int = 0, shape_id: int = 0, device="cuda"):
    """Full-size bench weights drawn directly in the NVFP4 domain ON THE DEVICE (torch RNG):
    uniform random code bytes, scale bytes uniform in 0x64..0x7E (the range the oracle produces
    for W ~ N(0, 0.02): DESIGN.md "Input recipe"), and a fixed global scale.  Returns
    (codes u8 [N,K/2], scales u8 [N,K/16], g float).  Kernel time does not depend on the values;
    parity at these sizes is tested separately on oracle-quantised weights."""
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed((int(seed) * 1000003 + int(shape_id)) & 0x7FFFFFFF)
    codes = torch.randint(0, 256, (N, K // 2), dtype=torch.uint8, device=device, generator=gen)
    scales = torch.randint(0x64, 0x7F, (N, K // 16), dtype=torch.uint8, device=device, generator=gen)
    return codes, scales, 3.0e-5
