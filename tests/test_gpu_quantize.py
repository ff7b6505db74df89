"""GPU parity: nvfp4_quantize_act (through the C ABI) vs the oracle -- codes, scales and the
global scale must be BIT-IDENTICAL (north_star; R1-R5)."""
import os

import numpy as np
import pytest
import torch

from oracle import nvfp4_oracle as orc
from paper_2606_13233_b200 import inputs
import _gpu_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_13233_b200 import binding
    return binding


def _golden(path):
    out = {}
    for line in open(path):
        line = line.strip()
        if line and not line.startswith("#"):
            k, v = line.split(":", 1)
            out[k.strip()] = v.split()
    return out


def run_gpu(B, bits, static_g=None, ld=None):
    M, K = bits.shape
    if ld is None:
        x = U.dev_bf16_from_bits(bits)
    else:
        buf = np.full((M, ld), 0x7F80, dtype=np.uint16)   # +inf in the padding: must never be read
        buf[:, :K] = bits
        x = U.dev_bf16_from_bits(buf)[:, :K]
    if static_g is None:
        c, s, g = B.nvfp4_quantize_act(x)
    else:
        c, s, g = B.nvfp4_quantize_act(x, gscale=U.dev_f32(static_g), gscale_mode=B.GSCALE_STATIC)
    torch.cuda.synchronize()
    return U.host_u8(c), U.host_u8(s), np.float32(g.cpu().numpy()[0])


def assert_same(B, bits, static_g=None, ld=None):
    c, s, g = run_gpu(B, bits, static_g, ld)
    oc, os_, og = orc.quantize(orc.bf16_bits_to_f32(bits), g=static_g)
    assert g.view(np.uint32) == np.float32(og).view(np.uint32), (g, og)
    assert np.array_equal(s, os_), f"{np.count_nonzero(s != os_)} scale bytes differ"
    assert np.array_equal(c, oc), f"{np.count_nonzero(c != oc)} code bytes differ"


def test_worked_examples(B, golden_dir):
    G = _golden(os.path.join(golden_dir, "quant_example_A.txt"))
    x = np.array([float(v) for v in G["x"]], dtype=np.float32)[None, :]
    c, s, g = run_gpu(B, orc.f32_to_bf16_bits(x))
    assert int(g.view(np.uint32)) == int(G["g_bits"][0], 16)
    assert [int(v) for v in s[0]] == [int(v, 16) for v in G["scales"]]
    assert [int(v) for v in c[0]] == [int(v, 16) for v in G["packed"]]
    G = _golden(os.path.join(golden_dir, "quant_example_B.txt"))
    x = np.array([float(v) for v in G["x0"] + G["x1"]], dtype=np.float32)[None, :]
    c, s, g = run_gpu(B, orc.f32_to_bf16_bits(x))
    assert int(g.view(np.uint32)) == int(G["g_bits"][0], 16)
    assert [int(v) for v in s[0]] == [int(v, 16) for v in G["scales"]]
    assert [int(v) for v in c[0]] == [int(v, 16) for v in G["packed"]]


@pytest.mark.parametrize("M,K", [(1, 2048), (1, 5120), (1, 8192), (1, 25600), (2, 5120), (3, 8192), (4, 25600),
                                 (6, 5120), (8, 5120), (8, 8192), (8, 25600), (1, 16), (3, 48), (5, 1040), (7, 16400)])
def test_config_activations_bit_exact(B, M, K):
    assert_same(B, inputs.make_activation_bits(M, K, seed=0, shape_id=M * 100000 + K))


def test_large_tensor_two_kernel_path(B):
    # 8 x 131072 = 1 Mi elements > one cluster's register capacity -> generic path
    assert_same(B, inputs.make_activation_bits(8, 131072, seed=1, shape_id=9))


def test_static_gscale_and_row_stride(B):
    bits = inputs.make_activation_bits(4, 5120, seed=2, shape_id=3)
    assert_same(B, bits, static_g=np.float32(0.01))
    assert_same(B, bits, static_g=np.float32(3e-5))       # many saturated scales
    assert_same(B, bits, ld=5120 + 64)                    # padded rows (ldx > K)
    assert_same(B, bits, static_g=np.float32(0.02), ld=5120 + 8)


def test_edge_cases(B):
    # (i) binary32 sequence vs exact division (R2)
    x = np.zeros((1, 32), dtype=np.float32); x[0, 0] = 28.0; x[0, 16] = 3.875; x[0, 17] = -1.0
    c, s, g = run_gpu(B, orc.f32_to_bf16_bits(x))
    assert int(g.view(np.uint32)) == 0x3C2AAAAB and list(s[0]) == [0x7E, 0x67]
    # (ii) subnormal scale tie, flushed block
    x = np.zeros((1, 48), dtype=np.float32)
    x[0, 0] = 2688.0; x[0, 16] = 6 * 1.5 * 2.0 ** -9; x[0, 17] = 2.0 ** -9
    x[0, 32] = 6 * 2.0 ** -11; x[0, 33] = -6 * 2.0 ** -11
    assert_same(B, orc.f32_to_bf16_bits(x))
    c, s, g = run_gpu(B, orc.f32_to_bf16_bits(x))
    assert g == np.float32(1.0) and list(s[0]) == [0x7E, 0x02, 0x00]
    # (iii) all zero, negative zero
    z = np.zeros((2, 64), dtype=np.float32); z[1, 5] = -0.0
    c, s, g = run_gpu(B, orc.f32_to_bf16_bits(z))
    assert g == 0 and not c.any() and not s.any()
    # (iv) sign of tiny negatives is kept, ties go to the even code
    t = np.zeros((1, 16), dtype=np.float32)
    t[0, :8] = [6.0, -0.25, 0.25, -0.75, 1.25, -1.75, 2.5, -3.5]
    t[0, 8:] = [5.0, -5.0, -0.0, 0.0, -0.001, 0.001, 3.5, -2.5]
    assert_same(B, orc.f32_to_bf16_bits(t), static_g=np.float32(1.0 / 448.0))


def test_exhaustive_bf16_over_divisors(B):
    """every positive BF16 magnitude in a range that covers all E2M1 decision points, against
    several block divisors d = g*s: catches any deviation from true binary32 division / RNE."""
    rng = np.random.default_rng(5)
    mags = np.arange(0x3A00, 0x4200, dtype=np.uint16)     # 2^-11 .. 32
    for g in [np.float32(1.0 / 448.0), np.float32(0.0026041667), np.float32(7.3e-3), np.float32(1.37e-2)]:
        bits = np.concatenate([mags, mags | 0x8000])
        rng.shuffle(bits)
        K = (bits.size // 16) * 16
        assert_same(B, bits[:K][None, :].copy(), static_g=g)


def test_quantizer_feeds_idempotence(B):
    """quantize(dequantize(q)) == q on the GPU too (oracle invariant)."""
    bits = inputs.make_activation_bits(2, 5120, seed=3, shape_id=1)
    c, s, g = run_gpu(B, bits)
    v = orc.dequantize(c, s, g).astype(np.float32)
    bits2 = orc.f32_to_bf16_bits(v)
    if np.array_equal(orc.bf16_bits_to_f32(bits2), v):     # representable in BF16 (g is not a power of two: usually not)
        c2, s2, g2 = run_gpu(B, bits2)
        assert np.array_equal(c, c2) and np.array_equal(s, s2)
    assert_same(B, bits2)
