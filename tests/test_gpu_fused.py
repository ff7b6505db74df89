"""GPU: nvfp4_gemv_fused_quant (activation quantizer inside the GEMV) vs the oracle and vs the two-call path."""
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
    binding.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)
    return binding


@pytest.mark.parametrize("M,N,K", [(1, 2048, 2048), (1, 300, 1296), (2, 1000, 2576), (4, 96, 1040), (8, 257, 400),
                                   (1, 5120, 8192), (3, 64, 16), (1, 2048 + 96, 5120)])
def test_fused_matches_oracle_and_two_call_path(B, M, N, K):
    wc, ws, gw = U.oracle_weight(N, K, 3, M)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    d_gw = U.dev_f32(gw)
    xbits = inputs.make_activation_bits(M, K, 3, M)
    x = U.dev_bf16_from_bits(xbits)
    gx_out = torch.zeros(1, dtype=torch.float32, device="cuda")
    y = B.nvfp4_gemv_fused_quant(blob, d_gw, N, K, x, x_gscale_out=gx_out, y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    assert np.float32(gx_out.item()).view(np.uint32) == np.float32(ogx).view(np.uint32)      # global scale bit-exact
    Y, A = orc.gemv_w4a4(wc, ws, gw, oxc, oxs, ogx)
    U.check_gemv(U.host_y_f64(y), Y, A, f"fused M={M} N={N} K={K}")
    if M == 1:      # same arithmetic path as quantize_act + gemv: identical bits
        xq = B.nvfp4_quantize_act(x)
        y2 = B.nvfp4_gemv(B.MODE_W4A4, blob, d_gw, N, K, *xq, y_dtype=B.DTYPE_F32)
        assert torch.equal(y, y2)
    yb = B.nvfp4_gemv_fused_quant(blob, d_gw, N, K, x, y_dtype=B.DTYPE_BF16)
    assert np.array_equal(U.host_bf16_bits(yb), orc.f32_to_bf16_bits(y.cpu().numpy()))


def test_fused_edge_inputs(B):
    """all-zero activations (g = 0), a flushed block, padded rows (ldx > K)."""
    N, K, M = 64, 512, 2
    wc, ws, gw = U.oracle_weight(N, K, 4, 1)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    z = torch.zeros((M, K), dtype=torch.bfloat16, device="cuda")
    y = B.nvfp4_gemv_fused_quant(blob, U.dev_f32(gw), N, K, z, y_dtype=B.DTYPE_F32)
    assert not y.any()
    xf = np.zeros((M, K), dtype=np.float32); xf[0, 0] = 2688.0; xf[0, 32] = 6 * 2.0 ** -11; xf[1, 100] = -3.0
    bits = orc.f32_to_bf16_bits(xf)
    buf = np.full((M, K + 64), 0x7F80, dtype=np.uint16); buf[:, :K] = bits          # +inf padding must not be read
    x = U.dev_bf16_from_bits(buf)[:, :K]
    y = B.nvfp4_gemv_fused_quant(blob, U.dev_f32(gw), N, K, x, y_dtype=B.DTYPE_F32)
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(bits))
    Y, A = orc.gemv_w4a4(wc, ws, gw, oxc, oxs, ogx)
    U.check_gemv(U.host_y_f64(y), Y, A, "fused edge")
