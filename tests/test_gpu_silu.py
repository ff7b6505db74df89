"""GPU: SiLU*mul glue (step a8) vs the float64 oracle, tolerance 1 BF16 ulp."""
import numpy as np
import pytest
import torch

from oracle import nvfp4_oracle as orc
import _gpu_util as U

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("M,I", [(1, 25600), (8, 25600), (3, 8), (2, 1000)])
def test_silu_mul(M, I):
    from paper_2606_13233_b200 import binding as B
    rng = np.random.default_rng(M + I)
    gu = (rng.standard_normal((M, 2 * I)) * 3).astype(np.float32)
    bits = orc.f32_to_bf16_bits(gu)
    h = B.nvfp4_silu_mul(U.dev_bf16_from_bits(bits))
    torch.cuda.synchronize()
    want = orc.silu_mul(orc.bf16_bits_to_f32(bits))
    got = U.host_y_f64(h)
    ulp = np.maximum(np.abs(want), 2.0 ** -120) * 2.0 ** -7       # one BF16 ulp is at most 2^-7 relative
    assert np.all(np.abs(got - want) <= ulp)
