"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(the tuned table), on SAMPLED output rows the oracle computes one by one.

Weights: an oracle-quantised slab of 512 rows of the config generator (W ~ N(0,0.02) -> BF16 ->
NVFP4) is laid down N/512 times, each copy with its rows rolled by 37*copy, so every output row
has a distinct, known source row; the O projection is additionally checked with the whole
matrix quantised by the oracle."""
import numpy as np
import pytest
import torch

from oracle import nvfp4_oracle as orc
from paper_2606_13233_b200 import inputs
import _gpu_util as U

pytestmark = pytest.mark.gpu
SLAB = 512


@pytest.fixture(scope="module")
def B():
    from paper_2606_13233_b200 import binding
    binding.nvfp4_gemv_set_config(0, 0, 0, 0)
    return binding


def slab_weight(N, K, shape_id):
    sc, ss, g = U.oracle_weight(SLAB, K, 0, shape_id)
    idx = (np.arange(N) % SLAB + 37 * (np.arange(N) // SLAB)) % SLAB
    return sc, ss, g, idx


def sample_rows(N, rng):
    fixed = [0, 1, 31, 32, 33, 255, 256, 257, N // 2 - 1, N // 2, N - 257, N - 33, N - 32, N - 2, N - 1]
    return np.unique(np.concatenate([np.array(fixed), rng.integers(0, N, size=241)]))


@pytest.mark.parametrize("sid,name,N,K", [(i + 1, *s) for i, s in enumerate(inputs.QWEN3_32B_SHAPES)])
@pytest.mark.parametrize("M", [1, 4, 8])
def test_qwen3_32b_shapes_sampled_rows(B, sid, name, N, K, M):
    sc, ss, gw, idx = slab_weight(N, K, sid)
    d_codes = U.dev_u8(sc)[torch.from_numpy(idx).cuda()].contiguous()
    d_scales = U.dev_u8(ss)[torch.from_numpy(idx).cuda()].contiguous()
    blob = B.nvfp4_repack_weight(d_codes, d_scales)
    del d_codes, d_scales
    xbits = inputs.make_activation_bits(M, K, 0, sid)
    xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits))
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    torch.cuda.synchronize()
    assert np.array_equal(U.host_u8(xq[0]), oxc) and np.array_equal(U.host_u8(xq[1]), oxs)
    rows = sample_rows(N, np.random.default_rng(sid))
    Y, A = orc.gemv_w4a4(sc[idx[rows]], ss[idx[rows]], gw, oxc, oxs, ogx)
    y = B.nvfp4_gemv(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, *xq, y_dtype=B.DTYPE_BF16)
    torch.cuda.synchronize()
    got = U.host_y_f64(y)
    U.check_gemv(got[:, rows], Y, A, f"{name} M={M} w4a4 bf16")
    # property that holds at any size: rows with the same source row give identical outputs
    same = np.where(idx == idx[0])[0]
    assert np.all(got[:, same] == got[:, same[:1]])
    if M in (1, 8):
        y = B.nvfp4_gemv(B.MODE_W4A16, blob, U.dev_f32(gw), N, K, U.dev_bf16_from_bits(xbits), y_dtype=B.DTYPE_F32)
        Y, A = orc.gemv_w4a16(sc[idx[rows]], ss[idx[rows]], gw, orc.bf16_bits_to_f32(xbits))
        U.check_gemv(U.host_y_f64(y)[:, rows], Y, A, f"{name} M={M} w4a16 f32")


def test_o_proj_whole_matrix_oracle_quantised(B):
    """configs[1] O projection exactly as specified: the whole W quantised by the oracle."""
    N, K, M = 5120, 8192, 2
    wc, ws, gw = U.oracle_weight(N, K, 0, 2)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    xbits = inputs.make_activation_bits(M, K, 0, 2)
    xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits))
    y = B.nvfp4_gemv(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, *xq, y_dtype=B.DTYPE_BF16)
    torch.cuda.synchronize()
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    Y, A = orc.gemv_w4a4(wc, ws, gw, oxc, oxs, ogx)
    worst = U.check_gemv(U.host_y_f64(y), Y, A, "o_proj full")
    print("o_proj bf16 max err/tol", worst)
