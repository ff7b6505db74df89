"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(the tuned table), on SAMPLED output rows the oracle computes one by one.

Every (config, M, mode, output dtype) BASELINE.json lists appears here: configs[1]/[2] = W4A4 with BF16
output at M in {1,2,3,4,6,8}; configs[3] = W4A16 at M in {1,2,4,8} with FP32 and BF16 output; all four
Qwen3-32B shapes.  Both work splits of the GEMV (whole units / data-parallel + stream-K) are run on every
shape at M = 1 and 4.

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
SHAPES = [(i + 1, *s) for i, s in enumerate(inputs.QWEN3_32B_SHAPES)]


@pytest.fixture(scope="module")
def B():
    from paper_2606_13233_b200 import binding
    binding.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)
    yield binding
    binding.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)


_STATE = {}


def shape_state(B, sid, N, K):
    """slab weight (oracle-quantised), its device blob and the sampled rows: built once per shape."""
    if sid not in _STATE:
        _STATE.clear()                                   # one 148 MB blob at a time
        sc, ss, g = U.oracle_weight(SLAB, K, 0, sid)
        idx = (np.arange(N) % SLAB + 37 * (np.arange(N) // SLAB)) % SLAB
        d_idx = torch.from_numpy(idx).cuda()
        blob = B.nvfp4_repack_weight(U.dev_u8(sc)[d_idx].contiguous(), U.dev_u8(ss)[d_idx].contiguous())
        rng = np.random.default_rng(sid)
        fixed = [0, 1, 31, 32, 33, 255, 256, 257, N // 2 - 1, N // 2, N - 257, N - 33, N - 32, N - 2, N - 1]
        rows = np.unique(np.concatenate([np.array(fixed), rng.integers(0, N, size=241)]))
        _STATE[sid] = dict(sc=sc, ss=ss, gw=g, idx=idx, blob=blob, rows=rows, d_gw=U.dev_f32(g))
    return _STATE[sid]


def run_w4a4(B, st, name, N, K, M, sid, what):
    xbits = inputs.make_activation_bits(M, K, 0, sid)
    xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits))
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    torch.cuda.synchronize()
    assert np.array_equal(U.host_u8(xq[0]), oxc) and np.array_equal(U.host_u8(xq[1]), oxs)
    rows, idx = st["rows"], st["idx"]
    Y, A = orc.gemv_w4a4(st["sc"][idx[rows]], st["ss"][idx[rows]], st["gw"], oxc, oxs, ogx)
    y = B.nvfp4_gemv(B.MODE_W4A4, st["blob"], st["d_gw"], N, K, *xq, y_dtype=B.DTYPE_BF16)
    torch.cuda.synchronize()
    got = U.host_y_f64(y)
    U.check_gemv(got[:, rows], Y, A, f"{name} M={M} w4a4 bf16 {what}")          # tolerance as written (no BF16 slack)
    # property that holds at any size: rows with the same source row give identical outputs
    same = np.where(idx == idx[0])[0]
    assert np.all(got[:, same] == got[:, same[:1]])
    assert np.all(np.isfinite(got))


@pytest.mark.parametrize("sid,name,N,K", SHAPES)
@pytest.mark.parametrize("M", [1, 2, 3, 4, 6, 8])
def test_w4a4_bf16_sampled_rows(B, sid, name, N, K, M):
    """configs[1] (M = 1) and configs[2] (M in {1,2,3,4,6,8}): quantize_act on the GPU + W4A4 GEMV, BF16 output."""
    st = shape_state(B, sid, N, K)
    run_w4a4(B, st, name, N, K, M, sid, "tuned")


@pytest.mark.parametrize("sid,name,N,K", SHAPES)
@pytest.mark.parametrize("M", [1, 4])
@pytest.mark.parametrize("balance", [1, 2])
def test_w4a4_both_work_splits(B, sid, name, N, K, M, balance):
    """the two balance modes of the GEMV (1 = data-parallel + stream-K through the workspace, 2 = whole units)."""
    st = shape_state(B, sid, N, K)
    try:
        B.nvfp4_gemv_set_config(0, 0, 0, 0, 0, balance)
        assert B.nvfp4_gemv_get_config(B.MODE_W4A4, M, N, K)["balance"] == balance
        run_w4a4(B, st, name, N, K, M, sid, f"balance={balance}")
    finally:
        B.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)


@pytest.mark.parametrize("sid,name,N,K", SHAPES)
@pytest.mark.parametrize("M", [1, 2, 4, 8])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_w4a16_sampled_rows(B, sid, name, N, K, M, dtype):
    """configs[3]: NVFP4 weights, BF16 activations consumed directly, FP32 accumulation; FP32 and BF16 output."""
    st = shape_state(B, sid, N, K)
    xbits = inputs.make_activation_bits(M, K, 0, sid)
    rows, idx = st["rows"], st["idx"]
    y = B.nvfp4_gemv(B.MODE_W4A16, st["blob"], st["d_gw"], N, K, U.dev_bf16_from_bits(xbits),
                     y_dtype=B.DTYPE_F32 if dtype == "f32" else B.DTYPE_BF16)
    torch.cuda.synchronize()
    Y, A = orc.gemv_w4a16(st["sc"][idx[rows]], st["ss"][idx[rows]], st["gw"], orc.bf16_bits_to_f32(xbits))
    U.check_gemv(U.host_y_f64(y)[:, rows], Y, A, f"{name} M={M} w4a16 {dtype}")


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
