"""GPU parity: nvfp4_gemm_w4a16 (tensor-core W4A16: NVFP4 weights expanded to FP16 in shared memory, BF16 activations,
tcgen05.mma kind::f16) vs the float64 oracle (gemv_w4a16), element by element, north_star tolerance; BF16 output ==
RN_bf16 of the kernel's own FP32 output."""
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


def make_case(M, N, K, seed=0):
    wc, ws, gw = U.oracle_weight(N, K, seed, 0)
    xbits = inputs.make_activation_bits(M, K, seed, 0)
    xf = orc.bf16_bits_to_f32(xbits)
    Y, A = orc.gemv_w4a16(wc, ws, gw, xf)
    return dict(M=M, N=N, K=K, wc=wc, ws=ws, gw=gw, xbits=xbits, Y=Y, A=A)


def test_all_ones_gives_K(B):
    for N, K in [(128, 256), (70, 512), (300, 1024)]:
        wc = np.full((N, K // 2), 0x22, np.uint8); ws = np.full((N, K // 16), 0x38, np.uint8)
        blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
        for M in (1, 8, 9, 40):
            x = torch.ones((M, K), dtype=torch.bfloat16, device="cuda")
            y = B.nvfp4_gemm_w4a16(blob, U.dev_f32(1), N, K, x, y_dtype=B.DTYPE_F32)
            assert np.all(U.host_y_f64(y) == K), (N, K, M)


def test_single_nonzero_weight_lights_one_output(B):
    """one non-zero code at (n, k) x one-hot activation at k: exactly output n is non-zero, with the exact product -- every
    row / chunk / nibble / scale slot of the in-kernel FP16 expansion and of the activation re-layout."""
    N, K, M = 260, 512, 3
    rng = np.random.default_rng(2)
    picks = [(0, 0), (1, 1), (7, 31), (8, 32), (31, 63), (32, 64), (127, 255), (128, 256), (259, 511), (200, 300), (5, 15), (5, 16)]
    picks += [(int(rng.integers(N)), int(rng.integers(K))) for _ in range(12)]
    for n, k in picks:
        wc = np.zeros((N, K // 2), np.uint8); ws = np.zeros((N, K // 16), np.uint8)
        wc[n, k // 2] = 0xB << (4 * (k & 1))            # -1.5
        ws[n, k // 16] = 0x41                           # scale 2.25
        x = torch.zeros((M, K), dtype=torch.bfloat16, device="cuda")
        x[2, k] = 3.0
        blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
        y = U.host_y_f64(B.nvfp4_gemm_w4a16(blob, U.dev_f32(0.5), N, K, x, y_dtype=B.DTYPE_F32))
        want = np.zeros((M, N)); want[2, n] = -1.5 * 2.25 * 3.0 * 0.5
        assert np.array_equal(y, want), (n, k, np.argwhere(y != 0))


def test_extreme_scales_exact_in_fp16(B):
    """largest code x largest scale (6 x 448 = 2688) and the smallest subnormal scale (2^-9 x 0.5): the FP16 expansion is exact."""
    N, K = 128, 256
    wc = np.full((N, K // 2), 0x77, np.uint8); ws = np.full((N, K // 16), 0x7E, np.uint8)
    ws[1::2] = 0x01; wc[1::2] = 0x99                    # odd rows: -0.5 x 2^-9
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    x = torch.zeros((1, K), dtype=torch.bfloat16, device="cuda"); x[0, 7] = 1.0; x[0, 200] = 2.0
    y = U.host_y_f64(B.nvfp4_gemm_w4a16(blob, U.dev_f32(1), N, K, x, y_dtype=B.DTYPE_F32))[0]
    assert np.all(y[0::2] == 2688.0 * 3) and np.all(y[1::2] == -0.5 * 2.0 ** -9 * 3)


CASES = [(1, 128, 256), (8, 128, 256), (3, 100, 512), (5, 300, 1024), (8, 1000, 768), (16, 384, 2048), (17, 257, 1280),
         (32, 640, 1024), (33, 200, 512), (70, 129, 256), (8, 2048, 2048), (2, 19000, 256), (4, 5120, 8192), (1, 5120, 5120)]


@pytest.mark.parametrize("M,N,K", CASES)
def test_parity_vs_oracle(B, M, N, K):
    c = make_case(M, N, K, seed=M + N)
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    x = U.dev_bf16_from_bits(c["xbits"])
    y32 = B.nvfp4_gemm_w4a16(blob, U.dev_f32(c["gw"]), N, K, x, y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    U.check_gemv(U.host_y_f64(y32), c["Y"], c["A"], f"w4a16 tc f32 M={M} N={N} K={K}")
    y16 = B.nvfp4_gemm_w4a16(blob, U.dev_f32(c["gw"]), N, K, x, y_dtype=B.DTYPE_BF16)
    assert np.array_equal(U.host_bf16_bits(y16), orc.f32_to_bf16_bits(y32.cpu().numpy()))


def test_matches_cuda_core_w4a16_and_is_deterministic(B):
    M, N, K = 6, 640, 16384
    c = make_case(M, N, K, seed=3)
    x = U.dev_bf16_from_bits(c["xbits"])
    blob_tc = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    blob_v = B.nvfp4_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    ws = torch.zeros(B.lib.nvfp4_gemm_w4a16_workspace_bytes(M, N, K), dtype=torch.uint8, device="cuda")
    y0 = B.nvfp4_gemm_w4a16(blob_tc, U.dev_f32(c["gw"]), N, K, x, y_dtype=B.DTYPE_F32, workspace=ws).clone()
    y_v = B.nvfp4_gemv(B.MODE_W4A16, blob_v, U.dev_f32(c["gw"]), N, K, x, y_dtype=B.DTYPE_F32)
    assert np.all(np.abs(U.host_y_f64(y0) - U.host_y_f64(y_v)) <= 2 * orc.tolerance(c["A"]))
    for _ in range(4):
        assert torch.equal(B.nvfp4_gemm_w4a16(blob_tc, U.dev_f32(c["gw"]), N, K, x, y_dtype=B.DTYPE_F32, workspace=ws), y0)
    torch.cuda.synchronize()
    assert int(ws[: 4 * ((N + 127) // 128)].view(torch.int32).abs().sum()) == 0


def test_strided_activations_and_wrong_blob(B):
    M, N, K = 4, 256, 512
    c = make_case(M, N, K, seed=4)
    big = torch.full((M, K + 64), float("inf"), dtype=torch.bfloat16, device="cuda")   # padding must never be read
    big[:, :K] = U.dev_bf16_from_bits(c["xbits"])
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    y = B.nvfp4_gemm_w4a16(blob, U.dev_f32(c["gw"]), N, K, big[:, :K], y_dtype=B.DTYPE_F32)
    U.check_gemv(U.host_y_f64(y), c["Y"], c["A"], "strided x")
    blob[8] ^= 1
    assert torch.isnan(B.nvfp4_gemm_w4a16(blob, U.dev_f32(c["gw"]), N, K, big[:, :K], y_dtype=B.DTYPE_F32)).all()


def test_many_back_to_back_launches_do_not_deadlock_or_drift(B):
    """regression for an intermittent deadlock (a dequant group running two buffer generations ahead of the MMAs passed an
    mbarrier wait on the parity of an older phase): hundreds of launches back to back, graph replayed, identical bits."""
    for M, N, K in [(4, 10240, 5120), (7, 5120, 8192)]:
        codes, scales, _ = inputs.make_nvfp4_weight_device(N, K, seed=1, shape_id=1)
        blob = B.nvfp4_gemm_repack_weight(codes, scales)
        gw = U.dev_f32(3e-5)
        x = U.dev_bf16_from_bits(inputs.make_activation_bits(M, K, 0, 1))
        ws = torch.zeros(B.lib.nvfp4_gemm_w4a16_workspace_bytes(M, N, K), dtype=torch.uint8, device="cuda")
        y0 = B.nvfp4_gemm_w4a16(blob, gw, N, K, x, y_dtype=B.DTYPE_BF16, workspace=ws).clone()
        y = torch.empty_like(y0)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for _ in range(20):
                B.nvfp4_gemm_w4a16(blob, gw, N, K, x, y=y, y_dtype=B.DTYPE_BF16, workspace=ws)
        for _ in range(15):
            g.replay()
        torch.cuda.synchronize()
        assert torch.equal(y, y0)
