"""GPU parity: nvfp4_gemm (tensor-core block-scaled MMA path, through the C ABI) vs the float64 oracle, element by
element.  Same acceptance as the GEMV (north_star): |y_gpu - y_ref| <= 1e-3 * sum_k|w_k x_k| + 1e-6; the BF16 output
must be bit-identical to RN_bf16 of the same kernel's FP32 output."""
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


def make_case(M, N, K, seed=0, shape_id=0):
    wc, ws, gw = U.oracle_weight(N, K, seed, shape_id)
    xbits = inputs.make_activation_bits(M, K, seed, shape_id)
    xc, xs, gx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    Y, A = orc.gemv_w4a4(wc, ws, gw, xc, xs, gx)
    return dict(M=M, N=N, K=K, wc=wc, ws=ws, gw=gw, xc=xc, xs=xs, gx=gx, Y=Y, A=A, xbits=xbits)


def run(B, c, dtype, blob=None):
    blob = blob if blob is not None else B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    y = B.nvfp4_gemm(blob, U.dev_f32(c["gw"]), c["N"], c["K"], U.dev_u8(c["xc"]), U.dev_u8(c["xs"]), U.dev_f32(c["gx"]),
                     y_dtype=dtype)
    torch.cuda.synchronize()
    return y


def test_repack_round_trip(B):
    rng = np.random.default_rng(0)
    for N, K in [(128, 256), (130, 512), (1000, 768), (5, 256)]:
        wc = rng.integers(0, 256, (N, K // 2), dtype=np.uint8)
        ws = rng.integers(0, 0x7F, (N, K // 16), dtype=np.uint8)
        blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
        assert blob.numel() == 128 + ((N + 127) // 128) * (K // 256) * 18432
        c2, s2 = B.nvfp4_gemm_unpack_weight(blob, N, K)
        assert np.array_equal(U.host_u8(c2), wc) and np.array_equal(U.host_u8(s2), ws)
        # a permutation: the multiset of bytes is preserved (padding rows are zero)
        body = U.host_u8(blob)[128:]
        pad = (-N) % 128
        want = np.bincount(np.concatenate([wc.ravel(), ws.ravel()]), minlength=256)
        want[0] += pad * (K // 2 + K // 16)
        assert np.array_equal(np.bincount(body, minlength=256), want)


def test_unsupported_shapes(B):
    assert B.lib.nvfp4_gemm_repacked_bytes(128, 384) == 0       # K % 256 != 0
    assert B.lib.nvfp4_gemm_repacked_bytes(128, 128) == 0
    assert B.lib.nvfp4_gemm_workspace_bytes(8, 128, 320) == 0


def test_all_ones_gives_K(B):
    """all codes +1.0, all scales 1.0, g = 1 -> Y = K exactly."""
    for N, K in [(128, 256), (70, 512), (300, 1024)]:
        wc = np.full((N, K // 2), 0x22, np.uint8); ws = np.full((N, K // 16), 0x38, np.uint8)
        blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
        for M in (1, 8, 9, 40):
            xc = np.full((M, K // 2), 0x22, np.uint8); xs = np.full((M, K // 16), 0x38, np.uint8)
            y = B.nvfp4_gemm(blob, U.dev_f32(1), N, K, U.dev_u8(xc), U.dev_u8(xs), U.dev_f32(1), y_dtype=B.DTYPE_F32)
            assert np.all(U.host_y_f64(y) == K), (N, K, M)


def test_single_nonzero_weight_lights_one_output(B):
    """one non-zero code at (n, k) and a one-hot activation at k: exactly output n is non-zero -- catches every
    row / chunk / nibble / scale-slot permutation error of the two re-layouts."""
    N, K, M = 260, 512, 3
    rng = np.random.default_rng(1)
    picks = [(0, 0), (1, 1), (7, 31), (8, 32), (31, 63), (32, 64), (127, 255), (128, 256), (259, 511), (200, 300)]
    picks += [(int(rng.integers(N)), int(rng.integers(K))) for _ in range(14)]
    for n, k in picks:
        wc = np.zeros((N, K // 2), np.uint8); ws = np.zeros((N, K // 16), np.uint8)
        wc[n, k // 2] = 0x3 << (4 * (k & 1))            # +1.5
        ws[n, k // 16] = 0x40                           # scale 2.0
        xc = np.zeros((M, K // 2), np.uint8); xs = np.zeros((M, K // 16), np.uint8)
        xc[1, k // 2] = 0xC << (4 * (k & 1))            # -2.0
        xs[1, k // 16] = 0x30                           # scale 0.5
        blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
        y = U.host_y_f64(B.nvfp4_gemm(blob, U.dev_f32(1), N, K, U.dev_u8(xc), U.dev_u8(xs), U.dev_f32(1), y_dtype=B.DTYPE_F32))
        want = np.zeros((M, N)); want[1, n] = 1.5 * 2.0 * -2.0 * 0.5
        assert np.array_equal(y, want), (n, k, np.argwhere(y != 0))


CASES = [
    # (M, N, K): one tile one stage; ragged N; several tiles and stages (stream-K partial tiles); every MT; M > 128
    (1, 128, 256), (8, 128, 256), (3, 100, 512), (5, 300, 1024), (8, 1000, 768), (16, 384, 2048), (17, 257, 1280),
    (33, 640, 1024), (64, 512, 512), (100, 384, 768), (128, 256, 1024), (130, 200, 512), (300, 129, 256),
    (8, 2048, 2048), (2, 19000, 256), (4, 5120, 8192),
]


@pytest.mark.parametrize("M,N,K", CASES)
def test_parity_vs_oracle(B, M, N, K):
    c = make_case(M, N, K, seed=M + N, shape_id=0)
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    y32 = run(B, c, B.DTYPE_F32, blob)
    U.check_gemv(U.host_y_f64(y32), c["Y"], c["A"], f"gemm f32 M={M} N={N} K={K}")
    y16 = run(B, c, B.DTYPE_BF16, blob)
    assert np.array_equal(U.host_bf16_bits(y16), orc.f32_to_bf16_bits(y32.cpu().numpy()))


def test_gpu_quantizer_feeds_gemm_and_matches_gemv(B):
    """the path of the configs: X quantised on the GPU; the tensor-core result agrees with the CUDA-core GEMV's to
    FP32 summation-order noise (both are inside the oracle tolerance)."""
    M, N, K = 8, 1024, 2048
    c = make_case(M, N, K, seed=5)
    xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(c["xbits"]))
    blob_tc = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    blob_v = B.nvfp4_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    y_tc = B.nvfp4_gemm(blob_tc, U.dev_f32(c["gw"]), N, K, *xq, y_dtype=B.DTYPE_F32)
    y_v = B.nvfp4_gemv(B.MODE_W4A4, blob_v, U.dev_f32(c["gw"]), N, K, *xq, y_dtype=B.DTYPE_F32)
    U.check_gemv(U.host_y_f64(y_tc), c["Y"], c["A"], "gemm after GPU quantizer")
    assert np.all(np.abs(U.host_y_f64(y_tc) - U.host_y_f64(y_v)) <= 2 * orc.tolerance(c["A"]))


def test_per_row_global_scales(B):
    M, N, K = 6, 300, 512
    wc, ws, gw = U.oracle_weight(N, K, 3, 0)
    xbits = inputs.make_activation_bits(M, K, 3, 0)
    xf = orc.bf16_bits_to_f32(xbits) * np.array([1, 24, 0.5, 3, 1, 7], np.float32)[:, None]
    rows = [orc.quantize(xf[m:m + 1]) for m in range(M)]
    xc = np.concatenate([r[0] for r in rows]); xs = np.concatenate([r[1] for r in rows])
    gxs = np.array([r[2] for r in rows], np.float32)
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    y = B.nvfp4_gemm(blob, U.dev_f32(gw), N, K, U.dev_u8(xc), U.dev_u8(xs), torch.from_numpy(gxs).cuda(),
                     y_dtype=B.DTYPE_F32, gscale_per_row=True)
    for m in range(M):
        Y, A = orc.gemv_w4a4(wc, ws, gw, rows[m][0], rows[m][1], rows[m][2])
        U.check_gemv(U.host_y_f64(y)[m:m + 1], Y, A, f"row {m}")


def test_wrong_blob_gives_nan(B):
    c = make_case(2, 256, 512)
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    blob[8] ^= 1                                        # N in the header no longer matches
    y = run(B, c, B.DTYPE_F32, blob)
    assert torch.isnan(y).all()


def test_deterministic_and_counters_left_zero(B):
    M, N, K = 8, 1000, 2048
    c = make_case(M, N, K, seed=9)
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    xp = B.nvfp4_gemm_pack_act(U.dev_u8(c["xc"]), U.dev_u8(c["xs"]))
    ws = B.nvfp4_gemm_packed_new_workspace(M, N, K, "cuda")
    args = (blob, U.dev_f32(c["gw"]), N, K, xp, U.dev_f32(c["gx"]), M)
    y0 = B.nvfp4_gemm_packed(*args, y_dtype=B.DTYPE_F32, workspace=ws).clone()
    U.check_gemv(U.host_y_f64(y0), c["Y"], c["A"], "packed")
    for _ in range(5):
        y = B.nvfp4_gemm_packed(*args, y_dtype=B.DTYPE_F32, workspace=ws)
        assert torch.equal(y, y0)
    torch.cuda.synchronize()
    ntiles = (N + 127) // 128                           # the workspace starts with one arrival counter per tile
    assert int(ws[: 4 * ntiles].view(torch.int32).abs().sum()) == 0


@pytest.mark.parametrize("M,K", [(1, 256), (3, 512), (8, 2048), (20, 1024), (128, 512)])
def test_quantize_packed_equals_pack_of_canonical(B, M, K):
    """the fused quantizer writes byte for byte what quantize_act + pack_act write (for the tokens < M)."""
    xbits = inputs.make_activation_bits(M, K, 1, 0)
    xc, xs, gx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    want = U.host_u8(B.nvfp4_gemm_pack_act(U.dev_u8(xc), U.dev_u8(xs)))
    buf = torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(M, K), dtype=torch.uint8, device="cuda")
    got, g = B.nvfp4_quantize_act_packed(U.dev_bf16_from_bits(xbits), xpack=buf)
    assert np.array_equal(U.host_u8(got), want)
    assert g.cpu().numpy().view(np.uint32)[0] == np.float32(gx).view(np.uint32)


def test_packed_chain_matches_oracle(B):
    """quantize_act_packed -> gemm_packed (the chain's two launches) against the oracle, M = 1..8 and a prefill-ish M."""
    for M, N, K in [(1, 640, 1024), (4, 1000, 2048), (8, 384, 5120), (48, 300, 1024)]:
        c = make_case(M, N, K, seed=7 + M)
        blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
        xp, g = B.nvfp4_quantize_act_packed(U.dev_bf16_from_bits(c["xbits"]))
        y = B.nvfp4_gemm_packed(blob, U.dev_f32(c["gw"]), N, K, xp, g, M, y_dtype=B.DTYPE_F32)
        U.check_gemv(U.host_y_f64(y), c["Y"], c["A"], f"packed chain M={M} N={N} K={K}")


def test_silu_mul_quantize_packed(B):
    M, I = 4, 1024
    rng = np.random.default_rng(3)
    gu = torch.from_numpy(rng.standard_normal((M, 2 * I)).astype(np.float32)).cuda().to(torch.bfloat16)
    xc, xs, g = B.nvfp4_silu_mul_quantize(gu)
    want = U.host_u8(B.nvfp4_gemm_pack_act(xc, xs))
    buf = torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(M, I), dtype=torch.uint8, device="cuda")
    got, g2 = B.nvfp4_silu_mul_quantize_packed(gu, xpack=buf)
    assert np.array_equal(U.host_u8(got), want) and torch.equal(g, g2)


def test_silu_mul_quantize_packed_static_any_size(B):
    """a STATIC scale needs no tensor-wide amax: plain wide grid, no M * I limit (the DYNAMIC modes keep theirs: one cluster)"""
    M, I = 32, 25600
    rng = np.random.default_rng(5)
    gu = torch.from_numpy((rng.standard_normal((M, 2 * I)) * 2).astype(np.float32)).cuda().to(torch.bfloat16)
    gs = U.dev_f32(np.float32(0.003))
    h = torch.empty((M, I), dtype=torch.bfloat16, device="cuda")
    zeros = lambda m: torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(m, I), dtype=torch.uint8, device="cuda")   # (records have unused bytes)
    got, _ = B.nvfp4_silu_mul_quantize_packed(gu, xpack=zeros(M), gscale=gs.clone(), gscale_mode=B.GSCALE_STATIC, h_out=h)
    h2 = B.nvfp4_silu_mul(gu)
    want, _ = B.nvfp4_quantize_act_packed(h2, xpack=zeros(M), gscale=gs.clone(), gscale_mode=B.GSCALE_STATIC)
    assert torch.equal(h, h2) and torch.equal(got, want)
    # rows 8..15 through the canonical quantizer (M <= 8 there) and the oracle
    xc, xs, _ = B.nvfp4_quantize_act(h2[8:16].contiguous(), gscale=gs.clone(), gscale_mode=B.GSCALE_STATIC)
    oc, os_, _ = orc.quantize(orc.bf16_bits_to_f32(U.host_bf16_bits(h2[8:16].contiguous())), g=np.float32(0.003))
    assert np.array_equal(U.host_u8(xc), oc) and np.array_equal(U.host_u8(xs), os_)
    sub, _ = B.nvfp4_quantize_act_packed(h2[8:16].contiguous(), xpack=zeros(8), gscale=gs.clone(), gscale_mode=B.GSCALE_STATIC)
    assert torch.equal(sub, B.nvfp4_gemm_pack_act(xc, xs, xpack=zeros(8)))
    with pytest.raises(B.Nvfp4Error):
        B.nvfp4_silu_mul_quantize_packed(gu)              # DYNAMIC: M * I > 524288


@pytest.mark.parametrize("M,N,K,nq", [(1, 512, 512, 512), (8, 1024, 2048, 768), (5, 5120, 1024, 5120), (24, 768, 512, 256),
                                       (100, 512, 768, 512), (4, 10240, 5120, 8192), (8, 5120, 8192, 5120)])
def test_fused_output_quantizer_equals_separate_quantizer_and_oracle(B, M, N, K, nq):
    """nvfp4_gemm_packed_quant_out: the packed records its epilogue writes == pack_act(quantize_act(STATIC) of the BF16
    output of the plain GEMM) byte for byte, and == the oracle's STATIC quantisation of that output; the optional y equals
    the plain GEMM's.  Covers whole tiles, K-sliced tiles (fix-up paths) and the bulk fix-up (M > 8)."""
    c = make_case(M, N, K, seed=N + K + M)
    blob = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    xp = B.nvfp4_gemm_pack_act(U.dev_u8(c["xc"]), U.dev_u8(c["xs"]))
    gw, gx = U.dev_f32(c["gw"]), U.dev_f32(c["gx"])
    y_ref = B.nvfp4_gemm_packed(blob, gw, N, K, xp, gx, M, y_dtype=B.DTYPE_BF16)
    torch.cuda.synchronize()
    yf = orc.bf16_bits_to_f32(U.host_bf16_bits(y_ref))[:, :nq]
    # a static scale as a calibration would give it: from the tensor's amax, made a bit too small so that some blocks saturate
    g_static = np.float32(np.max(np.abs(yf)) / 2688.0 * 0.8)
    d_g = U.dev_f32(g_static)
    out = torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(M, nq), dtype=torch.uint8, device="cuda")
    y = torch.zeros((M, N), dtype=torch.bfloat16, device="cuda")
    B.nvfp4_gemm_packed_quant_out(blob, gw, N, K, xp, gx, M, d_g, n_quant=nq, xpack_out=out, y=y)
    torch.cuda.synchronize()
    assert torch.equal(y, y_ref)
    # the separate GPU quantizer (STATIC, packed output) on the same BF16 values
    want = torch.zeros_like(out)
    B.nvfp4_quantize_act_packed(y_ref[:, :nq].contiguous(), xpack=want, gscale=d_g.clone(), gscale_mode=B.GSCALE_STATIC)
    torch.cuda.synchronize()
    assert torch.equal(out, want)
    # and the oracle's STATIC quantisation of those values, packed
    oc, os_, _ = orc.quantize(yf, g=g_static)
    assert torch.equal(out, B.nvfp4_gemm_pack_act(U.dev_u8(oc), U.dev_u8(os_)))
    assert np.any(os_ == 0x7E) or M * nq < 4096          # the 0.8 factor does make some block scales clamp
    # records only, no y
    out2 = torch.zeros_like(out)
    B.nvfp4_gemm_packed_quant_out(blob, gw, N, K, xp, gx, M, d_g, n_quant=nq, xpack_out=out2, y=None)
    torch.cuda.synchronize()
    assert torch.equal(out2, want)


def test_fused_output_quantizer_feeds_next_gemm(B):
    """two projections back to back with no quantizer launch in between: GEMM1 (+ fused quantizer) -> GEMM2, against the
    oracle run on GEMM1's BF16 output."""
    M, K1, N1, N2 = 6, 1024, 1536, 640
    c = make_case(M, N1, K1, seed=31)
    w2c, w2s, g2 = U.oracle_weight(N2, N1, 32, 0)
    blob1 = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    blob2 = B.nvfp4_gemm_repack_weight(U.dev_u8(w2c), U.dev_u8(w2s))
    xp = B.nvfp4_gemm_pack_act(U.dev_u8(c["xc"]), U.dev_u8(c["xs"]))
    y1 = torch.zeros((M, N1), dtype=torch.bfloat16, device="cuda")
    g_mid = U.dev_f32(np.float32(0.004))
    mid, _ = B.nvfp4_gemm_packed_quant_out(blob1, U.dev_f32(c["gw"]), N1, K1, xp, U.dev_f32(c["gx"]), M, g_mid, y=y1)
    y2 = B.nvfp4_gemm_packed(blob2, U.dev_f32(g2), N2, N1, mid, g_mid, M, y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    y1f = orc.bf16_bits_to_f32(U.host_bf16_bits(y1))
    oc, os_, og = orc.quantize(y1f, g=np.float32(0.004))
    Y2, A2 = orc.gemv_w4a4(w2c, w2s, g2, oc, os_, og)
    U.check_gemv(U.host_y_f64(y2), Y2, A2, "GEMM2 on records written by GEMM1's epilogue")


def test_gate_up_interleaved_repack_round_trip(B):
    rng = np.random.default_rng(5)
    for N, K in [(128, 256), (1024, 512), (1536, 256)]:
        wc = rng.integers(0, 256, (N, K // 2), dtype=np.uint8)
        ws = rng.integers(0, 0x7F, (N, K // 16), dtype=np.uint8)
        blob = B.nvfp4_gemm_repack_weight_gate_up(U.dev_u8(wc), U.dev_u8(ws))
        c2, s2 = B.nvfp4_gemm_unpack_weight_gate_up(blob, N, K)
        assert np.array_equal(U.host_u8(c2), wc) and np.array_equal(U.host_u8(s2), ws)
        # tile 0 of the interleaved blob = gate rows 0..63 then up rows I..I+63: its first code chunk rows
        plain = U.host_u8(B.nvfp4_gemm_repack_weight(U.dev_u8(np.concatenate([wc[:64], wc[N // 2:N // 2 + 64]])),
                                                     U.dev_u8(np.concatenate([ws[:64], ws[N // 2:N // 2 + 64]]))))
        KS = K // 256
        assert np.array_equal(U.host_u8(blob)[128:128 + KS * 18432], plain[128:128 + KS * 18432])


@pytest.mark.parametrize("M,I,K", [(1, 256, 512), (4, 512, 1024), (8, 1024, 512), (20, 512, 768), (2, 25600, 256), (8, 2560, 5120)])
def test_fused_gate_up_silu_quantizer(B, M, I, K):
    """gate_up GEMM + SiLU*mul + STATIC quantizer in ONE launch == plain GEMM (BF16 gate_up) -> nvfp4_silu_mul_quantize_packed
    (STATIC), byte for byte; h equals nvfp4_silu_mul's; the records feed the down GEMM within the oracle tolerance."""
    N = 2 * I
    c = make_case(M, N, K, seed=I + K + M)
    gw, gx = U.dev_f32(c["gw"] * 4), U.dev_f32(c["gx"])                # scaled up a little: silu sees both of its regimes, |gate| stays < 88
    blob_plain = B.nvfp4_gemm_repack_weight(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    blob_gu = B.nvfp4_gemm_repack_weight_gate_up(U.dev_u8(c["wc"]), U.dev_u8(c["ws"]))
    xp = B.nvfp4_gemm_pack_act(U.dev_u8(c["xc"]), U.dev_u8(c["xs"]))
    y_gu = B.nvfp4_gemm_packed(blob_plain, gw, N, K, xp, gx, M, y_dtype=B.DTYPE_BF16)
    h_ref = torch.empty((M, I), dtype=torch.bfloat16, device="cuda")
    B.nvfp4_silu_mul(y_gu, h_ref)
    torch.cuda.synchronize()
    hf = orc.bf16_bits_to_f32(U.host_bf16_bits(h_ref))
    g_static = U.dev_f32(np.float32(max(float(np.max(np.abs(hf))), 1e-6) / 2688.0 * 0.9))
    want = torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(M, I), dtype=torch.uint8, device="cuda")
    B.nvfp4_silu_mul_quantize_packed(y_gu, xpack=want, gscale=g_static.clone(), gscale_mode=B.GSCALE_STATIC)
    out = torch.zeros_like(want)
    h = torch.zeros((M, I), dtype=torch.bfloat16, device="cuda")
    B.nvfp4_gemm_packed_silu_quant_out(blob_gu, gw, N, K, xp, gx, M, g_static, xpack_out=out, h=h)
    torch.cuda.synchronize()
    assert torch.equal(h, h_ref)
    assert torch.equal(out, want)
    # against the oracle: silu_mul of the BF16 gate_up output (1 BF16 ulp), and the quantisation of h itself exactly
    want_h = orc.silu_mul(orc.bf16_bits_to_f32(U.host_bf16_bits(y_gu)))
    assert np.all(np.abs(U.host_y_f64(h) - want_h) <= np.maximum(np.abs(want_h), 2.0 ** -120) * 2.0 ** -7)
    oc, os_, _ = orc.quantize(hf, g=np.float32(g_static.item()))
    assert torch.equal(out, B.nvfp4_gemm_pack_act(U.dev_u8(oc), U.dev_u8(os_)))
    # records only (no h)
    out2 = torch.zeros_like(want)
    B.nvfp4_gemm_packed_silu_quant_out(blob_gu, gw, N, K, xp, gx, M, g_static, xpack_out=out2, h=None)
    torch.cuda.synchronize()
    assert torch.equal(out2, want)
    # the wrong blob kind must not produce plausible numbers
    hh = torch.zeros((M, I), dtype=torch.bfloat16, device="cuda")
    B.nvfp4_gemm_packed_silu_quant_out(blob_plain, gw, N, K, xp, gx, M, g_static, xpack_out=out2, h=hh)
    assert torch.isnan(hh).all()
    assert torch.isnan(B.nvfp4_gemm_packed(blob_gu, gw, N, K, xp, gx, M, y_dtype=B.DTYPE_F32)).all()
