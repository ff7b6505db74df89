"""GPU parity of the round-2 additions: per-token activation global scales, the fused
SiLU*mul + quantize producer, the versioned blob header / K-part override, and the Qwen3-8B / 14B projection
shapes of PAPER.md Table 4 (:223-230) as a wider shape set."""
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
    binding.nvfp4_set_layout_kparts(0)
    yield binding
    binding.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)
    binding.nvfp4_set_layout_kparts(0)


# ---- per-token (row-wise) global scales: SURVEY C5 #3 / 8(f)-4 ------------------------------------------------
@pytest.mark.parametrize("M,N,K", [(2, 300, 1296), (5, 1000, 2576), (8, 2048 + 96, 5120), (8, 513, 25600), (1, 64, 16)])
def test_per_row_quantizer_and_rowscale_gemv(B, M, N, K):
    xbits = inputs.make_activation_bits(M, K, 5, M)
    xbits[0] = orc.f32_to_bf16_bits(orc.bf16_bits_to_f32(xbits[0]) * np.float32(0.03125))     # rows of very different size
    x = U.dev_bf16_from_bits(xbits)
    xc, xs, gx = B.nvfp4_quantize_act(x, gscale_mode=B.GSCALE_DYNAMIC_PER_ROW)
    torch.cuda.synchronize()
    assert gx.numel() == M
    rows = [orc.quantize(orc.bf16_bits_to_f32(xbits[m:m + 1])) for m in range(M)]              # each row is its own tensor
    for m, (oc, os_, og) in enumerate(rows):
        assert np.array_equal(U.host_u8(xc)[m:m + 1], oc) and np.array_equal(U.host_u8(xs)[m:m + 1], os_), f"row {m}"
        assert np.float32(gx[m].item()).view(np.uint32) == np.float32(og).view(np.uint32), f"row {m} scale"
    wc, ws, gw = U.oracle_weight(N, K, 5, M)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    for dt in (B.DTYPE_F32, B.DTYPE_BF16):
        y = B.nvfp4_gemv_rowscale(blob, U.dev_f32(gw), N, K, xc, xs, gx, y_dtype=dt)
        torch.cuda.synchronize()
        got = U.host_y_f64(y)
        for m, (oc, os_, og) in enumerate(rows):
            Y, A = orc.gemv_w4a4(wc, ws, gw, oc, os_, og)
            U.check_gemv(got[m:m + 1], Y, A, f"rowscale M={M} row {m}", bf16_slack=(dt == B.DTYPE_BF16 and K < 1000))


def test_per_row_scales_are_batch_invariant(B):
    """with per-token scales a row's codes do not depend on the other rows of the batch (they do with the
    per-tensor scale: DESIGN.md R3)."""
    K = 5120
    xbits = inputs.make_activation_bits(8, K, 6, 1)
    xbits[0] = orc.f32_to_bf16_bits(orc.bf16_bits_to_f32(xbits[0]) * np.float32(24.0))      # another token is much larger
    alone = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits[3:4]), gscale_mode=B.GSCALE_DYNAMIC_PER_ROW)
    batch = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits), gscale_mode=B.GSCALE_DYNAMIC_PER_ROW)
    torch.cuda.synchronize()
    assert torch.equal(alone[0][0], batch[0][3]) and torch.equal(alone[1][0], batch[1][3])
    assert torch.equal(alone[2][0], batch[2][3])
    t_alone = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits[3:4]))
    t_batch = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits))
    assert not torch.equal(t_alone[0][0], t_batch[0][3])          # the per-tensor scale is NOT batch invariant


# ---- fused SiLU*mul + quantize producer: SURVEY 8(f)-1 --------------------------------------------------------
@pytest.mark.parametrize("M,I", [(1, 25600), (4, 25600), (8, 25600), (3, 512), (2, 16)])
@pytest.mark.parametrize("mode", ["dynamic", "per_row", "static"])
def test_silu_mul_quantize(B, M, I, mode):
    rng = np.random.default_rng(M * 1000 + I)
    gu_bits = orc.f32_to_bf16_bits((rng.standard_normal((M, 2 * I)) * 2.0).astype(np.float32))
    gu = U.dev_bf16_from_bits(gu_bits)
    gmode = {"dynamic": B.GSCALE_DYNAMIC, "per_row": B.GSCALE_DYNAMIC_PER_ROW, "static": B.GSCALE_STATIC}[mode]
    g_in = U.dev_f32(0.004) if mode == "static" else None
    h = torch.empty((M, I), dtype=torch.bfloat16, device="cuda")
    fc, fs, fg = B.nvfp4_silu_mul_quantize(gu, gscale=g_in, gscale_mode=gmode, h=h)
    # (1) bit-identical to the two-call path
    h2 = B.nvfp4_silu_mul(gu)
    g_in2 = U.dev_f32(0.004) if mode == "static" else None
    tc, ts, tg = B.nvfp4_quantize_act(h2, gscale=g_in2, gscale_mode=gmode)
    torch.cuda.synchronize()
    assert torch.equal(h, h2) and torch.equal(fc, tc) and torch.equal(fs, ts) and torch.equal(fg, tg)
    # (2) the intermediate is the oracle's SiLU*mul to one BF16 ulp
    want = orc.silu_mul(orc.bf16_bits_to_f32(gu_bits))
    got = U.host_y_f64(h)
    assert np.all(np.abs(got - want) <= np.maximum(np.abs(want), 2.0 ** -120) * 2.0 ** -7)
    # (3) codes / scales / g are the oracle's quantization of that intermediate, bit for bit
    hb = orc.bf16_bits_to_f32(U.host_bf16_bits(h))
    if mode == "per_row":
        for m in range(M):
            oc, os_, og = orc.quantize(hb[m:m + 1])
            assert np.array_equal(U.host_u8(fc)[m:m + 1], oc) and np.array_equal(U.host_u8(fs)[m:m + 1], os_)
            assert np.float32(fg[m].item()).view(np.uint32) == np.float32(og).view(np.uint32)
    else:
        oc, os_, og = orc.quantize(hb, g=np.float32(0.004) if mode == "static" else None)
        assert np.array_equal(U.host_u8(fc), oc) and np.array_equal(U.host_u8(fs), os_)
        assert np.float32(fg.item()).view(np.uint32) == np.float32(og).view(np.uint32)


# ---- versioned blob header and explicit K-part count: SURVEY section 5 ----------------------------------------
def test_blob_header_is_validated_on_the_device(B):
    N, K, M = 200, 1296, 3
    wc, ws, gw = U.oracle_weight(N, K, 7, 1)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    hdr = blob[:32].view(torch.int32).cpu().numpy()
    kp = B.nvfp4_get_layout_kparts(N, K)
    assert hdr[0] == 0x3446564E and hdr[1] == (B.nvfp4_version() << 16 | kp) and hdr[2] == N and hdr[3] == K
    assert hdr[4] == 4608
    xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(inputs.make_activation_bits(M, K, 7, 1)))
    y = B.nvfp4_gemv(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, *xq, y_dtype=B.DTYPE_F32)
    assert torch.isfinite(y).all()
    for word, val in ((0, 0x12345678), (1, (1 << 16) | kp), (2, N + 1), (3, K + 16)):      # magic, ABI version, N, K
        bad = blob.clone()
        bad[:16].view(torch.int32)[word] = val
        for mode, args in ((B.MODE_W4A4, xq), (B.MODE_W4A16, (U.dev_bf16_from_bits(inputs.make_activation_bits(M, K, 7, 1)),))):
            for dt in (B.DTYPE_F32, B.DTYPE_BF16):
                y = B.nvfp4_gemv(mode, bad, U.dev_f32(gw), N, K, *args, y_dtype=dt)
                torch.cuda.synchronize()
                assert torch.isnan(y).all(), f"header word {word} not checked"
    # a blob repacked under another K-part count is rejected too (never misread)
    try:
        B.nvfp4_set_layout_kparts(2 if kp != 2 else 4)
        other = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    finally:
        B.nvfp4_set_layout_kparts(0)
    big = torch.zeros(max(other.numel(), blob.numel()) + 4608 * 8, dtype=torch.uint8, device="cuda")
    big[: other.numel()] = other
    y = B.nvfp4_gemv(B.MODE_W4A4, big, U.dev_f32(gw), N, K, *xq, y_dtype=B.DTYPE_F32)
    assert torch.isnan(y).all()


@pytest.mark.parametrize("kp", [1, 2, 4, 8, 16, 32])
def test_every_kpart_layout_computes_the_same(B, kp):
    N, K, M = 333, 2576, 5
    wc, ws, gw = U.oracle_weight(N, K, 8, kp)
    xbits = inputs.make_activation_bits(M, K, 8, kp)
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    Y, A = orc.gemv_w4a4(wc, ws, gw, oxc, oxs, ogx)
    try:
        B.nvfp4_set_layout_kparts(kp)
        assert B.nvfp4_get_layout_kparts(N, K) == kp
        blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
        assert blob.numel() == B.nvfp4_repacked_bytes(N, K)
        c2, s2 = B.nvfp4_unpack_weight(blob, N, K)
        assert np.array_equal(U.host_u8(c2), wc) and np.array_equal(U.host_u8(s2), ws)
        xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits))
        for balance in (1, 2):
            B.nvfp4_gemv_set_config(0, 0, 0, 0, 0, balance)
            y = B.nvfp4_gemv(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, *xq, y_dtype=B.DTYPE_F32)
            torch.cuda.synchronize()
            U.check_gemv(U.host_y_f64(y), Y, A, f"kp={kp} balance={balance}")
    finally:
        B.nvfp4_set_layout_kparts(0)
        B.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)


# ---- the other projection shapes of PAPER.md Table 4 (Qwen3-8B, Qwen3-14B) -------------------------------------
TABLE4_OTHER = [("8b_qkv", 6144, 4096), ("8b_o", 4096, 4096), ("8b_gate_up", 12288, 4096), ("8b_down", 4096, 12288),
                ("14b_qkv", 7168, 5120), ("14b_o", 5120, 5120), ("14b_gate_up", 17408, 5120), ("14b_down", 5120, 17408)]


@pytest.mark.parametrize("name,N,K", TABLE4_OTHER)
@pytest.mark.parametrize("M", [1, 4, 8])
def test_table4_shapes_sampled_rows(B, name, N, K, M):
    SLAB = 256
    sid = 20 + [t[0] for t in TABLE4_OTHER].index(name)
    sc, ss, gw = U.oracle_weight(SLAB, K, 0, sid)
    idx = (np.arange(N) % SLAB + 37 * (np.arange(N) // SLAB)) % SLAB
    d_idx = torch.from_numpy(idx).cuda()
    blob = B.nvfp4_repack_weight(U.dev_u8(sc)[d_idx].contiguous(), U.dev_u8(ss)[d_idx].contiguous())
    xbits = inputs.make_activation_bits(M, K, 0, sid)
    xq = B.nvfp4_quantize_act(U.dev_bf16_from_bits(xbits))
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    rows = np.unique(np.concatenate([np.array([0, 1, 31, 32, N // 2, N - 33, N - 2, N - 1]),
                                     np.random.default_rng(sid).integers(0, N, size=120)]))
    Y, A = orc.gemv_w4a4(sc[idx[rows]], ss[idx[rows]], gw, oxc, oxs, ogx)
    y = B.nvfp4_gemv(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, *xq, y_dtype=B.DTYPE_BF16)
    torch.cuda.synchronize()
    got = U.host_y_f64(y)
    U.check_gemv(got[:, rows], Y, A, f"{name} M={M}")
    same = np.where(idx == idx[0])[0]
    assert np.all(got[:, same] == got[:, same[:1]])
    if M == 1:
        yf = B.nvfp4_gemv_fused_quant(blob, U.dev_f32(gw), N, K, U.dev_bf16_from_bits(xbits), y_dtype=B.DTYPE_BF16)
        assert torch.equal(yf, y)


# ---- any-M entry point (dispatch rule) --------------------------------------------------------
@pytest.mark.parametrize("M", [9, 20, 64])
def test_linear_any_m(B, M):
    N, K = 1000, 2576
    wc, ws, gw = U.oracle_weight(N, K, 9, 3)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    rng = np.random.default_rng(M)
    xf = (rng.standard_normal((M, K)) * rng.choice([0.5, 1.0, 4.0], size=(M, 1))).astype(np.float32)
    xbits = orc.f32_to_bf16_bits(xf)
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits))               # one global scale for the whole [M, K]
    Y, A = orc.gemv_w4a4(wc, ws, gw, oxc, oxs, ogx)
    y = B.nvfp4_linear(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, U.dev_u8(oxc), U.dev_u8(oxs), U.dev_f32(ogx), y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    U.check_gemv(U.host_y_f64(y), Y, A, f"linear w4a4 M={M}")
    y16 = B.nvfp4_linear(B.MODE_W4A16, blob, U.dev_f32(gw), N, K, U.dev_bf16_from_bits(xbits), y_dtype=B.DTYPE_BF16)
    Y2, A2 = orc.gemv_w4a16(wc, ws, gw, orc.bf16_bits_to_f32(xbits))
    U.check_gemv(U.host_y_f64(y16), Y2, A2, f"linear w4a16 M={M}")
    # chunks reproduce the 8-row GEMV exactly
    y8 = B.nvfp4_gemv(B.MODE_W4A4, blob, U.dev_f32(gw), N, K, U.dev_u8(oxc[:8]), U.dev_u8(oxs[:8]), U.dev_f32(ogx), y_dtype=B.DTYPE_F32)
    assert torch.equal(y[:8], y8)


# ---- pinned, device-mapped host buffers (zero-copy; bench.py's e2e form) -----------------------------------------
@pytest.mark.parametrize("M", [1, 5])
def test_pinned_host_activations_and_outputs(B, M):
    """BF16 activations read from, and BF16 outputs written to, pinned HOST memory by the kernels themselves: same bits
    as with device buffers (CUDA-core GEMV and tensor-core GEMM paths)."""
    N, K = 1024 + 32, 2048
    wc, ws, gw = U.oracle_weight(N, K, 5, M)
    d_gw = U.dev_f32(gw)
    xbits = inputs.make_activation_bits(M, K, 5, M)
    x_dev = U.dev_bf16_from_bits(xbits)
    x_pin = torch.from_numpy(xbits.view(np.int16)).view(torch.bfloat16).pin_memory()
    # CUDA-core path
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    c1, s1, g1 = B.nvfp4_quantize_act(x_dev)
    c2, s2, g2 = torch.empty_like(c1), torch.empty_like(s1), torch.zeros_like(g1)
    B.nvfp4_quantize_act(x_pin, c2, s2, g2)
    y_dev = B.nvfp4_gemv(B.MODE_W4A4, blob, d_gw, N, K, c1, s1, g1, y_dtype=B.DTYPE_BF16)
    y_pin = torch.zeros((M, N), dtype=torch.bfloat16).pin_memory()
    B.nvfp4_gemv(B.MODE_W4A4, blob, d_gw, N, K, c2, s2, g2, y=y_pin, y_dtype=B.DTYPE_BF16, workspace=B.new_workspace(M, N, K, "cuda"))
    torch.cuda.synchronize()
    assert torch.equal(c1, c2) and torch.equal(s1, s2) and torch.equal(g1, g2)
    assert torch.equal(y_dev.cpu(), y_pin)
    # tensor-core path (N a multiple of 128 there)
    Nt = 1024
    blob_tc = B.nvfp4_gemm_repack_weight(U.dev_u8(wc[:Nt]), U.dev_u8(ws[:Nt]))
    xp1, gx1 = B.nvfp4_quantize_act_packed(x_dev, xpack=torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(M, K), dtype=torch.uint8, device="cuda"))
    xp2, gx2 = B.nvfp4_quantize_act_packed(x_pin, xpack=torch.zeros(B.lib.nvfp4_gemm_packed_act_bytes(M, K), dtype=torch.uint8, device="cuda"),
                                           gscale=torch.zeros(1, dtype=torch.float32, device="cuda"))
    yt_dev = B.nvfp4_gemm_packed(blob_tc, d_gw, Nt, K, xp1, gx1, M, y_dtype=B.DTYPE_BF16)
    yt_pin = torch.zeros((M, Nt), dtype=torch.bfloat16).pin_memory()
    B.nvfp4_gemm_packed(blob_tc, d_gw, Nt, K, xp2, gx2, M, y=yt_pin, y_dtype=B.DTYPE_BF16,
                        workspace=B.nvfp4_gemm_packed_new_workspace(M, Nt, K, "cuda"))
    torch.cuda.synchronize()
    assert torch.equal(xp1, xp2) and torch.equal(gx1, gx2)
    assert torch.equal(yt_dev.cpu(), yt_pin)


# ---- quantizer -> GEMV through the GEMV's own activation records (M = 1) ------------------------------------------
@pytest.mark.parametrize("N,K", [(2048, 2048), (300, 1296), (64, 16), (1000, 2576), (5120, 8192), (10240, 5120), (512, 25600)])
@pytest.mark.parametrize("mode", ["dynamic", "static"])
def test_gemv_records_equal_canonical_path(B, N, K, mode):
    """nvfp4_quantize_act_records + nvfp4_gemv_records == nvfp4_quantize_act + nvfp4_gemv bit for bit (and so the oracle's
    tolerance holds); ragged K (half-filled last record), K parts > 1 (small N), K slices (long rows)."""
    wc, ws, gw = U.oracle_weight(N, K, 6, 1)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    d_gw = U.dev_f32(gw)
    xbits = inputs.make_activation_bits(1, K, 6, 1)
    x = U.dev_bf16_from_bits(xbits)
    gmode = B.GSCALE_STATIC if mode == "static" else B.GSCALE_DYNAMIC
    g_in = (lambda: U.dev_f32(0.004)) if mode == "static" else (lambda: None)
    c, s, g = B.nvfp4_quantize_act(x, gscale=g_in(), gscale_mode=gmode)
    y_ref = B.nvfp4_gemv(B.MODE_W4A4, blob, d_gw, N, K, c, s, g, y_dtype=B.DTYPE_F32)
    xrec = B.nvfp4_new_xrecords(N, K, "cuda")
    _, g2 = B.nvfp4_quantize_act_records(x, xrec, gscale=g_in(), gscale_mode=gmode)
    y = B.nvfp4_gemv_records(blob, d_gw, N, K, xrec, g2, y_dtype=B.DTYPE_F32)
    yb = B.nvfp4_gemv_records(blob, d_gw, N, K, xrec, g2, y_dtype=B.DTYPE_BF16)
    torch.cuda.synchronize()
    assert torch.equal(g, g2)
    assert torch.equal(y, y_ref)
    assert np.array_equal(U.host_bf16_bits(yb), orc.f32_to_bf16_bits(y.cpu().numpy()))
    oxc, oxs, ogx = orc.quantize(orc.bf16_bits_to_f32(xbits), g=np.float32(0.004) if mode == "static" else None)
    Y, A = orc.gemv_w4a4(wc, ws, gw, oxc, oxs, ogx)
    U.check_gemv(U.host_y_f64(y), Y, A, f"records N={N} K={K} {mode}")
    # a second token through the same (once zero-filled) buffer, under graph replay
    x2 = U.dev_bf16_from_bits(inputs.make_activation_bits(1, K, 7, 1))
    gsc = g_in() if mode == "static" else torch.zeros(1, dtype=torch.float32, device="cuda")
    wsp = B.new_workspace(1, N, K, "cuda")
    B.nvfp4_quantize_act_records(x2, xrec, gscale=gsc, gscale_mode=gmode); B.nvfp4_gemv_records(blob, d_gw, N, K, xrec, gsc, y=y, y_dtype=B.DTYPE_F32, workspace=wsp)
    torch.cuda.synchronize()
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr):
        B.nvfp4_quantize_act_records(x2, xrec, gscale=gsc, gscale_mode=gmode)
        B.nvfp4_gemv_records(blob, d_gw, N, K, xrec, gsc, y=y, y_dtype=B.DTYPE_F32, workspace=wsp)
    gr.replay(); gr.replay(); torch.cuda.synchronize()
    c2, s2, g3 = B.nvfp4_quantize_act(x2, gscale=g_in(), gscale_mode=gmode)
    assert torch.equal(y, B.nvfp4_gemv(B.MODE_W4A4, blob, d_gw, N, K, c2, s2, g3, y_dtype=B.DTYPE_F32))
    with pytest.raises(B.Nvfp4Error):
        B.nvfp4_gemv_records(blob, d_gw, N, K, xrec, gsc, M=2)


def test_silu_mul_quantize_records_equals_two_kernels(B):
    """nvfp4_silu_mul_quantize_records + nvfp4_gemv_records == nvfp4_silu_mul_quantize + nvfp4_gemv bit for bit (down_proj shape)"""
    I, N = 25600, 256
    rng = np.random.default_rng(11)
    gu = U.dev_bf16_from_bits(orc.f32_to_bf16_bits((rng.standard_normal((1, 2 * I)) * 2.0).astype(np.float32)))
    wc, ws, gw = U.oracle_weight(N, I, 8, 1)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws)); d_gw = U.dev_f32(gw)
    h1 = torch.empty((1, I), dtype=torch.bfloat16, device="cuda"); h2 = torch.empty_like(h1)
    c, s, g = B.nvfp4_silu_mul_quantize(gu, h=h1)
    y_ref = B.nvfp4_gemv(B.MODE_W4A4, blob, d_gw, N, I, c, s, g, y_dtype=B.DTYPE_F32)
    xrec = B.nvfp4_new_xrecords(N, I, "cuda")
    _, g2 = B.nvfp4_silu_mul_quantize_records(gu, xrec, h=h2)
    y = B.nvfp4_gemv_records(blob, d_gw, N, I, xrec, g2, y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    assert torch.equal(g, g2) and torch.equal(h1, h2) and torch.equal(y, y_ref)
