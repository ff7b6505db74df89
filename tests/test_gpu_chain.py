"""GPU: the decode-step projection chain (configs[4] data flow) -- every projection of every layer
is checked against the oracle run on that projection's own downloaded input and unpacked weights."""
import numpy as np
import pytest
import torch

from oracle import nvfp4_oracle as orc
from paper_2606_13233_b200 import inputs
import _gpu_util as U

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("M,fused,producer", [(1, False, True), (4, False, True), (1, True, True), (2, True, True),
                                              (3, False, False), (1, True, False)])
def test_chain_small_dims_every_stage(M, fused, producer):
    from paper_2606_13233_b200 import binding as B
    from paper_2606_13233_b200.chain import DecodeChain
    dims = dict(hidden=256, qkv=512, o_in=384, inter=512)
    ch = DecodeChain(layers=3, M=M, dims=dims, seed=5, fused=fused, fused_producer=producer)
    ch.calibrate(U.dev_bf16_from_bits(inputs.make_activation_bits(M, 256, 0, 77)))
    taps = []
    ch.step(taps)
    torch.cuda.synchronize()
    assert len(taps) == 12
    for l, name, x, y in taps:
        i = [s[0] for s in ch.shapes].index(name)
        blob, gw, N, K = ch.w[l][i]
        wc, ws = B.nvfp4_unpack_weight(blob, N, K)
        xf = orc.bf16_bits_to_f32(U.host_bf16_bits(x.contiguous()))
        assert np.all(np.isfinite(xf))
        oxc, oxs, ogx = orc.quantize(xf)
        Y, A = orc.gemv_w4a4(U.host_u8(wc), U.host_u8(ws), np.float32(gw.item()), oxc, oxs, ogx)
        U.check_gemv(U.host_y_f64(y), Y, A, f"layer {l} {name}", bf16_slack=True)      # toy K (256..512): no cancellation, R9
        if name == "gate_up":       # the glue that feeds `down`
            assert np.all(np.isfinite(U.host_y_f64(y)))
            want = orc.silu_mul(orc.bf16_bits_to_f32(U.host_bf16_bits(y)))
            nxt = [t for t in taps if t[0] == l and t[1] == "down"][0][2]
            got = U.host_y_f64(nxt)
            assert np.all(np.abs(got - want) <= np.maximum(np.abs(want), 2.0 ** -120) * 2.0 ** -7)
    # graph replay gives the same bits as the eager run (stateless calls, clean workspaces)
    h0 = U.dev_bf16_from_bits(inputs.make_activation_bits(M, 256, 0, 77))
    ch.set_input(h0); ch.step(); torch.cuda.synchronize()
    ref = ch.h.clone()
    if M == 1 and not fused and producer:
        # the same chain through the GEMV's activation records (nvfp4_*_records): same bits at every stage
        ch2 = DecodeChain(layers=3, M=M, dims=dims, seed=5, records=True)
        assert ch2.records
        ch2.calibrate(h0)
        taps2 = []
        ch2.step(taps2)
        torch.cuda.synchronize()
        for (l, name, x, y), (l2, name2, x2, y2) in zip(taps, taps2):
            assert (l, name) == (l2, name2) and torch.equal(x, x2) and torch.equal(y, y2), (l, name)
        assert torch.equal(ch2.h, ref)
    g = torch.cuda.CUDAGraph()
    ch.set_input(h0)
    with torch.cuda.graph(g):
        ch.step()
    ch.set_input(h0); g.replay(); torch.cuda.synchronize()
    assert torch.equal(ch.h, ref)


@pytest.mark.parametrize("M", [1, 4])
def test_chain_full_size_first_and_last_layer(M):
    """BASELINE.json configs[4] at full size: 64 layers x {QKV, O, gate_up, down} of the Qwen3-32B shapes, distinct
    weights per layer (17.5 GB).  Layer 0's four projections and the last layer's are checked against the oracle
    run on those projections' own downloaded inputs and unpacked weight bytes (sampled rows), tolerance as
    written (no BF16 slack)."""
    from paper_2606_13233_b200 import binding as B
    from paper_2606_13233_b200.chain import DecodeChain
    L = 64
    ch = DecodeChain(layers=L, M=M, seed=9)
    ch.calibrate(U.dev_bf16_from_bits(inputs.make_activation_bits(M, 5120, 0, 78)))
    taps = []
    ch.step(taps)
    torch.cuda.synchronize()
    assert len(taps) == 4 * L
    rng = np.random.default_rng(M)
    for l, name, x, y in taps:
        if l not in (0, L - 1):
            continue
        i = [s[0] for s in ch.shapes].index(name)
        blob, gw, N, K = ch.w[l][i]
        wc, ws = B.nvfp4_unpack_weight(blob, N, K)
        rows = np.unique(np.concatenate([np.array([0, 31, 32, N - 1]), rng.integers(0, N, size=60)]))
        d_rows = torch.from_numpy(rows).cuda()
        hw, hs = U.host_u8(wc[d_rows]), U.host_u8(ws[d_rows])
        del wc, ws
        xf = orc.bf16_bits_to_f32(U.host_bf16_bits(x.contiguous()))
        assert np.all(np.isfinite(xf)) and np.any(xf != 0)
        oxc, oxs, ogx = orc.quantize(xf)
        Y, A = orc.gemv_w4a4(hw, hs, np.float32(gw.item()), oxc, oxs, ogx)
        U.check_gemv(U.host_y_f64(y)[:, rows], Y, A, f"full-size chain layer {l} {name} M={M}")
    assert torch.isfinite(ch.h.float()).all()
    # graph replay of the whole 64-layer chain reproduces the eager bits
    h0 = U.dev_bf16_from_bits(inputs.make_activation_bits(M, 5120, 0, 78))
    ch.set_input(h0); ch.step(); torch.cuda.synchronize()
    ref = ch.h.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        ch.set_input(h0)
        ch.step()
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(ch.h, ref)


@pytest.mark.parametrize("M", [1, 8, 24])
def test_chain_tensor_core_small_dims_every_stage(M):
    """the same chain with every projection on the tcgen05 GEMM (quantize_act_packed / silu_mul_quantize_packed ->
    gemm_packed): each projection against the oracle on its own downloaded input and unpacked weights."""
    from paper_2606_13233_b200 import binding as B
    from paper_2606_13233_b200.chain import DecodeChain
    dims = dict(hidden=512, qkv=768, o_in=512, inter=768)
    ch = DecodeChain(layers=2, M=M, dims=dims, seed=6, tensor_core=True)
    h0 = U.dev_bf16_from_bits(inputs.make_activation_bits(M, 512, 0, 79))
    ch.calibrate(h0)
    taps = []
    ch.step(taps)
    torch.cuda.synchronize()
    assert len(taps) == 8
    for l, name, x, y in taps:
        i = [s[0] for s in ch.shapes].index(name)
        blob, gw, N, K = ch.w[l][i]
        wc, ws = B.nvfp4_gemm_unpack_weight(blob, N, K)
        xf = orc.bf16_bits_to_f32(U.host_bf16_bits(x.contiguous()))
        oxc, oxs, ogx = orc.quantize(xf)
        Y, A = orc.gemv_w4a4(U.host_u8(wc), U.host_u8(ws), np.float32(gw.item()), oxc, oxs, ogx)
        U.check_gemv(U.host_y_f64(y), Y, A, f"tc chain layer {l} {name} M={M}", bf16_slack=True)
    ch.set_input(h0); ch.step(); torch.cuda.synchronize()
    ref = ch.h.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        ch.set_input(h0)
        ch.step()
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(ch.h, ref)


def test_chain_tensor_core_full_size_m8():
    """configs[4] at full size on the tensor-core path, M = 8: first and last layer against the oracle (sampled rows)."""
    from paper_2606_13233_b200 import binding as B
    from paper_2606_13233_b200.chain import DecodeChain
    L, M = 64, 8
    ch = DecodeChain(layers=L, M=M, seed=11, tensor_core=True)
    ch.calibrate(U.dev_bf16_from_bits(inputs.make_activation_bits(M, 5120, 0, 80)))
    taps = []
    ch.step(taps)
    torch.cuda.synchronize()
    rng = np.random.default_rng(8)
    for l, name, x, y in taps:
        if l not in (0, L - 1):
            continue
        i = [s[0] for s in ch.shapes].index(name)
        blob, gw, N, K = ch.w[l][i]
        wc, ws = B.nvfp4_gemm_unpack_weight(blob, N, K)
        rows = np.unique(np.concatenate([np.array([0, 127, 128, N - 1]), rng.integers(0, N, size=60)]))
        d_rows = torch.from_numpy(rows).cuda()
        hw, hs = U.host_u8(wc[d_rows]), U.host_u8(ws[d_rows])
        del wc, ws
        xf = orc.bf16_bits_to_f32(U.host_bf16_bits(x.contiguous()))
        assert np.all(np.isfinite(xf)) and np.any(xf != 0)
        oxc, oxs, ogx = orc.quantize(xf)
        Y, A = orc.gemv_w4a4(hw, hs, np.float32(gw.item()), oxc, oxs, ogx)
        U.check_gemv(U.host_y_f64(y)[:, rows], Y, A, f"full-size tc chain layer {l} {name}")
    assert torch.isfinite(ch.h.float()).all()


@pytest.mark.parametrize("M,fuse", [(1, False), (1, True), (4, True), (8, False), (8, True), (24, False), (24, True)])
def test_chain_tensor_core_static_scales_fused_quantizers(M, fuse):
    """tensor-core chain with static activation scales: no quantizer launches between projections (each GEMM's epilogue
    writes the next GEMM's packed NVFP4 input; with `fuse`, gate_up's also applies SiLU * mul: 4 launches per layer).  Every projection
    is checked against the oracle: quantize(its BF16 input, static g) -> float64 GEMV on the unpacked weights."""
    from paper_2606_13233_b200 import binding as B
    from paper_2606_13233_b200.chain import DecodeChain
    dims = dict(hidden=512, qkv=768, o_in=512, inter=768)
    ch = DecodeChain(layers=3, M=M, dims=dims, seed=8, tensor_core=True, static_scales=True, fuse_gate_up=fuse)
    assert ch.fuse_gate_up == fuse and ch.launches_per_step == 1 + (4 if fuse else 5) * 3
    h0 = U.dev_bf16_from_bits(inputs.make_activation_bits(M, 512, 0, 81))
    ch.calibrate(h0)
    taps = []
    ch.step(taps)
    torch.cuda.synchronize()
    assert len(taps) == 12
    for l, name, x, y in taps:
        i = [s[0] for s in ch.shapes].index(name)
        blob, gw, N, K = ch.w[l][i]
        wc, ws = B.nvfp4_gemm_unpack_weight(blob, N, K)
        xf = orc.bf16_bits_to_f32(U.host_bf16_bits(x.contiguous()))
        g_static = np.float32(ch.gs[l][i].item())
        assert g_static > 0
        oxc, oxs, ogx = orc.quantize(xf, g=g_static)
        Y, A = orc.gemv_w4a4(U.host_u8(wc), U.host_u8(ws), np.float32(gw.item()), oxc, oxs, ogx)
        U.check_gemv(U.host_y_f64(y), Y, A, f"static tc chain layer {l} {name} M={M}", bf16_slack=True)
        if name == "gate_up" and ch.fuse_gate_up:
            # the fused kernel reads the SAME weights from the interleaved blob, and its h (the down tap's input, which the
            # oracle quantizes above) is SiLU(gate) * up of this projection's BF16 output
            wc2, ws2 = B.nvfp4_gemm_unpack_weight_gate_up(ch.gu_blobs[l], N, K)
            assert torch.equal(wc2, wc) and torch.equal(ws2, ws)
            act = torch.empty(M, N // 2, dtype=torch.bfloat16, device="cuda")
            B.nvfp4_silu_mul(y.contiguous(), act)
            assert torch.equal(act, taps[4 * l + 3][2])
    # the timed form (no BF16 outputs between projections) ends on the same bits, eagerly and under graph replay
    ref = ch.h.clone()
    ch.set_input(h0); ch.step(); torch.cuda.synchronize()
    assert torch.equal(ch.h, ref)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        ch.set_input(h0)
        ch.step()
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(ch.h, ref)
