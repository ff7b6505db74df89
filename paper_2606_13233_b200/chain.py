"""Decode-step projection chain of BASELINE.json configs[4]: L layers x {QKV, O, gate_up, down}, W4A4,
distinct NVFP4 weights per layer, `nvfp4_quantize_act` before every projection and SiLU*mul between
gate_up and down, all enqueued on the current stream (capture it in a CUDA graph to time it).

Data flow (R11, R12; there is no attention here, this isolates the projections):
    h [M,H] -> Q -> QKV -> first `o_in` columns -> Q -> O -> Q -> gate_up -> SiLU*mul -> Q -> down -> h'
Product code: uses only the ctypes binding (no oracle, no torch math on the path).
"""
from __future__ import annotations

import math

import torch

from . import binding as B
from . import inputs

QWEN3_32B_DIMS = dict(hidden=5120, qkv=10240, o_in=8192, inter=25600)


class DecodeChain:
    def __init__(self, layers: int, M: int, dims=None, seed: int = 0, device="cuda", fused: bool = False,
                 fused_producer: bool = True, tensor_core: bool = False, static_scales: bool = False,
                 fuse_gate_up: bool = False, records: bool = False):
        # static_scales (tensor-core path only; the paper's deployed flow): every projection's input global
        # scale is fixed by calibrate(), and each GEMM quantises the NEXT projection's input in its own epilogue
        # (nvfp4_gemm_packed_quant_out): 5 launches per layer -- 4 GEMMs + the SiLU*mul/quantize producer
        self.static_scales = static_scales and tensor_core
        # records (CUDA-core path, M = 1, two calls per projection): the quantizers write the GEMV's own activation records
        # (nvfp4_quantize_act_records / nvfp4_silu_mul_quantize_records -> nvfp4_gemv_records), bit-identical outputs
        self.records = records and not tensor_core and not fused and fused_producer and M == 1
        # fuse_gate_up: SiLU*mul + quantize in gate_up's own epilogue (nvfp4_gemm_packed_silu_quant_out, 4 launches per layer).
        # Off by default: measured slower in the chain at every M (profiles/r02_sweep.md) -- the separate producer launch
        # hides under the down GEMM's pipeline fill, while the fused epilogue lengthens gate_up's tail (and for M > 16 its
        # 8-row passes on two of the four epilogue warps outlast a tile's streaming time).
        self.fuse_gate_up = self.static_scales and bool(fuse_gate_up)
        self.tensor_core = tensor_core                # projections on the tcgen05 GEMM (nvfp4_quantize_act_packed +
                                                      # nvfp4_gemm_packed, M <= 128) instead of the CUDA-core GEMV
        if tensor_core:
            fused, fused_producer = False, True
        self.fused = fused                            # one nvfp4_gemv_fused_quant launch per projection
        self.fused_producer = fused_producer          # down's input: nvfp4_silu_mul_quantize (one launch) instead of
                                                      # nvfp4_silu_mul + nvfp4_quantize_act
        d = dict(QWEN3_32B_DIMS if dims is None else dims)
        self.M, self.layers, self.d = M, layers, d
        H, QKV, OIN, I = d["hidden"], d["qkv"], d["o_in"], d["inter"]
        self.shapes = (("qkv", QKV, H), ("o", H, OIN), ("gate_up", 2 * I, H), ("down", H, I))
        self.w = []                                   # per layer: list of (blob, gW tensor, N, K)
        self.canon = []                               # canonical bytes kept only when asked (tests)
        gu_blobs = []                                 # static chain: gate_up again, rows interleaved per tile (fused SiLU*mul epilogue)
        self.gu_blobs = gu_blobs
        for l in range(layers):
            row = []
            for sid, (name, N, K) in enumerate(self.shapes):
                codes, scales, _ = inputs.make_nvfp4_weight_device(N, K, seed=seed * 1000 + l, shape_id=sid + 1,
                                                                   device=device)
                g = 1.0 / (557.0 * math.sqrt(K))       # keeps activations O(1) through the chain
                blob = B.nvfp4_gemm_repack_weight(codes, scales) if tensor_core else B.nvfp4_repack_weight(codes, scales)
                row.append((blob, torch.tensor([g], dtype=torch.float32, device=device), N, K))
                if self.fuse_gate_up and name == "gate_up":
                    gu_blobs.append(B.nvfp4_gemm_repack_weight_gate_up(codes, scales))
                del codes, scales
            self.w.append(row)
        bf, u8 = torch.bfloat16, torch.uint8
        self.h = torch.zeros((M, H), dtype=bf, device=device)            # layer input / output
        self.y_qkv = torch.empty((M, QKV), dtype=bf, device=device)
        self.y_o = torch.empty((M, H), dtype=bf, device=device)
        self.y_gu = torch.empty((M, 2 * I), dtype=bf, device=device)
        self.act = torch.empty((M, I), dtype=bf, device=device)
        kmax = max(K for _, _, K in self.shapes)
        self.xc = torch.empty((M, kmax // 2), dtype=u8, device=device)   # reused NVFP4 activation buffers
        self.xs = torch.empty((M, kmax // 16), dtype=u8, device=device)
        self.gx = torch.zeros(1, dtype=torch.float32, device=device)
        self.xrec = [B.nvfp4_new_xrecords(N, K, device) for _, N, K in self.shapes] if self.records else None
        if tensor_core:
            self.ws = [B.nvfp4_gemm_packed_new_workspace(M, N, K, device) for _, N, K in self.shapes]
            self.xpack = torch.empty(B.lib.nvfp4_gemm_packed_act_bytes(M, kmax), dtype=u8, device=device)
            self.xpack2 = torch.empty(B.lib.nvfp4_gemm_packed_act_bytes(M, kmax), dtype=u8, device=device)
            self.gs = [[torch.zeros(1, dtype=torch.float32, device=device) for _ in self.shapes] for _ in range(layers)]
        else:
            self.ws = [B.new_workspace(M, N, K, device) for _, N, K in self.shapes]
        self.launches_per_step = layers * ((5 if fused else 8) if fused_producer else (5 if fused else 9))
        if self.static_scales:
            self.launches_per_step = 1 + (4 if self.fuse_gate_up else 5) * layers

    def set_input(self, h_bf16):
        self.h.copy_(h_bf16)

    def _down_from_gate_up(self, l, y, keep_h=False):
        """down projection fed by the fused producer: SiLU*mul + quantize in one launch, then the W4A4 GEMV."""
        blob, gw, N, K = self.w[l][3]
        if self.records:
            B.nvfp4_silu_mul_quantize_records(self.y_gu, self.xrec[3], self.gx, h=self.act if keep_h else None)
            B.nvfp4_gemv_records(blob, gw, N, K, self.xrec[3], self.gx, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[3])
            return
        if self.tensor_core:
            if self.M * K <= 524288:                      # the one-launch producer holds the whole [M, I] tensor in one cluster
                B.nvfp4_silu_mul_quantize_packed(self.y_gu, self.xpack, self.gx, h_out=self.act if keep_h else None)
            else:
                B.nvfp4_silu_mul(self.y_gu, self.act)
                B.nvfp4_quantize_act_packed(self.act, self.xpack, self.gx)
            B.nvfp4_gemm_packed(blob, gw, N, K, self.xpack, self.gx, self.M, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[3])
            return
        xc = self.xc.view(-1)[: self.M * (K // 2)].view(self.M, K // 2)
        xs = self.xs.view(-1)[: self.M * (K // 16)].view(self.M, K // 16)
        B.nvfp4_silu_mul_quantize(self.y_gu, xc, xs, self.gx, h=self.act if keep_h else None)
        B.nvfp4_gemv(B.MODE_W4A4, blob, gw, N, K, xc, xs, self.gx, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[3])

    def _proj(self, l, i, x, y):
        blob, gw, N, K = self.w[l][i]
        if self.records:
            B.nvfp4_quantize_act_records(x, self.xrec[i], self.gx)
            B.nvfp4_gemv_records(blob, gw, N, K, self.xrec[i], self.gx, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[i])
            return
        if self.tensor_core:
            B.nvfp4_quantize_act_packed(x, self.xpack, self.gx)
            B.nvfp4_gemm_packed(blob, gw, N, K, self.xpack, self.gx, self.M, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[i])
            return
        if self.fused:
            B.nvfp4_gemv_fused_quant(blob, gw, N, K, x, self.gx, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[i])
            return
        xc = self.xc.view(-1)[: self.M * (K // 2)].view(self.M, K // 2)
        xs = self.xs.view(-1)[: self.M * (K // 16)].view(self.M, K // 16)
        B.nvfp4_quantize_act(x, xc, xs, self.gx)
        B.nvfp4_gemv(B.MODE_W4A4, blob, gw, N, K, xc, xs, self.gx, y=y, y_dtype=B.DTYPE_BF16, workspace=self.ws[i])

    def _step_static(self, taps=None):
        """tensor-core chain with static activation scales: one quantizer launch for the token's input, then per layer
        QKV(+quant for O) -> O(+quant for gate_up) -> gate_up -> SiLU*mul+quantize -> down(+quant for the next QKV)
        (fuse_gate_up: gate_up(+SiLU*mul+quant for down) in one launch)."""
        d, M, S = self.d, self.M, B.GSCALE_STATIC
        H, OIN, I = d["hidden"], d["o_in"], d["inter"]
        keep = taps is not None
        a, b = self.xpack, self.xpack2
        B.nvfp4_quantize_act_packed(self.h, a, self.gs[0][0], gscale_mode=S)
        for l in range(self.layers):
            (bq, gq, Nq, Kq), (bo, go, No, Ko), (bg, gg, Ng, Kg), (bd, gd, Nd, Kd) = self.w[l]
            x_in = self.h.clone() if keep else None
            B.nvfp4_gemm_packed_quant_out(bq, gq, Nq, Kq, a, self.gs[l][0], M, self.gs[l][1], n_quant=OIN, xpack_out=b,
                                          y=self.y_qkv if keep else None, workspace=self.ws[0])
            B.nvfp4_gemm_packed_quant_out(bo, go, No, Ko, b, self.gs[l][1], M, self.gs[l][2], n_quant=H, xpack_out=a,
                                          y=self.y_o if keep else None, workspace=self.ws[1])
            if keep or not self.fuse_gate_up:             # (fused form: the plain BF16 gate_up output only for the tests)
                B.nvfp4_gemm_packed(bg, gg, Ng, Kg, a, self.gs[l][2], M, y=self.y_gu, y_dtype=B.DTYPE_BF16, workspace=self.ws[2])
            if self.fuse_gate_up:
                B.nvfp4_gemm_packed_silu_quant_out(self.gu_blobs[l], gg, Ng, Kg, a, self.gs[l][2], M, self.gs[l][3], xpack_out=b,
                                                   h=self.act if keep else None, workspace=self.ws[2])
            else:
                B.nvfp4_silu_mul_quantize_packed(self.y_gu, b, self.gs[l][3], gscale_mode=S, h_out=self.act if keep else None)
            if l + 1 < self.layers:
                B.nvfp4_gemm_packed_quant_out(bd, gd, Nd, Kd, b, self.gs[l][3], M, self.gs[l + 1][0], n_quant=H, xpack_out=a,
                                              y=self.h if keep else None, workspace=self.ws[3])
            else:
                B.nvfp4_gemm_packed(bd, gd, Nd, Kd, b, self.gs[l][3], M, y=self.h, y_dtype=B.DTYPE_BF16, workspace=self.ws[3])
            if keep:
                taps.append((l, "qkv", x_in, self.y_qkv.clone()))
                taps.append((l, "o", self.y_qkv[:, :OIN].clone(), self.y_o.clone()))
                taps.append((l, "gate_up", self.y_o.clone(), self.y_gu.clone()))
                taps.append((l, "down", self.act.clone(), self.h.clone()))

    def step(self, taps=None):
        """enqueue the whole chain once; `taps` (tests) collects (layer, name, input clone, output clone)."""
        d = self.d
        if self.static_scales:
            return self._step_static(taps)
        for l in range(self.layers):
            stages = (("qkv", self.h, self.y_qkv), ("o", self.y_qkv[:, : d["o_in"]], self.y_o),
                      ("gate_up", self.y_o, self.y_gu), ("down", self.act, self.h))
            for i, (name, x, y) in enumerate(stages):
                if name == "down" and self.fused_producer:
                    self._down_from_gate_up(l, y, keep_h=taps is not None)
                else:
                    if name == "down":
                        B.nvfp4_silu_mul(self.y_gu, self.act)
                    self._proj(l, i, x, y)
                if taps is not None:
                    taps.append((l, name, x.clone(), y.clone()))

    def calibrate(self, h_bf16):
        """set-up only (synthetic weights, not part of the timed path): walk the chain once and rescale every
        projection's global weight scale so that its output has unit RMS -- keeps activations O(1) through
        all layers whatever M and the input are."""
        d = self.d
        self.h.copy_(h_bf16)
        for l in range(self.layers):
            stages = (("qkv", self.h, self.y_qkv), ("o", self.y_qkv[:, : d["o_in"]], self.y_o),
                      ("gate_up", self.y_o, self.y_gu), ("down", self.act, self.h))
            for i, (name, x, y) in enumerate(stages):
                if name == "down":
                    B.nvfp4_silu_mul(self.y_gu, self.act)
                self._proj(l, i, x, y)
                rms = float(y.float().pow(2).mean().sqrt())
                if rms > 0 and math.isfinite(rms):
                    self.w[l][i][1].div_(rms)
                else:
                    self.w[l][i][1].mul_(2.0 ** -20 if not math.isfinite(rms) else 1.0)
                self._proj(l, i, x, y)
                if self.tensor_core:
                    self.gs[l][i].copy_(self.gx)        # the dynamic scale of this input becomes the static one
        torch.cuda.synchronize()
        self.h.copy_(h_bf16)

    def weight_bytes(self):
        return self.layers * sum(N * K * 9 // 16 for _, N, K in self.shapes)
