#!/usr/bin/env python
"""bench.py -- the NVFP4 GEMV hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--m M] [--impl ours|reference] [--sweep]

A "step" is one pass of the whole hot path over one batch: for each of the four Qwen3-32B
projections (BASELINE.json configs[1]: QKV 10240x5120, O 5120x8192, gate_up 51200x5120,
down 5120x25600) one `nvfp4_quantize_act` (BF16 -> NVFP4, dynamic global scale) followed by one
W4A4 `nvfp4_gemv` with BF16 output, at M rows (default 1).  The step is captured in a CUDA graph
(the paper times with graph replay) and replayed K times between CUDA events.
L2 is cold for the weights: a step streams 274 MB of weights (> 126 MB L2) and two distinct
weight sets alternate, so no weight byte is re-read before ~548 MB of other traffic.

`value` = algorithmic bytes of the step (N*K/2 + N*K/16 + activation + output bytes per
projection, north_star) / time, i.e. achieved GB/s of the whole step including the quantizers.
`roofline` is for the dominant kernel (the GEMV launches alone, timed in their own graph).
`e2e` runs the same step through the public API on pinned HOST buffers: the calls get the host pointers themselves
(pinned memory is device-mapped), so the BF16 activations cross PCIe in the quantizers' loads and the BF16 outputs in the
GEMVs' stores, inside the timed region; the form with explicit H2D / D2H copy nodes is reported beside it (`copy_nodes_*`).
`--impl reference` times the CPU oracle (test infrastructure) on a bounded sample.
The same run also fills `per_m` (the whole BASELINE.json metric: the step and every projection at M = 1, 2, 4, 8, with
W4A16 and cuBLAS BF16 beside the W4A4 numbers), `chain` (configs[4] at M = 1), and `roofline_alu_m8` (the integer
path's FMA-heavy-pipe roofline at M = 8).  `--headline-only` skips those legs.
`--sweep` additionally prints per-shape / per-M tables (cold and warm L2, W4A16, cuBLAS BF16) as
extra lines BEFORE the final JSON line, for profiles/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_13233_b200 import inputs  # noqa: E402

SHAPES = inputs.QWEN3_32B_SHAPES
METRIC = "nvfp4_gemv_achieved_hbm_gbs"
UNIT = "GB/s"
WORKLOAD = "configs[1]: Qwen3-32B qkv/o/gate_up/down projections, W4A4, BF16 out, quantize_act + gemv each"
L2_BYTES = 126 * 1024 * 1024


def algorithmic_bytes(M, N, K, with_quant=False):
    """north_star byte count of one projection: packed W + W scales + activation + output (BF16).
    GEMV alone reads the quantised activation (codes + scales); with the quantizer in front the
    activation bytes are the BF16 input of the quantizer plus its NVFP4 output and the re-read."""
    w = N * K // 2 + N * K // 16
    xq = M * (K // 2 + K // 16)
    y = M * N * 2
    if with_quant:
        return w + M * K * 2 + 2 * xq + y
    return w + xq + y


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.stop = [], threading.Event()
        self.index = index
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self.stop.wait(0.02)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


class Workload:
    """device state of the step: `copies` distinct weight sets, per-projection activation,
    NVFP4 activation, output and workspace buffers."""

    def __init__(self, M, copies=2, mode="w4a4", shapes=SHAPES, records=None):
        import torch
        from paper_2606_13233_b200 import binding as B
        self.torch, self.B, self.M, self.mode, self.shapes = torch, B, M, mode, shapes
        # M = 1, W4A4 on CUDA cores: quantizer -> GEMV through the GEMV's own activation records (nvfp4_quantize_act_records +
        # nvfp4_gemv_records: same arithmetic and bits as nvfp4_quantize_act + nvfp4_gemv, one bulk copy instead of the GEMV's
        # load / decode / store staging).  records=False: the canonical pair.
        self.records = (mode == "w4a4" and M == 1) if records is None else bool(records)
        self.proj = []
        for sid, (name, N, K) in enumerate(shapes, start=1):
            blobs = []
            for c in range(copies):
                codes, scales, g = inputs.make_nvfp4_weight_device(N, K, seed=c, shape_id=sid)
                blobs.append(B.nvfp4_gemm_repack_weight(codes, scales) if mode in ("tc", "w4a16tc") else B.nvfp4_repack_weight(codes, scales))
                del codes, scales
            xbits = inputs.make_activation_bits(M, K, seed=0, shape_id=sid)
            x = torch.from_numpy(xbits.view(np.int16)).cuda().view(torch.bfloat16)
            self.proj.append(dict(
                name=name, N=N, K=K, blobs=blobs, gw=torch.tensor([g], dtype=torch.float32, device="cuda"), x=x,
                x_host=torch.from_numpy(xbits.view(np.int16)).view(torch.bfloat16).pin_memory(),
                y_host=torch.empty((M, N), dtype=torch.bfloat16).pin_memory(),
                xc=torch.empty((M, K // 2), dtype=torch.uint8, device="cuda"),
                xs=torch.empty((M, K // 16), dtype=torch.uint8, device="cuda"),
                gx=torch.zeros(1, dtype=torch.float32, device="cuda"),
                y=torch.empty((M, N), dtype=torch.bfloat16, device="cuda"),
                xp=(torch.empty(B.lib.nvfp4_gemm_packed_act_bytes(M, K), dtype=torch.uint8, device="cuda") if mode == "tc" else None),
                xrec=(B.nvfp4_new_xrecords(N, K, "cuda") if self.records else None),
                ws=(B.nvfp4_gemm_packed_new_workspace(M, N, K, "cuda") if mode == "tc" else
                    torch.zeros(B.lib.nvfp4_gemm_w4a16_workspace_bytes(M, N, K), dtype=torch.uint8, device="cuda") if mode == "w4a16tc"
                    else B.new_workspace(M, N, K))))
        # e2e staging: the step's four activations / outputs as ONE pinned host buffer and ONE device buffer each
        # (element offsets are multiples of 8 BF16 = 16 B), so a step costs one H2D and one D2H copy
        def pack(key, host_key):
            n = sum(p[key].numel() for p in self.proj)
            dev = torch.empty(n, dtype=torch.bfloat16, device="cuda")
            host = torch.empty(n, dtype=torch.bfloat16).pin_memory()
            off = 0
            for p in self.proj:
                k = p[key].numel()
                dev[off:off + k].copy_(p[key].reshape(-1))
                host[off:off + k].copy_(p[host_key].reshape(-1))
                p[key] = dev[off:off + k].view(p[key].shape)
                off += k
            return dev, host
        self.x_all, self.x_all_host = pack("x", "x_host")
        self.y_all, self.y_all_host = pack("y", "y_host")
        # zero-copy form of e2e: the same pinned host buffers seen through per-projection views (pinned memory is mapped
        # into the device's address space, so the kernels can read / write it over PCIe themselves)
        offx = offy = 0
        for p in self.proj:
            kx, ky = p["x"].numel(), p["y"].numel()
            p["x_pinned"] = self.x_all_host[offx:offx + kx].view(p["x"].shape)
            p["y_pinned"] = self.y_all_host[offy:offy + ky].view(p["y"].shape)
            offx += kx; offy += ky
        torch.cuda.synchronize()

    # -- one projection, all on the current stream ------------------------------------------
    def quantize(self, p):
        if self.mode == "tc":
            self.B.nvfp4_quantize_act_packed(p["x"], p["xp"], p["gx"])
        elif self.records:
            self.B.nvfp4_quantize_act_records(p["x"], p["xrec"], p["gx"])
        else:
            self.B.nvfp4_quantize_act(p["x"], p["xc"], p["xs"], p["gx"])

    def gemv(self, p, copy):
        B = self.B
        if self.mode == "tc":          # the tcgen05 GEMM on packed activations
            B.nvfp4_gemm_packed(p["blobs"][copy], p["gw"], p["N"], p["K"], p["xp"], p["gx"], self.M, y=p["y"],
                                y_dtype=B.DTYPE_BF16, workspace=p["ws"])
        elif self.mode == "w4a16tc":   # W4A16 on the tensor cores (activation re-layout + GEMM)
            B.nvfp4_gemm_w4a16(p["blobs"][copy], p["gw"], p["N"], p["K"], p["x"], y=p["y"], y_dtype=B.DTYPE_BF16, workspace=p["ws"])
        elif self.mode == "w4a4" and self.records:
            B.nvfp4_gemv_records(p["blobs"][copy], p["gw"], p["N"], p["K"], p["xrec"], p["gx"], y=p["y"], y_dtype=B.DTYPE_BF16,
                                 workspace=p["ws"])
        elif self.mode == "w4a4":
            B.nvfp4_gemv(B.MODE_W4A4, p["blobs"][copy], p["gw"], p["N"], p["K"], p["xc"], p["xs"], p["gx"],
                         y=p["y"], y_dtype=B.DTYPE_BF16, workspace=p["ws"])
        else:
            B.nvfp4_gemv(B.MODE_W4A16, p["blobs"][copy], p["gw"], p["N"], p["K"], p["x"],
                         y=p["y"], y_dtype=B.DTYPE_BF16, workspace=p["ws"])

    def step(self, copy, quant=True, gemv=True, only=None, fused=False):
        n = 0
        for p in self.proj:
            if only is not None and p["name"] != only:
                continue
            if fused:          # one launch: quantizer inside the GEMV (nvfp4_gemv_fused_quant)
                self.B.nvfp4_gemv_fused_quant(p["blobs"][copy], p["gw"], p["N"], p["K"], p["x"], p["gx"], y=p["y"],
                                              y_dtype=self.B.DTYPE_BF16, workspace=p["ws"])
                n += 1
                continue
            if quant and self.mode in ("w4a4", "tc"):
                self.quantize(p); n += 1
            if gemv:
                self.gemv(p, copy); n += 1
        return n

    def capture(self, ncopies, same_weights=False, **kw):
        """CUDA graph of `ncopies` consecutive steps (one per weight set); returns (graph, launches)."""
        torch = self.torch
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            for c in range(ncopies):
                self.step(0 if same_weights else c, **kw)   # warm-up outside capture (sets func attributes)
        torch.cuda.current_stream().wait_stream(s)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        launches = 0
        with torch.cuda.graph(g):
            for c in range(ncopies):
                launches += self.step(0 if same_weights else c, **kw)
        return g, launches

    def step_e2e(self, copy, zero_copy=False):
        """public-API path from HOST buffers.  zero_copy=False: H2D copy of the activations, quantize, gemv, D2H copy of the
        outputs.  zero_copy=True: the calls get the pinned HOST buffers themselves -- the quantizer reads the BF16 activations
        over PCIe, the projection kernel writes its BF16 outputs into host memory (same bytes across the bus, no copy nodes)."""
        if zero_copy:
            for p in self.proj:
                xd, yd = p["x"], p["y"]
                p["x"], p["y"] = p["x_pinned"], p["y_pinned"]
                try:
                    if self.mode in ("w4a4", "tc"):
                        self.quantize(p)
                    self.gemv(p, copy)
                finally:
                    p["x"], p["y"] = xd, yd
            return
        self.x_all.copy_(self.x_all_host, non_blocking=True)          # H2D: the step's BF16 activations
        for p in self.proj:
            if self.mode in ("w4a4", "tc"):
                self.quantize(p)
            self.gemv(p, copy)
        self.y_all_host.copy_(self.y_all, non_blocking=True)          # D2H: the step's BF16 outputs

    def bytes_step(self, with_quant=True):
        return sum(algorithmic_bytes(self.M, p["N"], p["K"], with_quant) for p in self.proj)


def time_graph(torch, graph, reps, warmup):
    """ms per replay: W untimed replays, then `reps` replays between two events, synchronised."""
    for _ in range(warmup):
        graph.replay()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        graph.replay()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


# ---- CPU oracle legs (test infrastructure; the ONLY place bench.py touches oracle/) ------------
def oracle_sample(M, rows_per_shape):
    """bounded sample of the step for the oracle: the first `rows_per_shape` weight rows of each
    projection (whole K), the full activations.  Returns (seconds, algorithmic bytes, description)."""
    from oracle import nvfp4_oracle as orc
    t_total, bytes_total = 0.0, 0
    for sid, (name, N, K) in enumerate(SHAPES, start=1):
        n = min(rows_per_shape, N)
        rng = np.random.default_rng([0, sid, n])                              # NVFP4-domain weights, same
        wc = rng.integers(0, 256, size=(n, K // 2), dtype=np.uint8)          # recipe as the device generator
        ws = rng.integers(0x64, 0x7F, size=(n, K // 16), dtype=np.uint8)
        gw = np.float32(3.0e-5)
        xf = inputs.bf16_bits_as_f32(inputs.make_activation_bits(M, K, seed=0, shape_id=sid))
        t0 = time.perf_counter()
        xc, xs, gx = orc.quantize(xf)                                        # step a1+a2
        Y, A = orc.gemv_w4a4(wc, ws, gw, xc, xs, gx)                         # steps a3..a7
        orc.round_to_bf16(Y)
        t_total += time.perf_counter() - t0
        bytes_total += algorithmic_bytes(M, n, K, with_quant=True)
    return t_total, bytes_total, f"first min(N, {rows_per_shape}) weight rows of each of the 4 projections, whole K, M={M}"


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info()]
        return max(n) if n else 1
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rows = 4096
    for _ in range(args.warmup):
        oracle_sample(args.m, 32)
    ts, nbytes = [], 0
    for _ in range(args.steps):
        t, nbytes, desc = oracle_sample(args.m, rows)
        ts.append(t)
    t = float(np.mean(ts))
    val = nbytes / t / 1e9
    cores = cpu_threads()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "M": args.m, "sample": desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def max_over_ranks(ms, world, device):
    """replicas-only multi-GPU contract: every rank runs the same step on its own GPU; the job's time is
    the MAX over ranks (one all-reduce of a scalar; there is no data-path collective)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(bytes_per_rank_step, world, ms_step):
    """whole-job throughput of `world` replicas (weak scaling): all ranks' bytes / the slowest rank's time."""
    return world * bytes_per_rank_step / (ms_step * 1e-3) / 1e9


# ---- our arm -----------------------------------------------------------------------------------
MS = (1, 2, 4, 8)                      # BASELINE.json metric: "at M = 1, 2, 4, 8"
TC_MS = (1, 2, 4, 8, 16, 32, 64, 128)  # the tensor-core GEMM is timed beside the GEMV up to M = 128
MIN_REPLAYS = 200                      # timed graph replays, whatever --steps says
HEAVY_LANES_PER_CLK_SM = 64.0          # IDP.4A / FFMA2 / HFMA2 issue rate (profiles/r02_microbench.md)
NUM_SMS = 148


class ShapeBank:
    """>= 4 x L2 of DISTINCT repacked copies of one projection's weight (cold-L2 per-shape timing), shared by every
    M and mode; plus BF16 copies of the same shape for the cuBLAS comparator."""

    def __init__(self, sid, name, N, K):
        import torch
        from paper_2606_13233_b200 import binding as B
        self.torch, self.B, self.sid, self.name, self.N, self.K = torch, B, sid, name, N, K
        wbytes = N * K * 9 // 16
        self.copies = max(2, -(-4 * L2_BYTES // wbytes))
        self.blobs = []
        for c in range(self.copies):
            codes, scales, g = inputs.make_nvfp4_weight_device(N, K, seed=c, shape_id=sid)
            self.blobs.append(B.nvfp4_repack_weight(codes, scales))
            del codes, scales
        self.gw = torch.tensor([g], dtype=torch.float32, device="cuda")

    def time_mode(self, M, mode, reps_total=MIN_REPLAYS):
        """cold-L2 us per call of nvfp4_gemv(mode) at M rows: one graph walks all copies."""
        torch, B, N, K = self.torch, self.B, self.N, self.K
        xbits = inputs.make_activation_bits(M, K, seed=0, shape_id=self.sid)
        x = torch.from_numpy(xbits.view(np.int16)).cuda().view(torch.bfloat16)
        y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
        ws = B.new_workspace(M, N, K)
        if mode == "w4a4rec":      # M = 1: the GEMV fed by activation records (nvfp4_quantize_act_records)
            xrec = B.nvfp4_new_xrecords(N, K, "cuda")
            _, gx = B.nvfp4_quantize_act_records(x, xrec)
            call = lambda b: B.nvfp4_gemv_records(b, self.gw, N, K, xrec, gx, y=y, y_dtype=B.DTYPE_BF16, workspace=ws)
        elif mode == "w4a4":
            xc, xs, gx = B.nvfp4_quantize_act(x)
            call = lambda b: B.nvfp4_gemv(B.MODE_W4A4, b, self.gw, N, K, xc, xs, gx, y=y, y_dtype=B.DTYPE_BF16, workspace=ws)
        else:
            call = lambda b: B.nvfp4_gemv(B.MODE_W4A16, b, self.gw, N, K, x, y=y, y_dtype=B.DTYPE_BF16, workspace=ws)
        for b in self.blobs[:2]:
            call(b)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for b in self.blobs:
                call(b)
        us = time_graph(torch, g, max(3, reps_total // self.copies), 3) / self.copies * 1e3
        del g
        return us

    def time_tensor_core(self, Ms, reps_total=MIN_REPLAYS):
        """cold-L2 us per call of the tcgen05 GEMM (nvfp4_gemm_packed on pre-packed activations) at each M: {M: us}.
        The tensor-core blobs replace the GEMV blobs of this bank (same canonical bytes, other layout)."""
        torch, B, N, K = self.torch, self.B, self.N, self.K
        self.blobs = []
        torch.cuda.empty_cache()
        tcb = []
        for c in range(self.copies):
            codes, scales, _ = inputs.make_nvfp4_weight_device(N, K, seed=c, shape_id=self.sid)
            tcb.append(B.nvfp4_gemm_repack_weight(codes, scales))
            del codes, scales
        out = {}
        self.w4a16_tc = {}
        for M in Ms:
            xbits = inputs.make_activation_bits(min(M, 8), K, seed=0, shape_id=self.sid)
            x = torch.from_numpy(xbits.view(np.int16)).cuda().view(torch.bfloat16)
            x = x.repeat((M + 7) // 8, 1)[:M].contiguous()
            if M <= 32:      # W4A16 on the tensor cores (nvfp4_gemm_w4a16: activation re-layout + GEMM), same rotation
                y16 = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
                ws16 = torch.zeros(B.lib.nvfp4_gemm_w4a16_workspace_bytes(M, N, K), dtype=torch.uint8, device="cuda")
                call16 = lambda b: B.nvfp4_gemm_w4a16(b, self.gw, N, K, x, y=y16, y_dtype=B.DTYPE_BF16, workspace=ws16)
                for b in tcb[:2]:
                    call16(b)
                torch.cuda.synchronize()
                g16 = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g16):
                    for b in tcb:
                        call16(b)
                self.w4a16_tc[M] = time_graph(torch, g16, max(3, reps_total // self.copies), 3) / self.copies * 1e3
                del g16
            xp, gx = B.nvfp4_quantize_act_packed(x)
            y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
            ws = B.nvfp4_gemm_packed_new_workspace(M, N, K, "cuda")
            call = lambda b: B.nvfp4_gemm_packed(b, self.gw, N, K, xp, gx, M, y=y, y_dtype=B.DTYPE_BF16, workspace=ws)
            for b in tcb[:2]:
                call(b)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                for b in tcb:
                    call(b)
            out[M] = time_graph(torch, g, max(3, reps_total // self.copies), 3) / self.copies * 1e3
            del g
        del tcb
        torch.cuda.empty_cache()
        return out

    def time_cublas(self, Ms):
        """torch.matmul (cuBLAS) BF16 on BF16 weights of the same shape, same cold rotation: {M: us}."""
        torch, N, K = self.torch, self.N, self.K
        ncopy = max(2, -(-4 * L2_BYTES // (2 * N * K)))
        Ws = [torch.randn(N, K, device="cuda", dtype=torch.bfloat16) * 0.02 for _ in range(ncopy)]
        out = {}
        for M in Ms:
            x = torch.randn(M, K, device="cuda", dtype=torch.bfloat16)
            y = torch.empty(M, N, device="cuda", dtype=torch.bfloat16)
            for w in Ws:
                torch.matmul(x, w.t(), out=y)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                for w in Ws:
                    torch.matmul(x, w.t(), out=y)
            out[M] = time_graph(torch, g, max(3, 60 // ncopy), 3) / ncopy * 1e3
            del g
        del Ws
        torch.cuda.empty_cache()
        return out


def chain_ms_per_token(M, layers, peak, variants=("two_calls", "fused_quant", "tensor_core")):
    """BASELINE.json configs[4]: `layers` x {QKV, O, gate_up, down} + quantizers + SiLU*mul, distinct weights per layer,
    one CUDA graph; the best of the chain's launch variants is reported with its name.  Variants: the CUDA-core GEMV
    with separate quantizers / with the quantizer fused into the GEMV (M = 1) / with the quantizers writing the GEMV's
    activation records (M = 1), and the tcgen05 GEMM path."""
    import torch
    from paper_2606_13233_b200.chain import DecodeChain
    h0 = torch.from_numpy(inputs.make_activation_bits(M, 5120, 0, 99).view(np.int16)).cuda().view(torch.bfloat16)
    res = {}
    for label in variants:
        fused = label == "fused_quant"
        if fused and M > 1:
            continue
        ch = DecodeChain(layers=layers, M=M, fused=fused, tensor_core=label.startswith("tensor_core"),
                         static_scales=(label == "tensor_core_static"), records=(label == "records"))
        ch.calibrate(h0)
        ch.step()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            ch.set_input(h0)               # every replay is the same token (a 10-80 KB device copy)
            ch.step()
        ms = time_graph(torch, g, 20, 3)
        res[label] = {"ms_per_token": round(ms, 4), "launches": ch.launches_per_step,
                      "frac_of_copy_peak": round(ch.weight_bytes() / ms / 1e6 / peak, 3),
                      "finite": bool(torch.isfinite(ch.h.float()).all())}
        wb = ch.weight_bytes()
        del ch, g
        torch.cuda.empty_cache()
    best = min(res, key=lambda k: res[k]["ms_per_token"])
    return {"M": M, "layers": layers, "weight_gb": round(wb / 1e9, 2), "best": best, **res[best], "variants": res,
            "floor_ms_at_peak": round(wb / peak / 1e6, 3)}


def sampler_us_per_token(V=151936):
    """the ReSET sampler step (reset_sampler_step, Sec. 4) on a Qwen3-sized vocabulary: us per decoded token,
    CUDA-graph replay over 64 distinct logit rows (cold-ish: 39 MB), B = 1 and B = 8 sequences per launch."""
    import torch
    from paper_2606_13233_b200 import binding as B
    out = {"vocab": V, "paper_us_per_token": 100.0, "paper_ref": "PAPER.md:267 (~100 us per token on Qwen3-32B, context)"}
    gen = torch.Generator(device="cuda"); gen.manual_seed(1)
    for nb in (1, 8):
        rows = 64
        z = torch.randn((rows, nb, V), device="cuda", dtype=torch.float32, generator=gen) * 1.5
        z[:, :, :6] += 10.0
        st = B.reset_sampler_new_state(nb)
        tok = torch.empty(nb, dtype=torch.int32, device="cuda")
        B.reset_sampler_step(z[0], st, 0.5363, 0.3, 1.0, token_out=tok)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for r in range(rows):
                B.reset_sampler_step(z[r], st, 0.5363, 0.3, 1.0, 0.95, 32, 198, 7, token_out=tok)
        us = time_graph(torch, g, 10, 3) / rows * 1e3
        out[f"us_per_token_b{nb}"] = round(us, 2)
        del g, z
    out["algorithmic_bytes_per_token"] = V * 4
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peak, peak_src = measured_peak()
    M = args.m
    steps = max(args.steps, 2 * MIN_REPLAYS)         # one replay = 2 steps; never fewer than MIN_REPLAYS replays
    reps = (steps + 1) // 2
    wrep = max(3, (args.warmup + 1) // 2)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def time_step_graphs(wl):
        """(ms/step whole step, ms/step GEMVs alone, ms/step quantizers alone, ms/step fused, launches per replay)"""
        g_step, n_step = wl.capture(2)
        g_gemv, _ = wl.capture(2, quant=False)
        g_q, _ = wl.capture(2, gemv=False)
        g_fused, _ = wl.capture(2, fused=True)
        t = [time_graph(torch, g, reps, wrep) / 2 for g in (g_step, g_gemv, g_q, g_fused)]
        return t[0], t[1], t[2], t[3], n_step

    # ---- headline: the configs[1] step at M rows (default 1) -------------------------------------------------
    wl = Workload(M, copies=2)
    barrier()
    with ClockSampler(local) as clk:
        ms_step, ms_gemv, ms_q, ms_fused, n_step = time_step_graphs(wl)
    barrier()
    ms_step = max_over_ranks(ms_step, world, "cuda")
    canonical = None
    if wl.records and rank == 0:       # the same step through the canonical pair (nvfp4_quantize_act + nvfp4_gemv), for reference
        wc_ = Workload(M, copies=2, records=False)
        g_c, _ = wc_.capture(2)
        g_cg, _ = wc_.capture(2, quant=False)
        t_c, t_cg = time_graph(torch, g_c, reps, wrep) / 2, time_graph(torch, g_cg, reps, wrep) / 2
        same = all(bool(torch.equal(a["y"], b["y"])) for a, b in zip(wl.proj, wc_.proj))
        canonical = {"what": "same step with nvfp4_quantize_act + nvfp4_gemv (canonical codes / scales between the two)",
                     "ms_per_step": t_c, "gemv_only_ms": t_cg, "outputs_equal": same}
        del wc_, g_c, g_cg
        torch.cuda.empty_cache()

    # end to end through the public API from pinned HOST buffers, all transfers inside the timed region.  Three forms:
    # copy form as plain stream launches from Python (H2D of the BF16 activations, quantize_act, gemv, D2H of the BF16
    # outputs; launch-latency bound), the same as a CUDA graph (how a serving loop would replay it), and the zero-copy
    # graph (the calls work on the pinned host buffers directly) -- the fastest, reported as `e2e.value`.
    for c in range(max(3, args.warmup)):
        wl.step_e2e(c & 1)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_eager = min(steps, 400)
    e0.record()
    for i in range(n_eager):
        wl.step_e2e(i & 1)
    e1.record()
    barrier()
    ms_e2e_eager = max_over_ranks(e0.elapsed_time(e1) / n_eager, world, "cuda")
    g_e2e = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g_e2e):
        wl.step_e2e(0)
        wl.step_e2e(1)
    barrier()
    ms_e2e_copy = max_over_ranks(time_graph(torch, g_e2e, reps, wrep) / 2, world, "cuda")
    barrier()
    del g_e2e
    # the same step with the pinned HOST buffers handed to the calls themselves (zero-copy: the quantizers read the
    # activations and the projection kernels write the outputs over PCIe; no copy nodes).  Same bits as the copy form.
    torch.cuda.synchronize()
    y_copy_form = wl.y_all_host.clone()
    wl.y_all_host.zero_()
    wl.step_e2e(0, zero_copy=True); wl.step_e2e(1, zero_copy=True)
    torch.cuda.synchronize()
    g_e2e = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g_e2e):
        wl.step_e2e(0, zero_copy=True)
        wl.step_e2e(1, zero_copy=True)
    barrier()
    ms_e2e = max_over_ranks(time_graph(torch, g_e2e, reps, wrep) / 2, world, "cuda")
    barrier()
    torch.cuda.synchronize()
    e2e_same = bool(torch.equal(y_copy_form, wl.y_all_host))
    del g_e2e, y_copy_form

    b_step = wl.bytes_step(with_quant=True)
    b_gemv = wl.bytes_step(with_quant=False)
    value = job_value(b_step, world, ms_step)
    ach = b_gemv / (ms_gemv * 1e-3) / 1e9
    h2d = sum(M * p["K"] * 2 for p in wl.proj)
    d2h = sum(M * p["N"] * 2 for p in wl.proj)
    step_by_m = {M: (ms_step, ms_gemv, ms_q, ms_fused)}
    del wl
    torch.cuda.empty_cache()

    per_m, chain, roofline_alu, sampler, tensor_core = {}, None, None, None, None
    if rank == 0 and not args.headline_only:
        # ---- the whole metric: the step at M = 1, 2, 4, 8; per shape W4A4 / W4A16 / cuBLAS BF16, cold L2 --------
        for m in MS:
            if m not in step_by_m:
                w2 = Workload(m, copies=2)
                step_by_m[m] = time_step_graphs(w2)[:4]
                del w2
                torch.cuda.empty_cache()
        shape_rows = {m: {} for m in MS}
        tc_rows, tc_cross = {}, {}
        for sid, (name, N, K) in enumerate(SHAPES, start=1):
            bank = ShapeBank(sid, name, N, K)
            cub = bank.time_cublas(MS)
            for m in MS:
                us44 = bank.time_mode(m, "w4a4")
                us416 = bank.time_mode(m, "w4a16")
                nb44 = algorithmic_bytes(m, N, K)
                nb416 = N * K * 9 // 16 + m * K * 2 + m * N * 2
                shape_rows[m][name] = {
                    "us": round(us44, 2), "gbs": round(nb44 / us44 / 1e3, 1), "frac": round(nb44 / us44 / 1e3 / peak, 3),
                    "w4a16_us": round(us416, 2), "w4a16_frac": round(nb416 / us416 / 1e3 / peak, 3),
                    "cublas_bf16_us": round(cub[m], 2), "copies": bank.copies}
                if m == 1:
                    usr = bank.time_mode(1, "w4a4rec")
                    shape_rows[m][name]["records_us"] = round(usr, 2)
                    shape_rows[m][name]["records_frac"] = round(nb44 / usr / 1e3 / peak, 3)
            tc = bank.time_tensor_core(TC_MS)
            for m in TC_MS:
                nb = N * K * 9 // 16 + m * (K // 2 + K // 16) + m * N * 2
                tc_rows.setdefault(str(m), {})[name] = {"us": round(tc[m], 2), "frac": round(nb / tc[m] / 1e3 / peak, 3)}
                if m in shape_rows:
                    shape_rows[m][name]["tensor_core_us"] = round(tc[m], 2)
                    shape_rows[m][name]["w4a16_tensor_core_us"] = round(bank.w4a16_tc[m], 2)
                if m in bank.w4a16_tc:
                    tc_rows[str(m)][name]["w4a16_us"] = round(bank.w4a16_tc[m], 2)
            wins = [m for m in MS if tc[m] < shape_rows[m][name]["us"]]
            tc_cross[name] = min(wins) if wins else None
            del bank
            torch.cuda.empty_cache()
        tc_step = {}
        for m in MS:
            w2 = Workload(m, copies=2, mode="tc")
            g_s, _ = w2.capture(2)
            g_g, _ = w2.capture(2, quant=False)
            tc_step[m] = (time_graph(torch, g_s, reps, wrep) / 2, time_graph(torch, g_g, reps, wrep) / 2)
            if m == M:      # end to end from pinned host buffers on the tensor-core path, as for the headline
                g_e = torch.cuda.CUDAGraph()
                w2.step_e2e(0, zero_copy=True); w2.step_e2e(1, zero_copy=True); torch.cuda.synchronize()
                with torch.cuda.graph(g_e):
                    w2.step_e2e(0, zero_copy=True)
                    w2.step_e2e(1, zero_copy=True)
                tc_e2e_ms = time_graph(torch, g_e, reps, wrep) / 2
                del g_e
            del w2, g_s, g_g
            torch.cuda.empty_cache()
        for m in MS:
            t_step, t_gemv, t_q, t_fused = step_by_m[m]
            bs = sum(algorithmic_bytes(m, N, K, True) for _, N, K in SHAPES)
            bg = sum(algorithmic_bytes(m, N, K, False) for _, N, K in SHAPES)
            per_m[str(m)] = {"ms_per_step": round(t_step, 5), "value": round(bs / (t_step * 1e-3) / 1e9, 1), "unit": UNIT,
                             "gemv_only_ms": round(t_gemv, 5), "gemv_only_frac": round(bg / (t_gemv * 1e-3) / 1e9 / peak, 3),
                             "quantize_only_ms": round(t_q, 5), "fused_step_ms": round(t_fused, 5),
                             "tensor_core_step_ms": round(tc_step[m][0], 5), "tensor_core_gemm_only_ms": round(tc_step[m][1], 5),
                             "tensor_core_gemm_only_frac": round(bg / (tc_step[m][1] * 1e-3) / 1e9 / peak, 3),
                             "per_shape_gemv": shape_rows[m]}
        # ---- ALU roofline of the integer path at M = 8 (derivation in DESIGN.md section 7) ----------
        clk_mhz = clk.summary()["sm_mhz"] or 1965.0
        weights = sum(N * K for _, N, K in SHAPES)
        heavy_per_weight = (8 * 8 + 3 * 8) / 32.0                       # 8 dp4a + 3 packed FP32 per (m, 32 weights)
        ach_alu = heavy_per_weight * weights / (step_by_m[8][1] * 1e-3) / 1e12
        peak_alu = HEAVY_LANES_PER_CLK_SM * NUM_SMS * clk_mhz * 1e6 / 1e12
        roofline_alu = {"bound": "alu", "kernel": "gemv_kernel<W4A4 integer path, M=8> (4 launches per step, timed alone)",
                        "achieved": round(ach_alu, 3), "peak": round(peak_alu, 3), "unit": "T lane-instr/s (FMA-heavy pipe)",
                        "frac": round(ach_alu / peak_alu, 3), "traffic": None,
                        "how": "achieved = (8M dp4a + 3M packed FP32)/32 heavy-pipe lane-instructions per weight x weights/s at "
                               "M = 8; peak = 64 lanes/clk/SM (measured, profiles/r02_microbench.md) x 148 SMs x sampled SM clock",
                        "hbm_frac_same_kernels": per_m["8"]["gemv_only_frac"]}
        sampler = sampler_us_per_token()
        tensor_core = {
            "what": "nvfp4_gemm_packed: tcgen05 kind::mxf4nvf4 block-scaled MMA, weights as the A operand (swap-AB), persistent "
                    "stream-K; same cold-L2 rotation and byte count as per_shape_gemv (SURVEY 8(f) row 3, PAPER.md App. C.3)",
            "per_m": {m: {"per_shape": rows, "sum_us": round(sum(r["us"] for r in rows.values()), 2)} for m, rows in tc_rows.items()},
            "gemv_sum_us": {str(m): round(sum(r["us"] for r in shape_rows[m].values()), 2) for m in MS},
            "e2e_ms_per_step": round(tc_e2e_ms, 5), "e2e_value": round(b_step / (tc_e2e_ms * 1e-3) / 1e9, 1),
            "crossover_M": tc_cross,
            "crossover_note": "smallest M in {1,2,4,8} at which the tensor-core kernel is faster than the CUDA-core GEMV on "
                              "that shape (null: never); the paper's runtime switches at M ~ 16 (PAPER.md:532)",
            "paper_m128_us": {"qkv": 14.94, "o": 12.74, "gate_up_N25600": 24.99, "down": 24.80,
                              "ref": "PAPER.md:570-573 Table 16, B200, another machine: context"}}
        if not args.no_chain:
            try:
                chain = chain_ms_per_token(1, args.layers, peak, variants=("two_calls", "fused_quant", "records"))
                chain["tensor_core_m1"] = chain_ms_per_token(1, args.layers, peak, variants=("tensor_core", "tensor_core_static"))
                chain["tensor_core_m8"] = chain_ms_per_token(8, args.layers, peak, variants=("tensor_core", "tensor_core_static"))
            except Exception as e:                                        # e.g. not enough free memory on a shared GPU
                chain = {"unavailable": str(e)[:200]}

    cpu = None
    if rank == 0 and not args.no_cpu:
        t, nb, desc = oracle_sample(M, 32768)
        cpu = {"value": nb / t / 1e9, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle", "sample": desc,
               "seconds": round(t, 2)}

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": ("f16 (HFMA2, exact in-block) + f32 across blocks" if M == 1 else
                      "int8 (dp4a, exact in-block) + f32 across blocks"), "data": "synthetic",
            "config": {"workload": WORKLOAD, "M": M, "l2": "cold: inputs larger than L2 (274 MB weights per step, "
                       "2 distinct weight sets alternate; L2 = 126 MB); per-shape numbers walk >= 4 x L2 of distinct copies",
                       "timing": f"CUDA graph replay, CUDA events, {reps} timed replays of 2 steps (>= {MIN_REPLAYS} whatever --steps)",
                       "calls": ("nvfp4_quantize_act_records + nvfp4_gemv_records per projection (the GEMV's own activation records "
                                 "between the two; bit-identical to the canonical pair, see canonical_step)" if canonical is not None or M == 1
                                 else "nvfp4_quantize_act + nvfp4_gemv per projection"),
                       "multi_gpu": "replicas only"},
            "canonical_step": canonical,
            "us_per_projection": {"step_mean": round(ms_step * 1e3 / 4, 2), "gemv_mean": round(ms_gemv * 1e3 / 4, 2),
                                  "quantize_mean": round(ms_q * 1e3 / 4, 2),
                                  "per_shape_gemv": per_m.get(str(M), {}).get("per_shape_gemv")},
            "fused_step": {"what": "same step with nvfp4_gemv_fused_quant (quantizer inside the GEMV: 4 launches)",
                           "ms_per_step": ms_fused, "value": job_value(b_step, world, ms_fused), "unit": UNIT},
            "per_m": per_m,
            "chain": chain,
            "sampler": sampler,
            "tensor_core": tensor_core,
            "roofline": {"bound": "hbm", "kernel": "gemv_kernel<W4A4> (4 launches per step, timed alone" + (", fed by activation records)" if M == 1 else ")"),
                         "achieved": ach, "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": ach / peak,
                         "traffic": TRAFFIC_BYTES_PER_STEP.get(M),
                         "traffic_source": TRAFFIC_SOURCE if M in TRAFFIC_BYTES_PER_STEP else None},
            "roofline_alu_m8": roofline_alu,
            "e2e": {"value": job_value(b_step, world, ms_e2e), "unit": UNIT, "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "how": "CUDA graph of the 8 calls on the pinned HOST buffers (zero-copy: the quantizers read the BF16 "
                           "activations and the GEMVs write the BF16 outputs over PCIe inside the timed region)",
                    "outputs_equal_copy_form": e2e_same,
                    "copy_nodes_value": job_value(b_step, world, ms_e2e_copy), "copy_nodes_ms_per_step": ms_e2e_copy,
                    "copy_nodes_how": "CUDA graph of H2D copy + 8 calls on device buffers + D2H copy",
                    "eager_value": job_value(b_step, world, ms_e2e_eager), "eager_ms_per_step": ms_e2e_eager,
                    "eager_how": "the copy form as plain stream launches from Python"},
            "cpu_baseline": cpu,
            "gpu_launches": n_step * reps,
            "clocks": clk.summary(),
        }
        if args.sweep:
            sweep(None, peak)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# per-step DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum of the 4 GEMV launches) from the committed
# `ncu --set full` capture of the same kernels; a constant taken from that file, NOT produced by this run.
TRAFFIC_BYTES_PER_STEP = {1: 279.01e6}
TRAFFIC_SOURCE = ("constant from profiles/r02_ncu_full.md (ncu --set full capture of the 4 GEMV launches of this step; "
                  "algorithmic: 274.4 MB; the tensor-core path: 280.09 MB); not measured by this run")


def sweep(wl0, peak):
    """per-shape x per-M table: cold L2 (rotating >= 4 distinct weight copies, >= 512 MB), warm L2
    (same weight replayed), W4A4 and W4A16, and cuBLAS BF16 (torch.matmul) on the same shapes."""
    import torch
    from paper_2606_13233_b200 import binding as B
    del wl0
    torch.cuda.empty_cache()
    for sid, (name, N, K) in enumerate(SHAPES, start=1):
        wbytes = N * K * 9 // 16
        copies = max(2, -(-4 * L2_BYTES // wbytes))
        for mode in ("w4a4", "w4a16"):
            for M in ((1, 2, 3, 4, 6, 8) if mode == "w4a4" else (1, 2, 4, 8)):
                wl = Workload(M, copies=copies, mode=mode, shapes=((name, N, K),))
                p = wl.proj[0]
                cfg = B.nvfp4_gemv_get_config(B.MODE_W4A4 if mode == "w4a4" else B.MODE_W4A16, M, N, K)
                g_cold, _ = wl.capture(copies, quant=False)
                g_warm, _ = wl.capture(16, same_weights=True, quant=False)      # 16 back-to-back calls, one weight
                g_q, _ = wl.capture(16, same_weights=True, gemv=False) if mode == "w4a4" else (None, 0)
                reps = max(3, 200 // copies)
                us_cold = time_graph(torch, g_cold, reps, 3) / copies * 1e3
                us_warm = time_graph(torch, g_warm, 20, 3) / 16 * 1e3
                us_q = time_graph(torch, g_q, 20, 3) / 16 * 1e3 if g_q is not None else 0.0
                nb = algorithmic_bytes(M, N, K) if mode == "w4a4" else wbytes + M * K * 2 + M * N * 2
                print(json.dumps({"sweep": "nvfp4", "shape": name, "N": N, "K": K, "mode": mode, "M": M, "cfg": cfg,
                                  "us_cold": round(us_cold, 2), "gbs_cold": round(nb / us_cold / 1e3, 1),
                                  "frac_cold": round(nb / us_cold / 1e3 / peak, 3), "us_warm": round(us_warm, 2),
                                  "us_quant": round(us_q, 2), "copies": copies}), flush=True)
                del wl, g_cold, g_warm, g_q, p
                torch.cuda.empty_cache()
        # cuBLAS BF16 on BF16 weights of the same shape (2*N*K bytes): cold rotation and warm
        ncopy = max(2, -(-4 * L2_BYTES // (2 * N * K)))
        Ws = [torch.randn(N, K, device="cuda", dtype=torch.bfloat16) * 0.02 for _ in range(ncopy)]
        for M in (1, 2, 4, 8):
            x = torch.randn(M, K, device="cuda", dtype=torch.bfloat16)
            y = torch.empty(M, N, device="cuda", dtype=torch.bfloat16)
            for w in Ws:
                torch.matmul(x, w.t(), out=y)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                for w in Ws:
                    torch.matmul(x, w.t(), out=y)
            us_cold = time_graph(torch, g, 20, 3) / ncopy * 1e3
            g2 = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g2):
                for _ in range(16):
                    torch.matmul(x, Ws[0].t(), out=y)
            us_warm = time_graph(torch, g2, 20, 3) / 16 * 1e3
            nb = 2 * N * K + 2 * M * K + 2 * M * N
            print(json.dumps({"sweep": "cublas_bf16", "shape": name, "N": N, "K": K, "M": M, "us_cold": round(us_cold, 2),
                              "gbs_cold": round(nb / us_cold / 1e3, 1), "us_warm": round(us_warm, 2)}), flush=True)
            del g, g2
        del Ws
        torch.cuda.empty_cache()


def run_profile(args):
    """no graphs, no events: `steps` plain launches per kernel so that ncu sees ordinary launches."""
    import torch
    shapes = tuple(s for s in SHAPES if args.profile_shape in ("all", s[0]))
    copies = 4 if args.profile_shape != "all" else 2
    wl = Workload(args.m, copies=copies, mode=args.mode, shapes=shapes)
    n = 0
    for i in range(args.warmup + args.steps):
        n += wl.step(i % copies)
    torch.cuda.synchronize()
    print(json.dumps({"profile_shape": args.profile_shape, "M": args.m, "mode": args.mode, "launches": n}))


# PAPER.md:219-234 Table 4 (M = 1 kernel latency on the paper's B200, us): (model, layer, N, K, vLLM CUTLASS GEMM, paper's GEMV).
# Quoted for context beside this build's numbers; L2 state of the paper's graph replays is not stated.
TABLE4 = (("Qwen3-8B", "qkv", 6144, 4096, 8.69, 4.28), ("Qwen3-8B", "o", 4096, 4096, 7.69, 3.75),
          ("Qwen3-8B", "gate_up", 12288, 4096, 11.45, 6.40), ("Qwen3-8B", "down", 4096, 12288, 16.61, 6.66),
          ("Qwen3-14B", "qkv", 7168, 5120, 10.79, 5.53), ("Qwen3-14B", "o", 5120, 5120, 9.08, 4.64),
          ("Qwen3-14B", "gate_up", 17408, 5120, 14.93, 9.49), ("Qwen3-14B", "down", 5120, 17408, 23.77, 10.35),
          ("Qwen3-32B", "qkv", 10240, 5120, 13.41, 6.62), ("Qwen3-32B", "o", 5120, 8192, 12.40, 7.73),
          ("Qwen3-32B", "gate_up", 25600, 5120, 25.89, 13.25), ("Qwen3-32B", "down", 5120, 25600, 33.26, 15.00))


def run_table4(args):
    """the twelve shapes of the paper's Table 4 at M = 1: CUDA-core GEMV and tensor-core GEMM, cold L2 (rotation over
    >= 4 x L2 of distinct weight copies, this repo's protocol) and warm L2 (one weight set replayed, which is what a
    graph replay of a single shape measures); one JSON line per shape."""
    import torch
    from paper_2606_13233_b200 import binding as B
    peak, _ = measured_peak()
    for sid, (model, layer, N, K, vllm_us, paper_us) in enumerate(TABLE4, start=20):
        bank = ShapeBank(sid, layer, N, K)
        cold = bank.time_mode(1, "w4a4")
        xbits = inputs.make_activation_bits(1, K, seed=0, shape_id=sid)
        x = torch.from_numpy(xbits.view(np.int16)).cuda().view(torch.bfloat16)
        y = torch.empty((1, N), dtype=torch.bfloat16, device="cuda")

        def warm_us(call, n=32):
            call(); torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                for _ in range(n):
                    call()
            us = time_graph(torch, g, max(3, MIN_REPLAYS // n), 3) / n * 1e3
            del g
            return us
        xc, xs, gx = B.nvfp4_quantize_act(x)
        ws = B.new_workspace(1, N, K)
        b0 = bank.blobs[0]
        warm = warm_us(lambda: B.nvfp4_gemv(B.MODE_W4A4, b0, bank.gw, N, K, xc, xs, gx, y=y, y_dtype=B.DTYPE_BF16, workspace=ws))
        quant = warm_us(lambda: B.nvfp4_quantize_act(x, xc, xs, gx))
        tc_cold = bank.time_tensor_core([1])[1]                      # (replaces the bank's GEMV blobs by tensor-core blobs)
        codes, scales, _ = inputs.make_nvfp4_weight_device(N, K, seed=0, shape_id=sid)
        tb = B.nvfp4_gemm_repack_weight(codes, scales)
        del codes, scales
        xp, gxp = B.nvfp4_quantize_act_packed(x)
        wst = B.nvfp4_gemm_packed_new_workspace(1, N, K, "cuda")
        tc_warm = warm_us(lambda: B.nvfp4_gemm_packed(tb, bank.gw, N, K, xp, gxp, 1, y=y, y_dtype=B.DTYPE_BF16, workspace=wst))
        wb = algorithmic_bytes(1, N, K, False)
        print(json.dumps({"table4": model, "layer": layer, "N": N, "K": K, "M": 1,
                          "gemv_cold_us": round(cold, 2), "gemv_cold_frac": round(wb / cold / 1e3 / peak, 3),
                          "gemv_warm_us": round(warm, 2), "tc_cold_us": round(tc_cold, 2), "tc_cold_frac": round(wb / tc_cold / 1e3 / peak, 3),
                          "tc_warm_us": round(tc_warm, 2), "quantize_us": round(quant, 2),
                          "paper_gemv_us": paper_us, "paper_vllm_cutlass_us": vllm_us}), flush=True)
        del bank, tb
        torch.cuda.empty_cache()


def run_chain(args):
    """BASELINE.json configs[4]: 64 layers x 4 projections (+ quantizers + SiLU*mul), distinct weights per
    layer (17.5 GB, every call HBM-cold), one CUDA graph per M; prints one JSON line per M."""
    import torch
    from paper_2606_13233_b200.chain import DecodeChain
    peak, _ = measured_peak()
    for M, fused, producer, tc in ((1, False, True, 0), (2, False, True, 0), (4, False, True, 0), (8, False, True, 0),
                                   (1, True, True, 0), (1, False, False, 0), (1, True, False, 0), (1, False, True, -1),
                                   (1, False, True, 1), (2, False, True, 1), (4, False, True, 1), (8, False, True, 1), (32, False, True, 1),
                                   (1, False, True, 2), (2, False, True, 2), (4, False, True, 2), (8, False, True, 2), (16, False, True, 2), (32, False, True, 2),
                                   (1, False, True, 3), (2, False, True, 3), (4, False, True, 3), (8, False, True, 3), (16, False, True, 3), (32, False, True, 3)):
        # tc: 0 = CUDA-core GEMV, 1 = tensor-core GEMM with quantizer launches, 2 = tensor-core GEMM, static scales, quantizers fused
        # into the GEMM epilogues (gate_up: own launch for SiLU*mul+quantize), 3 = 2 with SiLU*mul+quantize in gate_up's epilogue too
        # tc = -1: the CUDA-core chain through the GEMV's activation records (M = 1)
        ch = DecodeChain(layers=args.layers, M=M, fused=fused, fused_producer=producer, tensor_core=tc > 0, static_scales=tc >= 2,
                         fuse_gate_up=tc == 3, records=tc == -1)
        h0 = torch.from_numpy(inputs.make_activation_bits(M, 5120, 0, 99).view(np.int16)).cuda().view(torch.bfloat16)
        ch.calibrate(h0)
        ch.step()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            ch.set_input(h0)               # every replay is the same token (a 10-80 KB device copy)
            ch.step()
        ms = time_graph(torch, g, 20, 3)
        finite = bool(torch.isfinite(ch.h.float()).all())
        wb = ch.weight_bytes()
        print(json.dumps({"chain": "qwen3-32b projections", "layers": args.layers, "M": M, "fused_quant": fused, "fused_producer": producer, "tensor_core": tc, "ms_per_token": round(ms, 4),
                          "us_per_layer": round(ms * 1e3 / args.layers, 2), "weight_gb": round(wb / 1e9, 2),
                          "gbs": round(wb / ms / 1e6, 1), "frac_of_copy_peak": round(wb / ms / 1e6 / peak, 3),
                          "launches": ch.launches_per_step, "finite": finite}), flush=True)
        del ch, g
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--m", type=int, default=1, help="activation rows M (1..8)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sweep", action="store_true", help="also print per-shape / per-M / cuBLAS tables")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-chain", action="store_true", help="skip the configs[4] decode-chain leg (17.5 GB of weights)")
    ap.add_argument("--headline-only", action="store_true", help="only the configs[1] step at --m rows (no per_m table)")
    ap.add_argument("--profile-shape", default=None, help="qkv|o|gate_up|down|all: plain stream launches of "
                    "quantize_act + gemv on that shape only (for ncu); prints a short JSON line")
    ap.add_argument("--mode", default="w4a4", choices=["w4a4", "w4a16", "tc", "w4a16tc"], help="profile leg: CUDA-core W4A4 / W4A16 GEMV, tc = the tcgen05 W4A4 GEMM path, w4a16tc = the tensor-core W4A16 GEMM")
    ap.add_argument("--chain", action="store_true", help="configs[4]: decode-step projection chain, M = 1,2,4,8")
    ap.add_argument("--layers", type=int, default=64)
    ap.add_argument("--table4", action="store_true", help="the paper's Table 4 shapes (Qwen3-8B / 14B / 32B) at M = 1, cold and warm L2")
    args = ap.parse_args()
    if args.profile_shape:
        return run_profile(args)
    if args.chain:
        return run_chain(args)
    if args.table4:
        return run_table4(args)
    if args.impl == "reference":
        if args.steps == 2000 and args.warmup == 100:
            args.steps, args.warmup = 3, 1
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
