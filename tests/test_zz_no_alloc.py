"""GPU: nvfp4_gemv_noalloc (the GEMV on the library's built-in scratch array, include/nvfp4.h) against the existing
nvfp4_gemv path with a caller-allocated workspace -- same inputs, two calls in a row, tolerance of the GEMV tests
(north_star: |y - y_ref| <= 1e-3 * sum_k|w_k x_k| + 1e-6), plus the oracle itself.

Collected LAST on purpose (file name): the run is `pytest -x`, a failure here must not hide other tests.
The shapes are chosen so that the scratch is really used: K >= 16384 at M >= 2 takes the stream-K split whose CTAs
meet through the arrival counters and partials of the workspace."""
import ctypes

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
    binding.nvfp4_gemv_set_config(0, 0, 0, 0, 0, 0)        # tuned table, whatever ran before in this process
    binding.nvfp4_set_layout_kparts(0)
    return binding


def _case(B, M, N, K, seed):
    wc, ws, gw = U.oracle_weight(N, K, seed, 0)
    xbits = inputs.make_activation_bits(M, K, seed, 0)
    xc, xs, gx = orc.quantize(orc.bf16_bits_to_f32(xbits))
    Y, A = orc.gemv_w4a4(wc, ws, gw, xc, xs, gx)
    blob = B.nvfp4_repack_weight(U.dev_u8(wc), U.dev_u8(ws))
    return dict(M=M, N=N, K=K, blob=blob, gw=U.dev_f32(gw), xc=U.dev_u8(xc), xs=U.dev_u8(xs), gx=U.dev_f32(gx), Y=Y, A=A,
                xbits=xbits)


def _compare(B, c, dtype, what):
    args = (B.MODE_W4A4, c["blob"], c["gw"], c["N"], c["K"], c["xc"], c["xs"], c["gx"])
    y_new = B.nvfp4_gemv_noalloc(*args, y_dtype=dtype)
    y_old = B.nvfp4_gemv(*args, y_dtype=dtype)
    torch.cuda.synchronize()
    new, old = U.host_y_f64(y_new), U.host_y_f64(y_old)
    tol = orc.tolerance(c["A"])
    assert np.all(np.abs(new - old) <= tol), f"{what}: no-alloc vs workspace path, max err/tol {np.max(np.abs(new - old) / tol):.3g}"
    if dtype == B.DTYPE_F32:
        U.check_gemv(new, c["Y"], c["A"], what + " vs oracle")
    return y_new


def test_noalloc_matches_workspace_path_two_calls_in_a_row(B):
    assert B.lib.nvfp4_gemv_workspace_bytes(4, 1000, 16384) > 4096          # the shapes below do use partials
    a = _case(B, 4, 1000, 16384, seed=21)
    b = _case(B, 2, 520, 16384, seed=22)
    y1 = _compare(B, a, B.DTYPE_F32, "call 1 (M=4, N=1000, K=16384)")
    y2 = _compare(B, b, B.DTYPE_F32, "call 2 (M=2, N=520, K=16384), other shape on the same scratch")
    y3 = _compare(B, a, B.DTYPE_F32, "call 3 = call 1 again")
    assert torch.equal(y1, y3)                                              # stale scratch contents change nothing
    _compare(B, a, B.DTYPE_BF16, "BF16 output")
    del y2


def test_noalloc_back_to_back_without_sync(B):
    """a run of calls on one stream with no host synchronisation in between (each clears, then reuses, the array)."""
    c = _case(B, 8, 640, 16384, seed=23)
    args = (B.MODE_W4A4, c["blob"], c["gw"], c["N"], c["K"], c["xc"], c["xs"], c["gx"])
    ref = B.nvfp4_gemv(*args, y_dtype=B.DTYPE_F32)
    outs = [torch.empty_like(ref) for _ in range(6)]
    for y in outs:
        B.nvfp4_gemv_noalloc(*args, y=y, y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    tol = orc.tolerance(c["A"])
    for y in outs:
        assert np.all(np.abs(U.host_y_f64(y) - U.host_y_f64(ref)) <= tol)
    U.check_gemv(U.host_y_f64(outs[-1]), c["Y"], c["A"], "last of 6 back-to-back calls vs oracle")


def test_noalloc_w4a16_and_small_shape(B):
    """W4A16 mode and a shape that needs no cross-CTA scratch go through the same entry point."""
    c = _case(B, 3, 300, 512, seed=24)
    x = U.dev_bf16_from_bits(c["xbits"])
    y_new = B.nvfp4_gemv_noalloc(B.MODE_W4A16, c["blob"], c["gw"], c["N"], c["K"], x, y_dtype=B.DTYPE_F32)
    y_old = B.nvfp4_gemv(B.MODE_W4A16, c["blob"], c["gw"], c["N"], c["K"], x, y_dtype=B.DTYPE_F32)
    torch.cuda.synchronize()
    assert torch.equal(y_new, y_old)


def test_noalloc_rejects_shapes_beyond_the_scratch(B):
    M, N, K = 8, 151936, 5120                                               # an output head: 97 MB of partials at M = 8
    assert B.lib.nvfp4_gemv_workspace_bytes(M, N, K) > B.NOALLOC_SCRATCH_BYTES
    fake = ctypes.c_void_p(0x1000)                                          # never dereferenced: rejected before any launch
    rc = B.lib.nvfp4_gemv_noalloc(B.MODE_W4A4, fake, fake, N, K, fake, fake, fake, M, K // 2, fake, B.DTYPE_BF16, N, None)
    assert rc == -2
    msg = B.lib.nvfp4_last_cuda_error().decode()
    assert "nvfp4_gemv_noalloc" in msg and str(B.NOALLOC_SCRATCH_BYTES) in msg
