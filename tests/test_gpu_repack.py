"""GPU: the offline weight repack is a pure permutation (round trip byte-identical) and its
layout is the one the GEMV consumes (a single non-zero code lights exactly one output)."""
import numpy as np
import pytest
import torch

from oracle import nvfp4_oracle as orc
import _gpu_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_13233_b200 import binding
    return binding


@pytest.mark.parametrize("N,K", [(32, 128), (64, 256), (100, 208), (1, 16), (33, 144), (2048, 2048), (5120, 8192)])
def test_round_trip(B, N, K):
    rng = np.random.default_rng(N * 7 + K)
    codes = rng.integers(0, 256, size=(N, K // 2), dtype=np.uint8)
    scales = rng.integers(0, 0x7F, size=(N, K // 16), dtype=np.uint8)
    blob = B.nvfp4_repack_weight(U.dev_u8(codes), U.dev_u8(scales))
    assert blob.numel() == B.nvfp4_repacked_bytes(N, K)
    c2, s2 = B.nvfp4_unpack_weight(blob, N, K)
    torch.cuda.synchronize()
    assert np.array_equal(U.host_u8(c2), codes) and np.array_equal(U.host_u8(s2), scales)
    # a permutation of the canonical bytes plus zero padding: same multiset of byte values
    hb = U.host_u8(blob)[128:]          # cells only (the first 128 bytes are the versioned header)
    want = np.bincount(np.concatenate([codes.ravel(), scales.ravel()]), minlength=256)
    got = np.bincount(hb, minlength=256)
    pad = hb.size - codes.size - scales.size
    want[0] += pad
    assert np.array_equal(got, want)


def test_single_nonzero_code_lights_one_output(B):
    """all lane / vector / word / byte / nibble positions: W has ONE non-zero code at (n,k);
    X = all +1.0 with unit scales -> Y[n'] = value * [n' == n]   (SURVEY 8(c) C6 'Repack')."""
    N, K = 96, 384
    rng = np.random.default_rng(11)
    positions = [(0, 0), (0, 1), (31, 127), (32, 128), (95, 383), (33, 31), (64, 32), (17, 255)]
    positions += [(int(rng.integers(N)), int(rng.integers(K))) for _ in range(40)]
    xc = np.full((1, K // 2), 0x22, dtype=np.uint8)        # every activation = +1.0
    xs = np.full((1, K // 16), 0x38, dtype=np.uint8)       # E4M3 1.0
    one = U.dev_f32(1.0)
    for n, k in positions:
        codes = np.zeros((N, K // 2), dtype=np.uint8)
        code = int(rng.integers(1, 16))
        if code == 8:
            code = 9
        codes[n, k // 2] = code << (4 * (k & 1))
        scales = np.full((N, K // 16), 0x38, dtype=np.uint8)
        scales[n, k // 16] = 0x40                           # 2.0 on the block that holds the code
        blob = B.nvfp4_repack_weight(U.dev_u8(codes), U.dev_u8(scales))
        y = B.nvfp4_gemv(B.MODE_W4A4, blob, one, N, K, U.dev_u8(xc), U.dev_u8(xs), one, y_dtype=B.DTYPE_F32)
        torch.cuda.synchronize()
        want = np.zeros(N)
        want[n] = 2.0 * orc.e2m1_decode_scalar(code)
        assert np.array_equal(U.host_y_f64(y)[0], want), (n, k, code)
