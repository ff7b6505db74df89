"""Pins for oracle.quantize / dequantize.  CPU only."""
import os

import numpy as np
import pytest

from oracle import nvfp4_oracle as O


def _load(path):
    out = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, v = line.split(":", 1)
        out[k.strip()] = v.split()
    return out


def _f32bits(x):
    return int(np.float32(x).view(np.uint32))


def test_worked_example_A(golden_dir):
    G = _load(os.path.join(golden_dir, "quant_example_A.txt"))
    x = np.array([float(v) for v in G["x"]], dtype=np.float32)[None, :]
    codes, scales, g = O.quantize(x)
    assert _f32bits(g) == int(G["g_bits"][0], 16)
    assert [int(s) for s in scales[0]] == [int(v, 16) for v in G["scales"]]
    assert [int(c) for c in O.unpack_codes(codes)[0]] == [int(v, 16) for v in G["codes"]]
    assert [int(b) for b in codes[0]] == [int(v, 16) for v in G["packed"]]
    # intermediate values quoted in the fixture's derivation
    assert _f32bits(np.float32(7) / np.float32(6)) == 0x3F955555
    assert _f32bits(g * np.float32(448)) == 0x3F955556


def test_worked_example_B(golden_dir):
    G = _load(os.path.join(golden_dir, "quant_example_B.txt"))
    x = np.array([float(v) for v in G["x0"] + G["x1"]], dtype=np.float32)[None, :]
    assert np.signbit(x[0, 16 + 12])                      # the "-0" survived parsing
    assert np.array_equal(O.bf16_bits_to_f32(O.f32_to_bf16_bits(x)), x)   # all BF16-representable
    assert O.f32_to_bf16_bits(np.float32(0.2)) == 0x3E4D and x[0, 31] == O.bf16_bits_to_f32(np.uint16(0x3E4D))
    codes, scales, g = O.quantize(x)
    assert _f32bits(g) == int(G["g_bits"][0], 16)
    assert [int(s) for s in scales[0]] == [int(v, 16) for v in G["scales"]]
    assert [int(c) for c in O.unpack_codes(codes)[0]] == [int(v, 16) for v in G["codes0"] + G["codes1"]]
    assert [int(b) for b in codes[0]] == [int(v, 16) for v in G["packed"]]
    deq = O.dequantize(codes, scales, g)[0, 16:]
    want = np.array([float(v) for v in G["deq1"]])
    assert np.array_equal(deq, want) and np.array_equal(np.signbit(deq), np.signbit(want))


def test_edge_fp32_sequence_vs_exact_division():
    # tensor amax 28, block-1 amax 3.875: exact u = 62 is an E4M3 tie (-> 64, 0x68) but the
    # binary32 sequence gives u = 61.999996 -> 60 (0x67).  The binary32 sequence is the rule (R2).
    x = np.zeros((1, 32), dtype=np.float32)
    x[0, 0] = 28.0
    x[0, 16] = 3.875
    x[0, 17] = -1.0
    codes, scales, g = O.quantize(x)
    assert _f32bits(g) == 0x3C2AAAAB
    assert list(scales[0]) == [0x7E, 0x67]
    nib = O.unpack_codes(codes)[0]
    assert nib[16] == 0x7 and nib[17] == 0xB              # 3.875/d = 6.2 -> 6 ; -1/d = -1.6 -> -1.5
    # the exact-arithmetic answer differs, proving the test discriminates
    u_exact = (3.875 / 6.0) / (28.0 / 2688.0)
    assert abs(u_exact - 62.0) < 1e-12


def test_edge_subnormal_scales_and_flush():
    x = np.zeros((1, 48), dtype=np.float32)
    x[0, 0] = 2688.0                       # g = 1
    x[0, 16] = 6 * 1.5 * 2.0 ** -9         # u = 1.5*2^-9 : subnormal tie -> 0x02
    x[0, 17] = 2.0 ** -9
    x[0, 32] = 6 * 2.0 ** -11              # u = 2^-11 < 2^-10 -> scale 0 -> block flushed
    x[0, 33] = -6 * 2.0 ** -11
    codes, scales, g = O.quantize(x)
    assert g == np.float32(1.0)
    assert list(scales[0]) == [0x7E, 0x02, 0x00]
    nib = O.unpack_codes(codes)[0]
    # block 1: scale 0x02 = 2^-8 = d; x16/d = 4.5 is nearer 4 (0.5 away) than 6 (1.5 away)
    assert nib[0] == 7
    assert nib[16] == O.e2m1_encode(np.float32(x[0, 16] / 2.0 ** -8)) == 6     # 4.5 -> 4.0 (code 6)
    assert nib[17] == 1                                                       # 0.5
    assert nib[32] == 0 and nib[33] == 0                                      # flushed, sign dropped
    assert np.all(O.dequantize(codes, scales, g)[0, 32:] == 0)


def test_all_zero_and_static_zero():
    x = np.zeros((2, 32), dtype=np.float32)
    codes, scales, g = O.quantize(x)
    assert g == 0 and not codes.any() and not scales.any()
    x[1, 3] = -0.0
    codes, scales, g = O.quantize(x)
    assert g == 0 and not codes.any()
    codes, scales, g = O.quantize(np.ones((1, 16), dtype=np.float32), g=np.float32(0))
    assert g == 0 and not codes.any() and not scales.any()


def _representable_tensor(rng, R, nb, gexp):
    """T = g*s*e with g = 2^gexp, normal E4M3 scales, every block holding a +-6 code and
    one element equal to 6*448*g; such T is BF16-representable (<= 6 significant bits)."""
    codes = rng.integers(0, 16, size=(R, nb * 16), dtype=np.uint8)
    scales = rng.integers(0x08, 0x7F, size=(R, nb), dtype=np.uint8)
    pos = rng.integers(0, 16, size=(R, nb))
    for r in range(R):
        for b in range(nb):
            codes[r, b * 16 + pos[r, b]] = 0x7 if rng.random() < 0.5 else 0xF
    scales[0, 0] = 0x7E
    codes[0, pos[0, 0]] = 0x7
    g = np.float32(2.0 ** gexp)
    packed = (codes[:, 0::2] | (codes[:, 1::2] << 4)).astype(np.uint8)
    T = O.dequantize(packed, scales, g)
    return packed, scales, g, T


@pytest.mark.parametrize("gexp", [-9, 0, 5, -20])
def test_exact_on_representable_inputs_and_idempotent(gexp):
    rng = np.random.default_rng(100 + gexp)
    packed, scales, g, T = _representable_tensor(rng, 5, 7, gexp)
    T32 = T.astype(np.float32)
    assert np.array_equal(T32.astype(np.float64), T)
    assert np.array_equal(O.bf16_bits_to_f32(O.f32_to_bf16_bits(T32)), T32)
    c2, s2, g2 = O.quantize(T32)
    assert g2 == g and np.array_equal(s2, scales)
    # codes identical up to the sign of zero-magnitude codes, which follows the sign of T
    assert np.array_equal(c2, packed)
    c3, s3, g3 = O.quantize(O.dequantize(c2, s2, g2).astype(np.float32))
    assert g3 == g2 and np.array_equal(c3, c2) and np.array_equal(s3, s2)


def _random_bf16(rng, R, K, outliers=True):
    x = rng.standard_normal((R, K)).astype(np.float32)
    if outliers:
        x[:, rng.random(K) < 0.02] *= 20
    return O.bf16_bits_to_f32(O.f32_to_bf16_bits(x))


def test_invariants_scale_permute_negate():
    rng = np.random.default_rng(3)
    T = _random_bf16(rng, 6, 128)
    c, s, g = O.quantize(T)
    for j in (-7, 3, 11):
        c2, s2, g2 = O.quantize((T * np.float32(2.0 ** j)).astype(np.float32))
        assert g2 == np.float32(g * np.float32(2.0 ** j)) and np.array_equal(c2, c) and np.array_equal(s2, s)
    # permute rows
    p = rng.permutation(6)
    c2, s2, g2 = O.quantize(T[p])
    assert g2 == g and np.array_equal(c2, c[p]) and np.array_equal(s2, s[p])
    # permute whole 16-blocks inside rows
    pb = rng.permutation(8)
    Tp = T.reshape(6, 8, 16)[:, pb].reshape(6, 128)
    c2, s2, g2 = O.quantize(Tp)
    assert g2 == g and np.array_equal(s2, s[:, pb])
    assert np.array_equal(c2, c.reshape(6, 8, 8)[:, pb].reshape(6, 64))
    # negate: only sign bits flip (no flushed blocks in this data)
    c2, s2, g2 = O.quantize(-T)
    assert g2 == g and np.array_equal(s2, s) and np.array_equal(c2, c ^ 0x88)


def test_quantize_against_independent_library_pipeline():
    """Same binary32 op sequence, but with ml_dtypes' cast routines doing both roundings:
    an implementation that shares nothing with the nearest-of-table encoders."""
    ml = pytest.importorskip("ml_dtypes")
    rng = np.random.default_rng(4)
    for R, K in ((8, 1024), (3, 4096)):
        T = _random_bf16(rng, R, K)
        T[1, 32:48] = 0                                   # a zero block
        T[2, 64:80] *= np.float32(1e-7)                   # a block whose scale flushes to 0
        T = O.bf16_bits_to_f32(O.f32_to_bf16_bits(T))
        c, s, g = O.quantize(T)
        f32 = np.float32
        g2 = f32(np.max(np.abs(T)) / f32(2688.0))
        Tb = T.reshape(R, K // 16, 16)
        u = ((np.max(np.abs(Tb), axis=2) / f32(6.0)).astype(f32) / g2).astype(f32)
        s2 = np.minimum(u, f32(448)).astype(ml.float8_e4m3fn)
        d = (g2 * s2.astype(f32)).astype(f32)
        with np.errstate(divide="ignore", invalid="ignore"):
            q = (Tb / d[:, :, None]).astype(f32)
        nib = q.astype(ml.float4_e2m1fn).view(np.uint8) & 0xF
        nib = np.where((d == 0)[:, :, None], 0, nib).reshape(R, K).astype(np.uint8)
        assert g2 == g
        assert np.array_equal(s2.view(np.uint8), s)
        assert np.array_equal(nib[:, 0::2] | (nib[:, 1::2] << 4), c)
        assert (s[2, 4] == 0) and not c[2, 32:40].any()


def _tie_tensor():
    """g = 2^-9 exactly; one block per normal E4M3 scale s holding 6*s*g (fixes the block
    scale to s) and the seven E2M1 tie midpoints times s*g (all BF16-representable, <= 7
    significant bits).  True quotients x/d are exactly the midpoints."""
    g = 2.0 ** -9
    mids = np.array([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0])
    sb = np.arange(0x08, 0x7F, dtype=np.uint8)
    s = O.e4m3_decode(sb)
    T = np.zeros((1, 16 * (len(sb) + 1)), dtype=np.float64)
    T[0, 0] = 5.25                                          # = 2688 * 2^-9 -> g = 2^-9
    for i, sv in enumerate(s):
        blk = T[0, 16 * (i + 1): 16 * (i + 2)]
        blk[0] = 6 * sv * g
        blk[1:8] = mids * sv * g
        blk[8:15] = -mids * sv * g
    T32 = T.astype(np.float32)
    assert np.array_equal(T32.astype(np.float64), T)
    assert np.array_equal(O.bf16_bits_to_f32(O.f32_to_bf16_bits(T32)), T32)
    return T32, sb


def test_exact_ties_need_true_division():
    """Mathematically fixed expectation: every quotient is an exact tie -> even code.  IEEE
    division returns the exact quotient; x*(1/d) does not (R2), so a reciprocal-multiply
    quantiser fails this pin."""
    T, sb = _tie_tensor()
    c, s, g = O.quantize(T)
    assert g == np.float32(2.0 ** -9)
    assert np.array_equal(s[0, 1:], sb) and s[0, 0] == 0x7E
    nib = O.unpack_codes(c)[0].reshape(-1, 16)[1:]
    want = np.array([7, 0, 2, 2, 4, 4, 6, 6, 8, 10, 10, 12, 12, 14, 14, 0], dtype=np.uint8)
    assert np.array_equal(nib, np.broadcast_to(want, nib.shape))
    d = (g * O.e4m3_decode(s).astype(np.float32)).astype(np.float32)
    q_alt = (T.reshape(1, -1, 16) * (np.float32(1.0) / d)[:, :, None]).astype(np.float32)
    alt = O.e2m1_encode(q_alt).reshape(-1, 16)[1:]
    assert np.count_nonzero(alt != nib) > 50               # the reciprocal form is a different function


def test_static_global_scale_matches_dynamic_on_row_subset():
    rng = np.random.default_rng(5)
    T = _random_bf16(rng, 16, 256)
    c, s, g = O.quantize(T)
    rows = [3, 7, 12]
    c2, s2, g2 = O.quantize(T[rows], g=g)
    assert g2 == g and np.array_equal(c2, c[rows]) and np.array_equal(s2, s[rows])


def test_dequantize_is_exact_product():
    from fractions import Fraction
    rng = np.random.default_rng(6)
    codes = rng.integers(0, 256, size=(2, 16), dtype=np.uint8)
    scales = rng.integers(0, 0x7F, size=(2, 2), dtype=np.uint8)
    g = np.float32(0.0123)
    v = O.dequantize(codes, scales, g)
    nib = O.unpack_codes(codes)
    for r in range(2):
        for k in range(32):
            want = Fraction(float(g)) * Fraction(O.e4m3_decode_scalar(scales[r, k // 16])) * \
                Fraction(O.e2m1_decode_scalar(nib[r, k]))
            assert Fraction(float(v[r, k])) == want
