"""Pins for the oracle GEMV.  CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import nvfp4_oracle as O
from test_oracle_quantize import _load, _random_bf16


def _example_B(golden_dir):
    G = _load(os.path.join(golden_dir, "quant_example_B.txt"))
    x = np.array([float(v) for v in G["x0"] + G["x1"]], dtype=np.float32)[None, :]
    return G, x


def test_tiny_worked_gemv(golden_dir):
    G, x = _example_B(golden_dir)
    W = np.concatenate([x, x[:, ::-1]], axis=0)
    wc, ws, gw = O.quantize(W)
    xc, xs, gx = O.quantize(x)
    assert gw == np.float32(2.0 ** -9) and list(ws[0]) == [0x7E, 0x76] and list(ws[1]) == [0x76, 0x7E]
    Y, A = O.gemv_w4a4(wc, ws, gw, xc, xs, gx)
    assert [float(v) for v in Y[0]] == [float(v) for v in G["gemv_w4a4_Y"]]
    assert [float(v) for v in A[0]] == [float(v) for v in G["gemv_w4a4_A"]]
    assert float(Y[0, 0]).hex() == "0x1.2c38800000000p+7" and float(Y[0, 1]).hex() == "-0x1.6f80000000000p+3"
    assert list(O.round_to_bf16(Y)[0]) == [150.0, -11.5]
    Y16, A16 = O.gemv_w4a16(wc, ws, gw, x)
    assert float(Y16[0, 1]) == float(G["gemv_w4a16_Y1"][0]) and float(A16[0, 1]) == float(G["gemv_w4a16_A1"][0])
    assert abs(float(Y16[0, 0]) - 154.92562866) < 1e-7 and A16[0, 0] == Y16[0, 0]


def test_gemv_equals_fraction_brute_force():
    rng = np.random.default_rng(7)
    M, N, K = 3, 5, 64
    X = _random_bf16(rng, M, K)
    W = _random_bf16(rng, N, K, outliers=False) * np.float32(0.02)
    W = O.bf16_bits_to_f32(O.f32_to_bf16_bits(W))
    wc, ws, gw = O.quantize(W)
    xc, xs, gx = O.quantize(X)
    Y, A = O.gemv_w4a4(wc, ws, gw, xc, xs, gx)
    Y16, A16 = O.gemv_w4a16(wc, ws, gw, X)
    wn, xn = O.unpack_codes(wc), O.unpack_codes(xc)

    def val(nib, sc, g, r, k):
        return Fraction(float(g)) * Fraction(O.e4m3_decode_scalar(sc[r, k // 16])) * Fraction(O.e2m1_decode_scalar(nib[r, k]))
    for m in range(M):
        for n in range(N):
            y = sum(val(xn, xs, gx, m, k) * val(wn, ws, gw, n, k) for k in range(K))
            a = sum(abs(val(xn, xs, gx, m, k) * val(wn, ws, gw, n, k)) for k in range(K))
            assert abs(Fraction(float(Y[m, n])) - y) <= Fraction(1, 2 ** 45) * a
            assert abs(Fraction(float(A[m, n])) - a) <= Fraction(1, 2 ** 45) * a
            y16 = sum(Fraction(float(X[m, k])) * val(wn, ws, gw, n, k) for k in range(K))
            a16 = sum(abs(Fraction(float(X[m, k])) * val(wn, ws, gw, n, k)) for k in range(K))
            assert abs(Fraction(float(Y16[m, n])) - y16) <= Fraction(1, 2 ** 45) * a16
            assert abs(Fraction(float(A16[m, n])) - a16) <= Fraction(1, 2 ** 45) * a16
    assert np.all(A >= np.abs(Y)) and np.all(A16 >= np.abs(Y16))


def test_gemv_textbook_special_cases():
    K, N = 96, 4
    ones = np.full((N, K // 2), 0x22, dtype=np.uint8)           # every code = +1.0
    s1 = np.full((N, K // 16), 0x38, dtype=np.uint8)            # every scale = 1.0
    xo = np.full((1, K // 2), 0x22, dtype=np.uint8)
    Y, A = O.gemv_w4a4(ones, s1, np.float32(1), xo, s1[:1], np.float32(1))
    assert np.all(Y == K) and np.all(A == K)
    # one-hot X row picks a dequantised W column
    rng = np.random.default_rng(8)
    wc = rng.integers(0, 256, size=(N, K // 2), dtype=np.uint8)
    ws = rng.integers(0x20, 0x50, size=(N, K // 16), dtype=np.uint8)
    gw = np.float32(0.37)
    vW = O.dequantize(wc, ws, gw)
    for k in (0, 1, 17, 95):
        X = np.zeros((1, K), dtype=np.float32)
        X[0, k] = 1.0
        Y, _ = O.gemv_w4a16(wc, ws, gw, X)
        assert np.array_equal(Y[0], vW[:, k])
        xc, xs, gx = O.quantize(X * np.float32(6.0))            # 6 -> g = 6/2688, code 6.0, scale 448: exact
        Y4, _ = O.gemv_w4a4(wc, ws, gw, xc, xs, gx)
        np.testing.assert_allclose(Y4[0], 6.0 * vW[:, k], rtol=1e-7)   # g = 6/2688 is rounded once in binary32
    # linear in gX*gW
    xc = rng.integers(0, 256, size=(2, K // 2), dtype=np.uint8)
    xs = rng.integers(0x20, 0x50, size=(2, K // 16), dtype=np.uint8)
    Y1, _ = O.gemv_w4a4(wc, ws, np.float32(1), xc, xs, np.float32(1))
    Y2, _ = O.gemv_w4a4(wc, ws, np.float32(0.25), xc, xs, np.float32(8))
    assert np.array_equal(Y2, 2.0 * Y1)


def test_transposed_operand_would_fail():
    # Y[m,n] pairs X row m with W row n; a transposed/row-swapped W changes the tiny example
    rng = np.random.default_rng(9)
    W = _random_bf16(rng, 4, 32)
    X = _random_bf16(rng, 2, 32)
    wc, ws, gw = O.quantize(W)
    Y, _ = O.gemv_w4a16(wc, ws, gw, X)
    assert Y.shape == (2, 4)
    vW = O.dequantize(wc, ws, gw)
    assert np.allclose(Y[1, 2], float(np.dot(X[1].astype(np.float64), vW[2])), rtol=1e-12)


def test_silu_mul():
    gu = np.array([[0.0, 1.0, -2.0, 3.0, 2.0, 0.5, 4.0, -1.0]], dtype=np.float32)
    h = O.silu_mul(gu)
    # literal constants (40-digit decimal arithmetic, not the oracle's expression):
    # silu(1) = 0.73105857863000487925..., silu(-2) = -0.23840584404423517..., silu(3) = 2.85772238046729965...
    want = [0.0, 0.7310585786300048793 * 0.5, -0.2384058440442351119 * 4.0, 2.857722380467299657 * -1.0]
    np.testing.assert_allclose(h[0], want, rtol=4e-16, atol=0)
    # silu(-x) = silu(x) - x (identity of the logistic function), and h is odd in `up`
    x = np.array([[0.375, 2.5, -7.0, 11.0, 1.0, 1.0, 1.0, 1.0]], dtype=np.float32)
    xm = x.copy(); xm[0, :4] = -xm[0, :4]
    np.testing.assert_allclose(O.silu_mul(xm)[0], O.silu_mul(x)[0] - x[0, :4].astype(np.float64), rtol=0, atol=4e-15)
