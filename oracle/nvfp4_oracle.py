"""NVFP4 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain, slow, obviously-correct CPU (NumPy) statement of what the hot path of
arxiv/paper_2606_13233 computes: NVFP4 quantisation (an encoding, followed step
by step) and the NVFP4 GEMV (which has a plain definition: a dense matmul of the
exactly dequantised operands, accumulated in float64).

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this module.  It shares no code with the CUDA
path under `paper_2606_13233_b200/` and imports nothing from it.

What it follows
---------------
* Format: PAPER.md:344-349 (App. A, Table 7: NVFP4 = FP4 E2M1 elements, FP8 E4M3
  block scale, FP32 global scale, block size 16), PAPER.md:359 ("block size of
  16 ... block scale in FP8 (E4M3), supplemented by an additional FP32 global
  scale"), PAPER.md:175 (Sec. 6.1: "E2M1 elements, E4M3 block scales, group
  size 16").
* Operation: PAPER.md:143 (Sec. 5: "linear projection Y = XW, X in R^{MxK}, W in
  R^{KxN} at small M"); stored here as W[N,K] row-major by output channel, so
  Y[m,n] = sum_k X[m,k] * W[n,k]  (reading R7).
* Everything the paper leaves out (formula of the global scale g = amax/(6*448),
  of the block scale (amax_b/6)/g, round-to-nearest-even, saturation at +-6 and
  448, nibble order "low nibble = even k", the binary32 operation order) is the
  reading listed in DESIGN.md section "Readings" (R1..R13), taken from
  BASELINE.json north_star / configs[0] and SURVEY.md section 8(c).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed-form value tables,
independent library casts (ml_dtypes, torch), hand-worked 16- and 32-element
examples under tests/golden/, tie and edge cases, exactness on representable
inputs, invariants, brute-force Fraction matmul on tiny shapes.  No function in
this file is "parity unpinned".

Data conventions
----------------
* BF16 tensors are carried as uint16 bit patterns (`bf16 bits`) or as float32
  arrays whose values are BF16-representable; `bf16_bits_to_f32` /
  `f32_to_bf16_bits` convert.
* codes  : uint8 [R, K/2]; byte j of a row holds element k=2j in its LOW nibble
  and k=2j+1 in its HIGH nibble; a nibble is sign-magnitude E2M1 `s e1 e0 m`.
* scales : uint8 [R, K/16]; E4M3 ("fn": no infinities), always in 0x00..0x7E.
* g      : numpy.float32 scalar, the per-tensor global scale.
* dequantised value v[r,k] = g * E4M3(scales[r,k//16]) * E2M1(code[r,k]).
"""
from __future__ import annotations

import numpy as np

F32 = np.float32
BLOCK = 16                      # NVFP4 block size (Table 7)
E2M1_MAX = 6.0                  # largest E2M1 magnitude
E4M3_MAX = 448.0                # largest finite E4M3 ("fn") magnitude
GLOBAL_DIV = F32(6.0 * 448.0)   # g = amax / 2688  (R1)


# --------------------------------------------------------------------------
# C1. codecs -- closed forms (Table 7 names the formats)
# --------------------------------------------------------------------------
def e2m1_decode_scalar(code: int) -> float:
    """E2M1 nibble `s e1 e0 m` -> real value (closed form).

    e == 0: m * 0.5 (subnormal);  e > 0: (1 + m/2) * 2^(e-1);  bit 3 = sign.
    """
    code = int(code) & 0xF
    s = (code >> 3) & 1
    e = (code >> 1) & 3
    m = code & 1
    mag = m * 0.5 if e == 0 else (1.0 + m / 2.0) * 2.0 ** (e - 1)
    return -mag if s else mag


def e4m3_decode_scalar(byte: int) -> float:
    """E4M3 ("fn") byte `s eeee mmm` -> real value (closed form).

    e == 0: (m/8) * 2^-6 (subnormal);  e > 0: (1 + m/8) * 2^(e-7);
    0x7F / 0xFF are NaN (never produced by the quantiser).
    """
    byte = int(byte) & 0xFF
    s = (byte >> 7) & 1
    e = (byte >> 3) & 0xF
    m = byte & 7
    if e == 15 and m == 7:
        return float("nan")
    mag = (m / 8.0) * 2.0 ** -6 if e == 0 else (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return -mag if s else mag


# value tables built from the closed forms above (exact in float64)
E2M1_TABLE = np.array([e2m1_decode_scalar(c) for c in range(16)], dtype=np.float64)
E2M1_MAG = E2M1_TABLE[:8].copy()                       # 0, .5, 1, 1.5, 2, 3, 4, 6
E4M3_TABLE = np.array([e4m3_decode_scalar(b) for b in range(256)], dtype=np.float64)
E4M3_POS = E4M3_TABLE[:0x7F].copy()                    # 0x00..0x7E, increasing


def e2m1_decode(codes: np.ndarray) -> np.ndarray:
    """nibble codes (uint8, values 0..15) -> float64 values."""
    return E2M1_TABLE[np.asarray(codes, dtype=np.uint8) & 0xF]


def e4m3_decode(b: np.ndarray) -> np.ndarray:
    """E4M3 bytes -> float64 values."""
    return E4M3_TABLE[np.asarray(b, dtype=np.uint8)]


def _nearest_even_index(mag: np.ndarray, table: np.ndarray) -> np.ndarray:
    """index of the table entry nearest to each mag >= 0; ties go to the EVEN index.

    `table` is increasing and exact in float64; `mag` is float64 holding
    binary32 values, so every difference below is exact.  This is the plain
    definition of round-to-nearest, ties-to-even-code (the even index is the
    entry whose mantissa LSB is 0, for both E2M1 magnitudes and E4M3 bytes).
    """
    mag = np.asarray(mag, dtype=np.float64)
    out = np.empty(mag.shape, dtype=np.int64)
    flat_in = mag.reshape(-1)
    flat_out = out.reshape(-1)
    chunk = 1 << 16
    for lo in range(0, flat_in.size, chunk):
        x = flat_in[lo:lo + chunk]
        d = np.abs(x[:, None] - table[None, :])          # exact distances
        best = d.min(axis=1)
        is_best = d == best[:, None]
        first = is_best.argmax(axis=1)
        last = table.size - 1 - is_best[:, ::-1].argmax(axis=1)
        # at most two entries tie (they are adjacent); pick the even index
        flat_out[lo:lo + chunk] = np.where(first % 2 == 0, first, last)
    return out


def e2m1_encode(q: np.ndarray) -> np.ndarray:
    """real q (binary32) -> 4-bit sign-magnitude E2M1 code.

    Round to nearest table magnitude, ties to the even code; |q| > 6 saturates
    to 6 (the nearest entry); the sign bit is signbit(q), kept even when the
    magnitude rounds to zero (so -0.0 and tiny negatives give 0x8)  (R4).
    """
    q = np.asarray(q, dtype=F32)
    sign = np.signbit(q).astype(np.uint8)
    mag = np.abs(q.astype(np.float64))
    mag = np.minimum(mag, E2M1_MAX)                      # saturation (inf -> 6)
    idx = _nearest_even_index(mag, E2M1_MAG).astype(np.uint8)
    return (sign << 3) | idx


def e4m3_encode(u: np.ndarray) -> np.ndarray:
    """real u >= 0 (binary32) -> E4M3 byte in 0x00..0x7E.

    Clamp to 448, then round to the nearest representable value (subnormals
    included), ties to the even byte (= even mantissa).
    """
    u = np.asarray(u, dtype=F32).astype(np.float64)
    u = np.minimum(u, E4M3_MAX)
    return _nearest_even_index(u, E4M3_POS).astype(np.uint8)


# --------------------------------------------------------------------------
# BF16 helpers (storage format of the un-quantised tensors)
# --------------------------------------------------------------------------
def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    bits = np.asarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << np.uint32(16)).view(F32)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """binary32 -> BF16 bits, round to nearest even (finite inputs)."""
    u = np.ascontiguousarray(np.asarray(x, dtype=F32)).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = u + np.uint32(0x7FFF) + lsb
    return (r >> np.uint32(16)).astype(np.uint16)


def round_to_bf16(y: np.ndarray) -> np.ndarray:
    """float64 -> nearest BF16 value (returned as float32).  Goes through
    binary32 first only when that is exact enough: to avoid double rounding the
    float64 value is rounded straight to 8 significant bits."""
    y = np.asarray(y, dtype=np.float64)
    m, e = np.frexp(y)                                   # y = m * 2^e, 0.5<=|m|<1
    e = np.maximum(e, -125)                              # binary32/bf16 subnormal floor (2^-133 grid)
    scaled = np.ldexp(y, 8 - e)                          # 8 significant bits
    r = np.rint(scaled)                                  # ties to even
    return np.ldexp(r, e - 8).astype(F32)


def round_to_f32(y: np.ndarray) -> np.ndarray:
    return np.asarray(y, dtype=np.float64).astype(F32)   # IEEE RNE


# --------------------------------------------------------------------------
# C2. quantise  (the bit-exact contract; every op is one binary32 RNE op)
# --------------------------------------------------------------------------
def global_scale(T: np.ndarray) -> np.float32:
    """g = amax / 2688 in binary32 (step 1; R1, R3)."""
    T = np.asarray(T, dtype=F32)
    amax = F32(np.max(np.abs(T))) if T.size else F32(0.0)
    return F32(amax / GLOBAL_DIV)


def quantize(T: np.ndarray, g=None):
    """T[R,K] (binary32 holding BF16 values) -> (codes[R,K/2], scales[R,K/16], g).

    Steps (every arithmetic op is a single IEEE binary32
    round-to-nearest-even operation, in this order):
      1. amax = max|T| over the whole tensor;  g = amax / 2688   (unless given)
      2. per block of 16 consecutive k:  a_b = max|T_b|;  t = a_b / 6;
         u = t / g;  scale = E4M3_encode(min(u, 448))
      3. d = g * E4M3_decode(scale)
      4. q = T / d;  code = E2M1_encode(q)   (sign of T kept)
      5. pack: byte = code[k even] | code[k odd] << 4
    Special cases: g == 0 -> everything zero;  d == 0 -> that block's codes are
    all 0x0 (sign dropped)  (R5).
    """
    T = np.ascontiguousarray(np.asarray(T, dtype=F32))
    assert T.ndim == 2 and T.shape[1] % BLOCK == 0, "K must be a multiple of 16"
    R, K = T.shape
    nb = K // BLOCK
    g = global_scale(T) if g is None else F32(g)
    codes = np.zeros((R, K // 2), dtype=np.uint8)
    scales = np.zeros((R, nb), dtype=np.uint8)
    if R == 0 or K == 0 or not (g > 0):
        return codes, scales, F32(g)

    Tb = T.reshape(R, nb, BLOCK)
    a_b = np.max(np.abs(Tb), axis=2).astype(F32)                   # exact
    with np.errstate(over="ignore", divide="ignore", invalid="ignore"):
        t = (a_b / F32(6.0)).astype(F32)                           # binary32 div
        u = (t / g).astype(F32)                                    # binary32 div
        scales = e4m3_encode(np.minimum(u, F32(E4M3_MAX)))
        d = (g * e4m3_decode(scales).astype(F32)).astype(F32)      # binary32 mul
        dz = d == 0
        d_safe = np.where(dz, F32(1.0), d)
        q = (Tb / d_safe[:, :, None]).astype(F32)                  # binary32 div
    c = e2m1_encode(q)                                             # [R, nb, 16]
    c = np.where(dz[:, :, None], np.uint8(0), c).reshape(R, K)
    codes = (c[:, 0::2] | (c[:, 1::2] << 4)).astype(np.uint8)
    return codes, scales.astype(np.uint8), F32(g)


def unpack_codes(codes: np.ndarray) -> np.ndarray:
    """codes[R,K/2] -> nibble array [R,K] (low nibble = even k)."""
    codes = np.asarray(codes, dtype=np.uint8)
    R, Kh = codes.shape
    out = np.empty((R, Kh * 2), dtype=np.uint8)
    out[:, 0::2] = codes & 0xF
    out[:, 1::2] = codes >> 4
    return out


# --------------------------------------------------------------------------
# C3. dequantise (exact: a 24-bit x 4-bit x 2-bit significand product)
# --------------------------------------------------------------------------
def dequantize(codes: np.ndarray, scales: np.ndarray, g) -> np.ndarray:
    """-> float64 [R,K], v = float64(g) * E4M3(scale) * E2M1(code)."""
    nib = unpack_codes(codes)
    e = e2m1_decode(nib)                                           # [R,K]
    s = np.repeat(e4m3_decode(scales), BLOCK, axis=1)              # [R,K]
    return np.float64(F32(g)) * s * e


# --------------------------------------------------------------------------
# C4. GEMV: Y[m,n] = sum_k vX[m,k] * vW[n,k] in float64, and A = sum |.|
# --------------------------------------------------------------------------
def gemv_dense(vX: np.ndarray, vW: np.ndarray):
    """float64 definition.  Returns (Y[M,N], A[M,N]) with A = sum_k |vX*vW|."""
    vX = np.asarray(vX, dtype=np.float64)
    vW = np.asarray(vW, dtype=np.float64)
    Y = vX @ vW.T
    A = np.abs(vX) @ np.abs(vW).T
    return Y, A


def gemv_w4a4(w_codes, w_scales, gW, x_codes, x_scales, gX):
    """W4A4: both operands NVFP4 ("W4A4")."""
    return gemv_dense(dequantize(x_codes, x_scales, gX),
                      dequantize(w_codes, w_scales, gW))


def gemv_w4a16(w_codes, w_scales, gW, X_bf16_as_f32):
    """W4A16: NVFP4 weights, BF16 activations used as they are."""
    return gemv_dense(np.asarray(X_bf16_as_f32, dtype=F32).astype(np.float64),
                      dequantize(w_codes, w_scales, gW))


def tolerance(A: np.ndarray) -> np.ndarray:
    """north_star acceptance: |y_gpu - y_ref| <= 1e-3 * sum_k|w_k x_k| + 1e-6."""
    return 1e-3 * np.asarray(A, dtype=np.float64) + 1e-6


# --------------------------------------------------------------------------
# a8. SiLU * mul glue of the decode chain (BASELINE.json configs[4])
# --------------------------------------------------------------------------
def silu_mul(gu_f32: np.ndarray) -> np.ndarray:
    """gu[M, 2I] (BF16 values) -> float64 h[M, I] = silu(gate) * up,
    gate = columns [0, I), up = columns [I, 2I)  (R11)."""
    gu = np.asarray(gu_f32, dtype=F32).astype(np.float64)
    I = gu.shape[1] // 2
    gate, up = gu[:, :I], gu[:, I:]
    return gate / (1.0 + np.exp(-gate)) * up
