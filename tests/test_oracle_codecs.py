"""Pins for the oracle's codecs: closed-form tables, independent
library casts, tie rules.  CPU only."""
import numpy as np
import pytest

from oracle import nvfp4_oracle as O


def test_e2m1_table_values():
    # PAPER.md:346-348 names the element type FP4 (E2M1); its 16 values, written out
    assert list(O.E2M1_TABLE[:8]) == [0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0]
    assert list(O.E2M1_TABLE[8:]) == [-0.0, -0.5, -1.0, -1.5, -2.0, -3.0, -4.0, -6.0]
    assert np.signbit(O.E2M1_TABLE[8])          # 0x8 is -0


def test_e4m3_table_landmarks():
    T = O.E4M3_TABLE
    assert T[0x00] == 0.0 and T[0x01] == 2.0 ** -9 and T[0x07] == 7 * 2.0 ** -9
    assert T[0x08] == 2.0 ** -6 and T[0x38] == 1.0 and T[0x40] == 2.0
    assert T[0x7E] == 448.0 and np.isnan(T[0x7F]) and np.isnan(T[0xFF])
    assert T[0x76] == 224.0 and T[0x77] == 240.0 and T[0x78] == 256.0 and T[0x67] == 60.0 and T[0x68] == 64.0
    assert np.all(np.diff(O.E4M3_POS) > 0)      # strictly increasing 0x00..0x7E
    assert np.all(T[0x80:0xFF] == -T[0x00:0x7F])


def test_tables_against_ml_dtypes():
    ml = pytest.importorskip("ml_dtypes")
    fp8 = np.arange(256, dtype=np.uint8).view(ml.float8_e4m3fn).astype(np.float64)
    ok = ~np.isnan(O.E4M3_TABLE)
    assert np.array_equal(fp8[ok], O.E4M3_TABLE[ok]) and np.all(np.isnan(fp8[~ok]))
    # float4_e2m1fn is stored one value per byte (low nibble)
    fp4 = np.arange(16, dtype=np.uint8).view(ml.float4_e2m1fn).astype(np.float64)
    assert np.array_equal(fp4, O.E2M1_TABLE)
    assert np.array_equal(np.signbit(fp4), np.signbit(O.E2M1_TABLE))


def test_e4m3_table_against_torch():
    torch = pytest.importorskip("torch")
    t = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    ok = ~np.isnan(O.E4M3_TABLE)
    assert np.array_equal(t[ok], O.E4M3_TABLE[ok])


def test_e2m1_tie_rules():
    # the seven midpoints: ties go to the even code
    mids = np.array([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0], dtype=np.float32)
    want = np.array([0, 2, 2, 4, 4, 6, 6], dtype=np.uint8)         # 0, 1.0, 1.0, 2.0, 2.0, 4.0, 4.0
    assert np.array_equal(O.e2m1_encode(mids), want)
    assert np.array_equal(O.e2m1_encode(-mids), want | 8)
    # just off the midpoints
    up = np.nextafter(mids, np.float32(np.inf))
    dn = np.nextafter(mids, np.float32(0))
    assert np.array_equal(O.e2m1_encode(up), np.array([1, 2, 3, 4, 5, 6, 7], dtype=np.uint8))
    assert np.array_equal(O.e2m1_encode(dn), np.array([0, 1, 2, 3, 4, 5, 6], dtype=np.uint8))
    # saturation and signed zero
    assert list(O.e2m1_encode(np.array([6, 6.5, 100, np.inf, -7, -np.inf], dtype=np.float32))) == [7, 7, 7, 7, 15, 15]
    assert list(O.e2m1_encode(np.array([0.0, -0.0, -0.1, 0.1], dtype=np.float32))) == [0, 8, 8, 0]


def test_e4m3_tie_rules():
    enc = lambda *v: list(O.e4m3_encode(np.array(v, dtype=np.float32)))
    assert enc(232.0) == [0x76]                 # midpoint of 224/240 -> even mantissa 224
    assert enc(248.0) == [0x78]                 # midpoint of 240/256 -> 256
    assert enc(449.0, 464.0, 1e9, np.inf) == [0x7E] * 4   # clamp to 448
    assert enc(1.5 * 2.0 ** -9) == [0x02]       # subnormal tie -> even
    assert enc(2.0 ** -10) == [0x00]            # tie between 0 and 2^-9 -> 0
    assert enc(float(np.nextafter(np.float32(2.0 ** -10), np.float32(1)))) == [0x01]
    assert enc(0.0, 2.0 ** -9, 2.0 ** -6, 1.0, 448.0) == [0x00, 0x01, 0x08, 0x38, 0x7E]
    assert enc(61.999996, 62.0) == [0x67, 0x68]  # below / at the 60|64 midpoint


def test_codecs_roundtrip_all_codes():
    assert np.array_equal(O.e2m1_encode(O.E2M1_TABLE.astype(np.float32)), np.arange(16, dtype=np.uint8))
    assert np.array_equal(O.e4m3_encode(O.E4M3_POS.astype(np.float32)), np.arange(0x7F, dtype=np.uint8))


def test_encoders_against_ml_dtypes_casts_random():
    """Independent cast routines (ml_dtypes) agree with the nearest-of-table encoders on
    dense random and on every binary32 value near every rounding boundary."""
    ml = pytest.importorskip("ml_dtypes")
    rng = np.random.default_rng(1)
    q = np.concatenate([
        rng.uniform(-7, 7, 200000).astype(np.float32),
        (rng.standard_normal(200000) * 2).astype(np.float32),
        np.array([0.25, 0.75, 1.25, 1.75, 2.5, 3.5, 5.0, 6.0, 0.0, -0.0], dtype=np.float32),
    ])
    lib = q.astype(ml.float4_e2m1fn).view(np.uint8) & 0xF
    assert np.array_equal(lib, O.e2m1_encode(q))
    u = np.concatenate([
        rng.uniform(0, 448, 200000).astype(np.float32),
        np.exp(rng.uniform(np.log(2.0 ** -12), np.log(448.0), 200000)).astype(np.float32),
        # midpoints between all adjacent representable values, and their float32 neighbours
        ((O.E4M3_POS[1:] + O.E4M3_POS[:-1]) / 2).astype(np.float32),
        np.nextafter(((O.E4M3_POS[1:] + O.E4M3_POS[:-1]) / 2).astype(np.float32), np.float32(0)),
        np.nextafter(((O.E4M3_POS[1:] + O.E4M3_POS[:-1]) / 2).astype(np.float32), np.float32(1e9)),
    ])
    u = np.minimum(u, np.float32(448.0))       # library cast overflows to NaN above 464
    lib8 = u.astype(ml.float8_e4m3fn).view(np.uint8)
    assert np.array_equal(lib8, O.e4m3_encode(u))


def test_bf16_helpers():
    ml = pytest.importorskip("ml_dtypes")
    rng = np.random.default_rng(2)
    x = np.concatenate([(rng.standard_normal(100000) * 3).astype(np.float32),
                        np.array([1.00390625, 1.01171875, 0.0, -0.0, 3.3895314e38], dtype=np.float32)])
    bits = O.f32_to_bf16_bits(x)
    assert np.array_equal(bits, x.astype(ml.bfloat16).view(np.uint16))
    assert np.array_equal(O.bf16_bits_to_f32(bits), x.astype(ml.bfloat16).astype(np.float32))
    y = rng.standard_normal(100000) * 100
    # float64 -> BF16 in ONE rounding: nearest BF16 neighbour of every y (brute force over the two candidates
    # around the truncated bit pattern), ties cannot occur for these random doubles
    r = O.round_to_bf16(y).astype(np.float64)
    lo = (y.astype(np.float32).view(np.uint32) & np.uint32(0xFFFF0000)).view(np.float32).astype(np.float64)
    cand = np.stack([lo, (lo.astype(np.float32).view(np.uint32) + np.uint32(0x10000)).view(np.float32).astype(np.float64),
                     (lo.astype(np.float32).view(np.uint32) - np.uint32(0x10000)).view(np.float32).astype(np.float64)])
    best = cand[np.argmin(np.abs(cand - y), axis=0), np.arange(y.size)]
    assert np.array_equal(r, best)
    assert np.all(np.abs(r - y) <= np.abs(y) * 2.0 ** -8)        # half an ulp of an 8-bit significand
    # exact ties go to even
    assert O.round_to_bf16(np.array([1.00390625]))[0] == np.float32(1.0)       # 1 + 2^-8 -> 1
    assert O.round_to_bf16(np.array([1.01171875]))[0] == np.float32(1.015625)  # 1 + 3*2^-8 -> 1 + 2^-6
