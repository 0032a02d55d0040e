"""Pins of the oracle's storage codecs against ml_dtypes / torch (SURVEY 8(c) 'bf16 codec', 'e4m3 codec').
The oracle is then the only thing the CUDA path is compared with."""
import ml_dtypes
import numpy as np
import torch

from oracle import kvr_oracle as orc


def test_bf16_decode_exhaustive():
    codes = np.arange(65536, dtype=np.uint32).astype(np.uint16)
    got = orc.bf16_decode(codes)
    ref = codes.view(ml_dtypes.bfloat16).astype(np.float64)
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan], ref[~nan])
    assert np.array_equal(np.signbit(got[~nan]), np.signbit(ref[~nan]))


def _bf16_ref_single_rounding(x):
    """fp64 -> bf16 with ONE round-to-nearest-even, done in exact rational arithmetic
    (fractions.Fraction), independent of the C code's nearbyint / ldexp route."""
    import math
    from fractions import Fraction
    out = np.empty(x.size, dtype=np.uint16)
    for i, v in enumerate(x.ravel()):
        v = float(v)
        sign = 0x8000 if math.copysign(1.0, v) < 0 else 0
        if v != v:
            out[i] = sign | 0x7FC0
            continue
        a = abs(v)
        if a == 0:
            out[i] = sign
            continue
        if a == math.inf:
            out[i] = sign | 0x7F80
            continue
        e = max(math.frexp(a)[1] - 1, -126)            # weight of the leading bit, clamped at the subnormal binade
        q = Fraction(a) / Fraction(2) ** (e - 7)        # in [128, 256) for normals, [0, 128) for subnormals
        fl = q.numerator // q.denominator
        rem = q - fl
        if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (fl & 1)):
            fl += 1
        if fl == 256:
            fl, e = 128, e + 1
        if e > 127:
            out[i] = sign | 0x7F80
        elif fl < 128:
            out[i] = sign | fl                          # subnormal, biased exponent 0
        else:
            out[i] = sign | ((e + 127) << 7) | (fl - 128)
    return out.reshape(x.shape)


def test_bf16_encode_random_and_ties():
    rng = np.random.default_rng(1)
    x = np.concatenate([
        rng.standard_normal(20000),
        rng.standard_normal(5000) * 1e-3,
        rng.standard_normal(2000) * 1e30,
        rng.standard_normal(2000) * 1e-39,          # bf16 subnormals
        np.array([0.0, -0.0, np.inf, -np.inf, 3.3895313892515355e38, 3.4e38, 1e39, -1e39,
                  2.0 ** -133, 2.0 ** -134, 2.0 ** -134 * 1.0000001, 2.0 ** -126, 2.0 ** -127]),
    ])
    # every tie between neighbouring bf16 numbers in a few binades: (u, u+1) midpoint
    codes = np.arange(0x3F00, 0x4100, dtype=np.uint16)
    lo = codes.view(ml_dtypes.bfloat16).astype(np.float64)
    hi = (codes + 1).astype(np.uint16).view(ml_dtypes.bfloat16).astype(np.float64)
    ties = (lo + hi) / 2
    x = np.concatenate([x, ties, -ties, np.nextafter(ties, np.inf), np.nextafter(ties, -np.inf)])
    got = orc.bf16_encode(x)
    ref = _bf16_ref_single_rounding(x)
    assert np.array_equal(got, ref)
    # ties must go to even: midpoint of codes (u, u+1) -> the even one
    t = orc.bf16_encode(ties)
    assert np.all(t % 2 == 0)
    # ONE rounding: an fp64 just above / below a tie must go up / down (via fp32 it would collapse onto the tie)
    assert np.array_equal(orc.bf16_encode(np.nextafter(ties, np.inf)), codes + 1)
    assert np.array_equal(orc.bf16_encode(np.nextafter(ties, -np.inf)), codes)
    # where fp64->fp32->bf16 double rounding is harmless (all fp32-representable inputs) agree with torch
    xf = x[np.isfinite(x)].astype(np.float32)
    tor = torch.from_numpy(xf).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(orc.bf16_encode(xf.astype(np.float64)), tor)
    mld = xf.astype(ml_dtypes.bfloat16).view(np.uint16)
    assert np.array_equal(tor, mld)


def test_bf16_roundtrip_all_codes():
    codes = np.arange(65536, dtype=np.uint32).astype(np.uint16)
    v = orc.bf16_decode(codes)
    back = orc.bf16_encode(v)
    nan = np.isnan(v)
    assert np.array_equal(back[~nan], codes[~nan])


def test_e4m3_decode_exhaustive():
    codes = np.arange(256, dtype=np.uint16).astype(np.uint8)
    got = orc.e4m3_decode(codes)
    ref = codes.view(ml_dtypes.float8_e4m3fn).astype(np.float64)
    nan = np.isnan(ref)
    assert nan.sum() == 2 and np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan], ref[~nan])
    assert np.array_equal(np.signbit(got[~nan]), np.signbit(ref[~nan]))
    assert got[0x7E] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6


def test_e4m3_encode_vs_ml_dtypes_in_range():
    rng = np.random.default_rng(2)
    x = np.concatenate([rng.standard_normal(20000) * 3, rng.uniform(-448, 448, 20000),
                        rng.standard_normal(5000) * 0.01, rng.standard_normal(2000) * 1e-3])
    # every tie between neighbouring finite codes
    codes = np.arange(0, 0x7E, dtype=np.uint8)
    lo = codes.view(ml_dtypes.float8_e4m3fn).astype(np.float64)
    hi = (codes + 1).astype(np.uint8).view(ml_dtypes.float8_e4m3fn).astype(np.float64)
    ties = (lo + hi) / 2
    x = np.concatenate([x, ties, -ties, np.nextafter(ties, np.inf), np.nextafter(ties, -np.inf), lo, hi])
    x = x[np.abs(x) <= 448]
    got = orc.e4m3_encode_sat(x)
    # ml_dtypes rounds from fp32/fp64 directly with RNE; make inputs fp32-exact to avoid double rounding
    xf = x.astype(np.float32)
    got = orc.e4m3_encode_sat(xf.astype(np.float64))
    ref = xf.astype(ml_dtypes.float8_e4m3fn).view(np.uint8)
    same = got == ref
    zero = (got & 0x7F) == 0
    assert np.all(same | (zero & ((ref & 0x7F) == 0)))
    assert np.array_equal(got[~zero], ref[~zero])
    # the two ties the survey names: 1.0625 -> 1.0 (even), 1.1875 -> 1.25 (even)
    assert orc.e4m3_decode(orc.e4m3_encode_sat(np.array([1.0625, 1.1875]))).tolist() == [1.0, 1.25]
    assert np.all(orc.e4m3_encode_sat(ties) % 2 == 0)


def test_e4m3_saturation_by_hand():
    # libraries give NaN above 464; cvt.rn.satfinite and the oracle clamp (reading R7)
    x = np.array([448.0, 449.0, 464.0, 465.0, 1e6, np.inf, -449.0, -1e30, -np.inf, 447.9, 432.0, 431.9])
    got = orc.e4m3_encode_sat(x)
    assert got[:6].tolist() == [0x7E] * 6
    assert got[6:9].tolist() == [0xFE] * 3
    assert got[9] == 0x7E                       # 447.9 -> nearest is 448
    assert got[10] == 0x7E                      # 432 is the tie between 416 (0x7D, odd) and 448 (0x7E, even)
    assert got[11] == 0x7D
    assert orc.e4m3_encode_sat(np.array([np.nan]))[0] & 0x7F == 0x7F


def test_e4m3_roundtrip_all_codes():
    codes = np.arange(256, dtype=np.uint16).astype(np.uint8)
    v = orc.e4m3_decode(codes)
    back = orc.e4m3_encode_sat(v)
    nan = np.isnan(v)
    assert np.array_equal(back[~nan], codes[~nan])
