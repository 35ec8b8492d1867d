"""oracle/kv_fp8.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The quantiser of the fp8 KV arm (sec. 4.1: "Orthogonal to KV
compression, which shrinks each token and slows the ramp: we bound which tokens stay resident, and the two
compose").  The paper names no format; reading R18 fixes the one stated here, plainly:

  * a K (or V) row of one token and one KV head, x[0..D), is stored as D codes in the 8-bit float format
    E4M3 ("e4m3fn": 1 sign, 4 exponent bits with bias 7, 3 mantissa bits, no infinities, the two codes
    S.1111.111 are NaN, largest finite value 448) and ONE float32 scale:
        amax  = max_d |x[d]|                                   (exact: x is bf16)
        scale = amax / 448   in float32                        (1.0 if amax == 0)
        y[d]  = x[d] / scale in float32 (IEEE division)
        code[d] = y[d] rounded to the nearest E4M3 value, ties to even   (|y| <= 448 up to rounding: it saturates at 448)
  * it decodes to  xhat[d] = value(code[d]) * scale  in float32 (one rounding).
Attention is then the bounded-window attention of attention_ref.c over the xhat rows (q stays bf16).

Everything is float32 numpy, element by element as written above, so that the product's codes and decoded rows can
be compared BIT FOR BIT (both sides take the rounding decision in float32).  Pins: tests/test_oracle_kv_fp8.py
(the 256-entry code table against the format's closed form, rounding against torch's float8_e4m3fn conversion and
against brute force over all codes, round-trip error bounds, exactly representable rows).
"""
from __future__ import annotations

import numpy as np

E4M3_MAX = np.float32(448.0)


def decode_table() -> np.ndarray:
    """value(code) for all 256 codes (NaN for the two NaN codes), from the format's definition."""
    out = np.empty(256, np.float32)
    for c in range(256):
        sign = -1.0 if c & 0x80 else 1.0
        e, m = (c >> 3) & 0xF, c & 0x7
        if e == 0xF and m == 0x7:
            out[c] = np.nan
        elif e == 0:
            out[c] = sign * (m / 8.0) * 2.0 ** -6               # subnormal
        else:
            out[c] = sign * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return out


_TABLE = decode_table()


def encode(y: np.ndarray) -> np.ndarray:
    """float32 -> E4M3 codes, round to nearest, ties to even, saturating at +-448."""
    y = np.asarray(y, np.float32)
    a = np.minimum(np.abs(y), E4M3_MAX).astype(np.float32)
    # the spacing of E4M3 values around a: 2^(floor(log2 a) - 3), never below the subnormal spacing 2^-9
    with np.errstate(divide="ignore"):
        e = np.floor(np.log2(np.maximum(a, np.float32(2.0 ** -20)))).astype(np.int32)
    e = np.clip(e, -6, 8)
    step = np.ldexp(np.float32(1.0), e - 3).astype(np.float32)
    n = np.rint(a / step).astype(np.int64)                  # rint: ties to even; a / step is exact (power of two)
    mag = (n.astype(np.float32) * step).astype(np.float32)  # may have carried into the next binade: still an E4M3 value
    mag = np.minimum(mag, E4M3_MAX)
    # magnitude -> code (exponent / mantissa fields)
    with np.errstate(divide="ignore"):
        e2 = np.floor(np.log2(np.maximum(mag, np.float32(2.0 ** -20)))).astype(np.int32)
    normal = mag >= np.float32(2.0 ** -6)
    e2 = np.where(normal, e2, -6)
    mant = np.where(normal, np.rint(mag / np.ldexp(np.float32(1.0), e2 - 3)).astype(np.int64) - 8,
                    np.rint(mag / np.float32(2.0 ** -9)).astype(np.int64))
    code = np.where(normal, ((e2 + 7) << 3) | mant, mant).astype(np.uint8)
    return (code | np.where(np.signbit(y), 0x80, 0).astype(np.uint8)).astype(np.uint8)


def decode(code: np.ndarray) -> np.ndarray:
    return _TABLE[np.asarray(code, np.uint8)]


def bf16_to_f32(u16: np.ndarray) -> np.ndarray:
    return (np.asarray(u16, np.uint16).astype(np.uint32) << 16).view(np.float32)


def quantize_rows(x_u16: np.ndarray):
    """x [n, H, D] bf16 bits -> (codes uint8 [n, H, D], scales float32 [n, H]), one scale per (token, head) row."""
    x = bf16_to_f32(x_u16)
    amax = np.abs(x).max(axis=-1).astype(np.float32)
    scale = np.where(amax > 0, amax / E4M3_MAX, np.float32(1.0)).astype(np.float32)
    y = (x / scale[..., None]).astype(np.float32)
    return encode(y), scale


def dequantize(codes: np.ndarray, scales: np.ndarray) -> np.ndarray:
    return (decode(codes) * np.asarray(scales, np.float32)[..., None]).astype(np.float32)


def roundtrip(x_u16: np.ndarray) -> np.ndarray:
    """What a stored row decodes to: float32 [n, H, D]."""
    return dequantize(*quantize_rows(x_u16))
