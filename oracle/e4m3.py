"""O1 — E4M3 ("E4M3FN") codec of the oracle (test infrastructure; see oracle/__init__.py).

Format ("E4M3 (4-bit exponent, 3-bit mantissa)", "E4M3FN format—1 sign
bit, 4-bit exponent, and 3-bit mantissa"; the OCP FP8 definition the paper cites as [30],
reading Q8 in DESIGN.md):

    code = s eeee mmm        bias 7
    eeee == 0      : subnormal, value = (-1)^s * (mmm / 8) * 2^-6      (min 2^-9)
    eeee in 1..15  : normal,    value = (-1)^s * (1 + mmm / 8) * 2^(eeee - 7)
    0x7F / 0xFF    : NaN (the only non-finite codes; there are no infinities)
    largest finite : 0x7E = 1.75 * 2^8 = 448

The decoder builds its 256-entry table from the bit fields ("dequantization via
integer bit manipulations").  The encoder is round-to-nearest-even on that grid (subnormals
included), saturating to +-448, preserving the sign of zero, never emitting NaN for finite input.
Neither uses a library fp8 type; `tests/test_oracle_e4m3.py` pins both against brute force and
against torch's independent float8_e4m3fn conversion.
"""

import numpy as np

E4M3_MAX = 448.0


def _build_decode_table():
    table = np.zeros(256, dtype=np.float64)
    for code in range(256):
        s = (code >> 7) & 1
        e = (code >> 3) & 0xF
        m = code & 0x7
        if e == 0xF and m == 0x7:
            v = float("nan")
        elif e == 0:
            v = (m / 8.0) * 2.0 ** -6
        else:
            v = (1.0 + m / 8.0) * 2.0 ** (e - 7)
        table[code] = -v if s else v
    return table


_DECODE = _build_decode_table()


def e4m3_decode(codes):
    """uint8 codes -> float64 values (exact)."""
    codes = np.asarray(codes, dtype=np.uint8)
    return _DECODE[codes]


def e4m3_encode_rne(values):
    """float (32 or 64) values -> uint8 codes: round-to-nearest-even on the e4m3 grid, saturating.

    Steps for a = |v| (all exact in float64 because v has at most 53 significant bits and every
    scaling is by a power of two):
      1. saturate: a = min(a, 448)
      2. e = floor(log2 a), clamped below at -6 (the subnormal binade shares the normal quantum
         of exponent -6)
      3. quantum q = 2^(e-3); n = rint(a / q)   (numpy rint is round-half-to-even)
      4. n == 16 carries into the next binade (e += 1, n = 8)
      5. n < 8 (only possible when e == -6) is a subnormal: code = n
         else code = (e + 7) << 3 | (n - 8)
    NaN input gives 0x7F (never produced for finite input).
    """
    v = np.asarray(values, dtype=np.float64)
    sign = np.signbit(v)
    a = np.minimum(np.abs(v), E4M3_MAX)
    nan = np.isnan(v)
    a = np.where(nan, 0.0, a)
    # floor(log2(a)) via frexp: a = m * 2^ex with m in [0.5, 1)  ->  e = ex - 1
    _, ex = np.frexp(a)
    e = np.maximum(ex.astype(np.int64) - 1, -6)
    e = np.where(a == 0.0, -6, e)
    q = np.ldexp(1.0, (e - 3).astype(np.int32))
    n = np.rint(a / q).astype(np.int64)
    carry = n == 16
    e = np.where(carry, e + 1, e)
    n = np.where(carry, 8, n)
    sub = n < 8
    code = np.where(sub, n, ((e + 7) << 3) | (n - 8))
    code = np.where(sign, code | 0x80, code)
    code = np.where(nan, 0x7F, code)
    return code.astype(np.uint8)
