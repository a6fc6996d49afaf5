"""Pins for the oracle's E4M3 codec (O1) and 1x128 / 128x128 block formats (O2, O4).

None of these re-type the oracle's formulas: they use values the format fixes, brute-force
nearest-code search on a grid obtained from torch's float8_e4m3fn (an independent library
routine), torch's own conversion, and error bounds.
"""

import numpy as np
import torch

from oracle import (e4m3_decode, e4m3_encode_rne, quantize_rows_1x128, dequantize_rows_1x128,
                    dequantize_weight_128x128)

ALL = np.arange(256, dtype=np.uint8)
FINITE = np.array([c for c in range(256) if (c & 0x7F) != 0x7F], dtype=np.uint8)


def torch_grid():
    return torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).double().numpy()


def test_decode_fixed_points():
    # OCP E4M3: max finite 448 = 0x7E, min subnormal 2^-9 = 0x01, min normal 2^-6 = 0x08
    assert e4m3_decode(np.uint8(0x7E)) == 448.0
    assert e4m3_decode(np.uint8(0xFE)) == -448.0
    assert e4m3_decode(np.uint8(0x01)) == 2.0 ** -9
    assert e4m3_decode(np.uint8(0x08)) == 2.0 ** -6
    assert e4m3_decode(np.uint8(0x38)) == 1.0
    assert e4m3_decode(np.uint8(0x00)) == 0.0 and not np.signbit(e4m3_decode(np.uint8(0x00)))
    assert e4m3_decode(np.uint8(0x80)) == 0.0 and np.signbit(e4m3_decode(np.uint8(0x80)))
    assert np.isnan(e4m3_decode(np.uint8(0x7F))) and np.isnan(e4m3_decode(np.uint8(0xFF)))
    assert np.isfinite(e4m3_decode(FINITE)).all()          # no infinities anywhere


def test_decode_matches_torch_float8():
    ours, ref = e4m3_decode(ALL), torch_grid()
    assert np.array_equal(np.isnan(ours), np.isnan(ref))
    m = ~np.isnan(ref)
    assert np.array_equal(ours[m], ref[m])
    assert np.array_equal(np.signbit(ours[m]), np.signbit(ref[m]))


def test_roundtrip_all_finite_codes():
    assert np.array_equal(e4m3_encode_rne(e4m3_decode(FINITE)), FINITE)


def test_midpoints_round_to_even_and_saturation():
    # grid around 16..20 is 16, 18, 20: 17 -> 16 (even mantissa 0), 19 -> 20 (mantissa 2)
    assert e4m3_decode(e4m3_encode_rne(np.float32(17.0))) == 16.0
    assert e4m3_decode(e4m3_encode_rne(np.float32(19.0))) == 20.0
    # subnormal midpoints: 1.5 * 2^-9 -> 2 * 2^-9 (even), 0.5 * 2^-9 -> 0
    assert e4m3_decode(e4m3_encode_rne(np.float32(1.5 * 2.0 ** -9))) == 2.0 ** -8
    assert e4m3_encode_rne(np.float32(0.5 * 2.0 ** -9)) == 0
    assert e4m3_encode_rne(np.float32(-0.5 * 2.0 ** -9)) == 0x80       # sign of zero kept
    big = np.array([449, 463.9, 464, 480, 1e4, 1e9, 3e38], dtype=np.float32)
    assert (e4m3_encode_rne(big) == 0x7E).all()
    assert (e4m3_encode_rne(-big) == 0xFE).all()
    assert e4m3_encode_rne(np.float32(np.inf)) == 0x7E
    assert e4m3_encode_rne(np.float32(np.nan)) == 0x7F


def test_monotone():
    x = np.sort(np.random.default_rng(0).normal(0, 100, 20000).astype(np.float32))
    d = e4m3_decode(e4m3_encode_rne(x))
    assert (np.diff(d) >= 0).all()


def test_exhaustive_bf16_vs_brute_force_nearest():
    """Every bf16 bit pattern: the encoder must pick the nearest finite code (ties -> even
    mantissa), saturating beyond 448.  Grid values come from torch, search is brute force."""
    grid = torch_grid()
    pos_codes = np.array([c for c in range(0x7F)], dtype=np.int64)           # 0x00..0x7E
    pos_vals = grid[pos_codes]
    bits = np.arange(65536, dtype=np.uint32)
    vals = (bits << 16).astype(np.uint32).view(np.float32).astype(np.float64)
    finite = np.isfinite(vals)
    a = np.abs(vals[finite])
    dist = np.abs(a[:, None] - pos_vals[None, :])                            # [n, 127]
    best = dist.min(axis=1)
    cand = dist == best[:, None]
    # among equidistant candidates prefer the even code (codes are consecutive -> one is even)
    even = (pos_codes % 2 == 0)[None, :]
    pick_even = (cand & even).any(axis=1)
    choice = np.where(pick_even, np.argmax(cand & even, axis=1), np.argmax(cand, axis=1))
    expect = pos_codes[choice]
    expect = np.where(a >= 448.0, 0x7E, expect)
    expect = np.where(np.signbit(vals[finite]), expect | 0x80, expect).astype(np.uint8)
    got = e4m3_encode_rne(vals[finite].astype(np.float32))
    assert np.array_equal(got, expect)


def test_encoder_matches_torch_conversion_in_range():
    rng = np.random.default_rng(1)
    x = np.concatenate([
        rng.normal(0, 1, 200000), rng.normal(0, 150, 200000), rng.normal(0, 1e-2, 200000),
        rng.uniform(-448, 448, 200000), rng.normal(0, 2e-3, 100000)]).astype(np.float32)
    x = np.clip(x, -448, 448)
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(e4m3_encode_rne(x), ref)


def test_row_quantiser_properties():
    rng = np.random.default_rng(2)
    x = rng.normal(0, 1, (37, 512)).astype(np.float32)
    x[3, 128:256] = 0.0                                   # an all-zero block (Q11)
    q, s = quantize_rows_1x128(x)
    qb = q.reshape(37, 4, 128)
    top = (qb & 0x7F).max(axis=2)
    assert top[3, 1] == 0 and s[3, 1] == 1.0
    mask = np.ones((37, 4), bool)
    mask[3, 1] = False
    assert (top[mask] == 0x7E).all()                      # block max always hits +-448
    assert np.allclose(s[mask], np.abs(x.reshape(37, 4, 128)).max(axis=2)[mask] / 448.0, rtol=1e-7)
    xh = dequantize_rows_1x128(q, s)
    # |x - x_hat| <= half a quantum of the element's binade: s * 2^(e-4) with e = floor(log2|x/s|)
    ratio = np.abs(x.reshape(37, 4, 128).astype(np.float64) / s[:, :, None])
    e = np.floor(np.log2(np.maximum(ratio, 2.0 ** -6)))
    bound = (s[:, :, None] * 2.0 ** (e - 4)).reshape(37, 512) * (1 + 1e-6)
    assert (np.abs(x - xh) <= bound).all()


def test_row_quantiser_lossless_on_grid():
    """Inputs on the e4m3 grid times a power-of-two scale, block amax exactly 448 * 2^j."""
    rng = np.random.default_rng(3)
    codes = rng.integers(0, 0x7F, (16, 256)).astype(np.uint8) | (rng.integers(0, 2, (16, 256)) << 7).astype(np.uint8)
    codes[:, 0] = 0x7E
    codes[:, 128] = 0xFE
    j = rng.integers(-6, 6, (16, 2))
    vals = torch.from_numpy(codes).view(torch.float8_e4m3fn).double().numpy().reshape(16, 2, 128)
    x = (vals * 2.0 ** j[:, :, None]).reshape(16, 256).astype(np.float32)
    q, s = quantize_rows_1x128(x)
    assert np.array_equal(s, (2.0 ** j).astype(np.float32))
    assert np.array_equal(dequantize_rows_1x128(q, s), x.astype(np.float64))
    nz = (codes & 0x7F) != 0
    assert np.array_equal(q[nz], codes[nz])


def test_weight_dequant_block_indexing():
    """w[n,k] uses s[n//128, k//128]: distinct scale per block makes a transposed index fail."""
    q = np.full((256, 384), 0x38, dtype=np.uint8)            # all ones
    s = np.arange(1, 7, dtype=np.float32).reshape(2, 3)
    w = dequantize_weight_128x128(q, s)
    for nb in range(2):
        for kb in range(3):
            blk = w[nb * 128:(nb + 1) * 128, kb * 128:(kb + 1) * 128]
            assert (blk == s[nb, kb]).all()
