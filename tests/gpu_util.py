"""Helpers shared by the GPU parity tests (reading the per-row expert outputs Y through the C ABI)."""

import numpy as np


def read_y_rows(layer, cfg, row0, nrows):
    """Rows [row0, row0 + nrows) of the per-row expert outputs as float64.  The library stores them as
    block-scaled fp16 (include/slp_moe.h, SLP_BUF_Y / SLP_BUF_YS): value = y16 * ys[row, column // 128]."""
    y16 = layer.debug_rows("y", np.float16, row0, nrows, cfg.H).astype(np.float64)
    stride = (cfg.H // 128 + 3) // 4 * 4
    ys = layer.debug_rows("ys", np.float32, row0, nrows, stride)[:, :cfg.H // 128].astype(np.float64)
    assert (np.frexp(ys[ys != 0])[0] == 0.5).all(), "block scales must be powers of two"
    return (y16.reshape(nrows, cfg.H // 128, 128) * ys[:, :, None]).reshape(nrows, cfg.H)


def y_tolerance(y_own, rms):
    """Allowed |Y_gpu - Y_f64| per element, Y_f64 = float64 product of the GPU's own codes: fp32 accumulation
    noise (2e-5 of the RMS) plus the fp16 rounding of the block-scaled value.  The block's amax is scaled
    into [2^14, 2^15), so elements within 2^-28 of it are fp16 normals: half an ulp is 2^-11 of the value."""
    blocks = np.abs(y_own).reshape(y_own.shape[0], -1, 128)
    floor = blocks.max(axis=2, keepdims=True) * 2.0 ** -39            # fp16 subnormal step below 2^-28 of amax
    return 2e-5 * rms + 1e-30 + (np.abs(blocks) * 2.0 ** -11 * 1.001 + floor).reshape(y_own.shape)
