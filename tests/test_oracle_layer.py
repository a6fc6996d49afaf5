"""Pins for the oracle's expert FFN (O5), shared expert (O6), combine (O7) and whole layer.

- brute force: pure-Python loops over a tiny layer, fp8 encode/decode through torch's
  float8_e4m3fn (independent of oracle/e4m3.py);
- dense reduction: E = 1, k = 1 equals routed_scale * a separately written dense SwiGLU;
- near-lossless special case: equals a textbook unquantised SwiGLU FFN to 1e-6;
- error bound against the unquantised FFN (catches dropped terms / transposes / signs);
- invariants: identical experts, linearity in w, permutation equivariance, chunking, poisoning;
- byte accounting against the numbers the paper prints (tests/golden/paper_constants.txt).
"""

import math
import os

import numpy as np
import torch

from oracle import (moe_layer, expert_ffn, quantize_rows_1x128, dequantize_weight_128x128,
                    bf16_bits_to_f64, f64_to_bf16_bits, router)
from paper_2606_10493_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def tiny_cfg(**kw):
    base = dict(name="tiny", T=6, H=128, E=4, k=2, G=1, Gk=1, I=128, n_shared=1,
                scoring="sigmoid_bias", norm_topk=True, routed_scale=2.5, seed=7,
                bias="normal", mode="resident")
    base.update(kw)
    return inputs.LayerConfig(**base)


def run_oracle(cfg, hidden_bits, W, tokens=None):
    return moe_layer(hidden_bits, W, top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk,
                     scoring=cfg.scoring, norm_topk=cfg.norm_topk,
                     routed_scale=cfg.routed_scale, tokens=tokens)


def make(cfg):
    W = inputs.weights_as_numpy(inputs.make_weights(cfg))
    hb = inputs.hidden_as_bits(inputs.make_hidden(cfg))
    return hb, W


# ---------------------------------------------------------------------------------------------
# independent restatement helpers (torch float8 as the codec)
# ---------------------------------------------------------------------------------------------
def t_decode(q):
    return torch.from_numpy(np.ascontiguousarray(q)).view(torch.float8_e4m3fn).double().numpy()


def t_quant_row(v32):
    """v32: 1-D float32 of length 128 -> (dequantised float64 values, scale)."""
    amax = np.float32(np.max(np.abs(v32)))
    s = np.float32(1.0) if amax == 0 else np.float32(amax / np.float32(448.0))
    r = np.clip((v32 / s).astype(np.float32), -448, 448)
    q = torch.from_numpy(r).to(torch.float8_e4m3fn).double().numpy()
    return q * float(s)


def loop_ffn(x32, gq, gs, uq, us, dq, ds):
    """Scalar-loop FFN of one token. x32: float32 [H]."""
    H, I = len(x32), gq.shape[0]
    xh = np.concatenate([t_quant_row(x32[b:b + 128]) for b in range(0, H, 128)])
    gd, ud, dd = t_decode(gq), t_decode(uq), t_decode(dq)
    a = np.zeros(I)
    for i in range(I):
        g = u = 0.0
        for h in range(H):
            g += xh[h] * gd[i, h] * float(gs[i // 128, h // 128])
            u += xh[h] * ud[i, h] * float(us[i // 128, h // 128])
        a[i] = g / (1.0 + math.exp(-g)) * u
    ah = np.concatenate([t_quant_row(a[b:b + 128].astype(np.float32)) for b in range(0, I, 128)])
    y = np.zeros(H)
    for h in range(H):
        acc = 0.0
        for i in range(I):
            acc += ah[i] * dd[h, i] * float(ds[h // 128, i // 128])
        y[h] = acc
    return y


def test_layer_vs_pure_python_brute_force():
    cfg = tiny_cfg()
    hb, W = make(cfg)
    res = run_oracle(cfg, hb, W)
    x32 = (hb.astype(np.uint32) << 16).view(np.float32)
    for t in range(cfg.T):
        exp = np.zeros(cfg.H)
        for j in range(cfg.k):
            e = int(res["route"]["idx"][t, j])
            exp += res["route"]["w"][t, j] * loop_ffn(
                x32[t], W["gate_q"][e], W["gate_s"][e], W["up_q"][e], W["up_s"][e],
                W["down_q"][e], W["down_s"][e])
        exp += loop_ffn(x32[t], W["shared_gate_q"], W["shared_gate_s"], W["shared_up_q"],
                        W["shared_up_s"], W["shared_down_q"], W["shared_down_s"])
        assert np.allclose(res["out_f64"][t], exp, rtol=1e-9, atol=1e-12)


def dense_swiglu_matvec(x_hat, Wg, Wu, Wd, requant):
    g = Wg @ x_hat
    u = Wu @ x_hat
    a = g / (1.0 + np.exp(-g)) * u
    if requant:
        a = np.concatenate([t_quant_row(a[b:b + 128].astype(np.float32)) for b in range(0, len(a), 128)])
    return Wd @ a


def test_dense_reduction_single_expert_top1():
    """E = 1, k = 1, no shared: out = routed_scale * FFN(x) with FFN a plain dense SwiGLU."""
    cfg = tiny_cfg(E=1, k=1, n_shared=0, T=9, H=256, I=256, routed_scale=2.5)
    hb, W = make(cfg)
    res = run_oracle(cfg, hb, W)
    assert np.allclose(res["route"]["w"], 2.5)
    Wg = dequantize_weight_128x128(W["gate_q"][0], W["gate_s"][0])
    Wu = dequantize_weight_128x128(W["up_q"][0], W["up_s"][0])
    Wd = dequantize_weight_128x128(W["down_q"][0], W["down_s"][0])
    x32 = (hb.astype(np.uint32) << 16).view(np.float32)
    for t in range(cfg.T):
        xh = np.concatenate([t_quant_row(x32[t, b:b + 128]) for b in range(0, cfg.H, 128)])
        ref = 2.5 * dense_swiglu_matvec(xh, Wg, Wu, Wd, requant=True)
        assert np.allclose(res["out_f64"][t], ref, rtol=1e-10, atol=1e-13)


def test_near_lossless_case_equals_textbook_swiglu():
    """x on the e4m3 grid (block amax = 448 * 2^j) and one live intermediate channel per
    128-block: both activation quantisers are exact up to one fp32 rounding of the scale, so the
    quantised FFN equals the unquantised float64 SwiGLU FFN to ~1e-7."""
    rng = np.random.default_rng(5)
    H, I, R = 256, 256, 5
    codes = rng.integers(1, 0x7F, (R, H)).astype(np.uint8) | (rng.integers(0, 2, (R, H)) << 7).astype(np.uint8)
    codes[:, 0] = 0x7E
    codes[:, 128] = 0x7E
    j = rng.integers(-9, -6, (R, 2))
    x = (t_decode(codes).reshape(R, 2, 128) * 2.0 ** j[:, :, None]).reshape(R, H)
    cfg = tiny_cfg(H=H, I=I, E=1, k=1, n_shared=0)
    W = inputs.weights_as_numpy(inputs.make_weights(cfg))
    live = np.zeros(I, bool)
    live[[17, 128 + 90]] = True
    uq = W["up_q"][0].copy()
    uq[~live] = 0                                           # dead channels: u = 0 -> a = 0
    xq, xs = quantize_rows_1x128(x.astype(np.float32))
    y, hq, hs = expert_ffn(xq, xs, W["gate_q"][0], W["gate_s"][0], uq, W["up_s"][0],
                           W["down_q"][0], W["down_s"][0])
    Wg = dequantize_weight_128x128(W["gate_q"][0], W["gate_s"][0])
    Wu = dequantize_weight_128x128(uq, W["up_s"][0])
    Wd = dequantize_weight_128x128(W["down_q"][0], W["down_s"][0])
    for r in range(R):
        ref = dense_swiglu_matvec(x[r], Wg, Wu, Wd, requant=False)
        # fp32 rounding of a and of the scale: ~1e-7 of the largest term (sums may cancel)
        assert np.abs(y[r] - ref).max() <= 3e-7 * np.abs(ref).max()
    assert ((hq & 0x7F) != 0).sum() == R * 2                # exactly the live channels survive


def test_error_bound_vs_unquantised_ffn():
    """Against the FFN with NO activation quantisation the relative L2 error must be of the size
    fp8 activations give (a few %), far below what a wrong sign/transposed operand would give."""
    cfg = tiny_cfg(E=1, k=1, n_shared=0, T=32, H=512, I=256, routed_scale=1.0)
    hb, W = make(cfg)
    res = run_oracle(cfg, hb, W)
    x = bf16_bits_to_f64(hb)
    Wg = dequantize_weight_128x128(W["gate_q"][0], W["gate_s"][0])
    Wu = dequantize_weight_128x128(W["up_q"][0], W["up_s"][0])
    Wd = dequantize_weight_128x128(W["down_q"][0], W["down_s"][0])
    g, u = x @ Wg.T, x @ Wu.T
    ref = (g / (1 + np.exp(-g)) * u) @ Wd.T
    rel = np.linalg.norm(res["out_f64"] - ref) / np.linalg.norm(ref)
    assert 1e-3 < rel < 8e-2, rel


def test_identical_experts_make_routing_irrelevant():
    cfg = tiny_cfg(T=12, E=4, k=2, n_shared=1)
    hb, W = make(cfg)
    for key in ("gate_q", "gate_s", "up_q", "up_s", "down_q", "down_s"):
        W[key] = np.stack([W[key][0]] * cfg.E)
    res = run_oracle(cfg, hb, W)
    x32 = (hb.astype(np.uint32) << 16).view(np.float32)
    xq, xs = quantize_rows_1x128(x32)
    y, _, _ = expert_ffn(xq, xs, W["gate_q"][0], W["gate_s"][0], W["up_q"][0], W["up_s"][0],
                         W["down_q"][0], W["down_s"][0])
    ys, _, _ = expert_ffn(xq, xs, W["shared_gate_q"], W["shared_gate_s"], W["shared_up_q"],
                          W["shared_up_s"], W["shared_down_q"], W["shared_down_s"])
    assert np.allclose(res["out_f64"], cfg.routed_scale * y + ys, rtol=1e-12, atol=1e-14)


def test_linearity_in_routed_scale_and_shared_unscaled():
    cfg1, cfg2 = tiny_cfg(routed_scale=1.0), tiny_cfg(routed_scale=3.0)
    hb, W = make(cfg1)
    a, b = run_oracle(cfg1, hb, W), run_oracle(cfg2, hb, W)
    Wn = dict(W)
    for key in list(Wn):
        if key.startswith("shared_"):
            Wn[key] = None
    a0, b0 = run_oracle(cfg1, hb, Wn), run_oracle(cfg2, hb, Wn)
    assert np.allclose(b0["out_f64"], 3.0 * a0["out_f64"], rtol=1e-12)
    shared = a["out_f64"] - a0["out_f64"]
    assert np.allclose(b["out_f64"] - b0["out_f64"], shared, rtol=1e-9, atol=1e-12)  # Q16


def test_token_permutation_equivariance_and_chunking():
    cfg = tiny_cfg(T=40, E=8, k=3, G=4, Gk=2, H=256)
    hb, W = make(cfg)
    full = run_oracle(cfg, hb, W)
    p = np.random.default_rng(0).permutation(cfg.T)
    shuf = run_oracle(cfg, hb[p], W)
    assert np.allclose(shuf["out_f64"], full["out_f64"][p], rtol=1e-11, atol=1e-14)
    parts = [run_oracle(cfg, hb[i:i + 8], W)["out_f64"] for i in range(0, cfg.T, 8)]     # Q20
    # (BLAS sums in a shape-dependent order, so float64 results agree to rounding, not bitwise)
    assert np.allclose(np.concatenate(parts), full["out_f64"], rtol=1e-11, atol=1e-14)
    sub = run_oracle(cfg, hb, W, tokens=np.array([3, 17, 39]))
    assert np.allclose(sub["out_f64"], full["out_f64"][[3, 17, 39]], rtol=1e-11, atol=1e-14)


def test_poisoned_unused_experts_do_not_matter():
    cfg = tiny_cfg(T=5, E=8, k=2)
    hb, W = make(cfg)
    base = run_oracle(cfg, hb, W)
    unused = [e for e in range(cfg.E) if base["route"]["counts"][e] == 0]
    assert unused, "test needs at least one expert without tokens"
    Wp = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in W.items()}
    for e in unused:
        for key in ("gate_q", "up_q", "down_q"):
            Wp[key][e][:] = 0x7F                                  # NaN bytes
    out = run_oracle(cfg, hb, Wp)["out_f64"]
    assert np.isfinite(out).all() and np.allclose(out, base["out_f64"], rtol=1e-11, atol=1e-14)


def test_bf16_output_rounding():
    x = np.array([1.0, 1.00390625, 1.005859375, -3.1415926, 1e-3, 65280.0, 0.0])
    bits = f64_to_bf16_bits(x)
    ref = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(bits, ref)
    assert np.array_equal(bf16_bits_to_f64(bits), torch.from_numpy(x).to(torch.bfloat16).double().numpy())
    # ties-to-even directly from float64: 1 + 2^-8 is halfway between 1 and 1 + 2^-7
    assert f64_to_bf16_bits(np.array([1.0 + 2.0 ** -8]))[0] == 0x3F80
    assert f64_to_bf16_bits(np.array([1.0 + 3 * 2.0 ** -8]))[0] == 0x3F82


def test_byte_accounting_matches_paper():
    gold = {}
    with open(os.path.join(HERE, "golden", "paper_constants.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, val, tol, _ = [s.strip() for s in line.split("|")]
            gold[name] = (float(val), float(tol))
    v3 = inputs.CONFIGS[1]
    per_layer = v3.E * inputs.routed_bytes_per_expert(v3)
    assert per_layer == 11274289152
    val, tol = gold["routed_fp8_bytes_per_layer_deepseek_v3_GB"]
    assert abs(per_layer / 1e9 - val) <= tol * val + 0.05
    val, tol = gold["routed_fp8_bytes_per_layer_kimi_k2_GB"]
    assert abs(384 * inputs.routed_bytes_per_expert(v3) / 1e9 - val) <= tol * val + 0.05
    val, tol = gold["expert_weight_tensors_deepseek_v3_K"]
    assert abs(58 * v3.E * 3 / 1e3 - val) <= 0.05
    assert inputs.BLOCK == gold["scale_block_k"][0]
    assert v3.k == gold["activated_experts"][0]
    assert inputs.fp8_flops_per_token(v3) == 704643072 + 88080384


def test_input_generator_shapes_and_prefix_property():
    c1, c2 = inputs.CONFIGS[1], inputs.CONFIGS[2]
    small1 = inputs.LayerConfig(**{**c1.__dict__, "H": 256, "T": 4096})
    small2 = inputs.LayerConfig(**{**c2.__dict__, "H": 256, "T": 8192})
    h1, h2 = inputs.make_hidden(small1), inputs.make_hidden(small2)
    assert torch.equal(h1, h2[:4096])
    w, b = inputs.make_router(inputs.CONFIGS[0])
    assert w.shape == (8, 256) and b.shape == (8,)
    assert abs(float(w.std()) - 1 / 16) < 0.01 and abs(float(b.std()) - 0.01) < 0.01
    q, s = inputs.quantize_weight_128x128(torch.randn(256, 128) * 0.02)
    assert q.dtype == torch.uint8 and s.shape == (2, 1)
    assert ((q.view(2, 128, 128) & 0x7F).amax(dim=(1, 2)) == 0x7E).all()


def test_zipf_bias_config_is_skewed():
    """cfg 3 recipe (at reduced T and H so it runs in seconds): several hot experts, many with
    0-3 rows, many exactly empty."""
    c3 = inputs.CONFIGS[3]
    cfg = inputs.LayerConfig(**{**c3.__dict__, "T": 4096, "H": 512})
    w, b = inputs.make_router(cfg)
    hb = inputs.hidden_as_bits(inputs.make_hidden(cfg))
    r = router(hb, w.numpy(), b.numpy(), top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk,
               scoring=cfg.scoring, norm_topk=True, routed_scale=cfg.routed_scale)
    c = r["counts"]
    assert (c > 0.05 * cfg.T).sum() >= 3
    assert (c <= 3).sum() >= 64
    assert (c == 0).sum() >= 32
