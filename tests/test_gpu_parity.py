"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs, with the north_star acceptance rule (oracle/acceptance.py).

Sizes: config 0 (tiny), a reduced DeepSeek-V3-like layer that spans several 128-row tiles with a
ragged tail and a shared expert, a reduced softmax layer (config 4's routing), and the skewed
config-3 recipe at reduced size (empty experts, 1-3-row experts).  Full-size sampled checks are in
test_gpu_fullsize.py.
"""

import numpy as np
import pytest
import torch

from oracle import moe_layer, permutation
from oracle.acceptance import compare_routing, compare_output
from paper_2606_10493_b200 import SlpMoeLayer, SlpError, inputs
from gpu_util import read_y_rows, y_tolerance

pytestmark = pytest.mark.gpu


def small_dsv3(**kw):
    base = dict(name="mini_dsv3", T=300, H=512, E=32, k=4, G=4, Gk=2, I=256, n_shared=1,
                scoring="sigmoid_bias", norm_topk=True, routed_scale=2.5, seed=11, bias="normal",
                mode="streamed")
    base.update(kw)
    return inputs.LayerConfig(**base)


CASES = {
    "cfg0": inputs.CONFIGS[0],
    "mini_dsv3": small_dsv3(),
    "mini_dsv3_ragged": small_dsv3(T=1000, seed=12, H=768, I=384),
    "mini_softmax": small_dsv3(name="mini_softmax", T=513, H=256, E=16, k=4, G=1, Gk=1, I=128, n_shared=0,
                               scoring="softmax", routed_scale=1.0, bias="none", seed=13),
    "mini_zipf": small_dsv3(name="mini_zipf", T=2048, H=256, E=64, k=8, G=8, Gk=4, I=128, bias="zipf", seed=14),
}

_cache = {}


def problem(name):
    if name not in _cache:
        cfg = CASES[name]
        W = inputs.make_weights(cfg, device="cpu", pin=True)
        hidden = inputs.make_hidden(cfg, device="cpu")
        ref = moe_layer(inputs.hidden_as_bits(hidden), inputs.weights_as_numpy(W), top_k=cfg.k,
                        n_group=cfg.G, topk_group=cfg.Gk, scoring=cfg.scoring,
                        norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
        _cache[name] = (cfg, W, hidden, ref)
    return _cache[name]


def run_gpu(cfg, W, hidden, mode, **kw):
    layer = SlpMoeLayer(cfg, W, device=0, **kw)
    try:
        layer.set_residency(mode)
        out = layer.prefill(hidden.cuda())
        torch.cuda.synchronize()
        idx, w, counts = layer.debug_routing(hidden.shape[0])
        xq, xs = layer.debug_quant_hidden(hidden.shape[0])
        extra = dict(pos=layer.debug_buffer("pos", np.int32).reshape(hidden.shape[0], cfg.k),
                     row_start=layer.debug_buffer("row_start", np.int32),
                     row_token=layer.debug_buffer("row_token", np.int32),
                     stats=layer.stats())
    finally:
        layer.close()
    return inputs.hidden_as_bits(out), idx, w, counts, xq, xs, extra


def check(name, mode, **kw):
    cfg, W, hidden, ref = problem(name)
    out, idx, w, counts, xq, xs, extra = run_gpu(cfg, W, hidden, mode, **kw)
    r = compare_routing(idx, w, ref["route"])
    o = compare_output(out, ref["out_f64"], r["members_equal"])
    print(name, mode, kw, {k: v for k, v in r.items() if k != "members_equal"}, o, extra["stats"])
    assert r["passed"], r
    assert o["passed"], o
    return r, o


@pytest.mark.parametrize("name", list(CASES))
def test_substeps_bit_exact(name):
    """Router indices (outside near-ties), quantised hidden bytes + scales (bit-exact, Q12) and
    the permutation (true inverse, expert-contiguous, ascending token id, 128-aligned ranges)."""
    cfg, W, hidden, ref = problem(name)
    out, idx, w, counts, xq, xs, extra = run_gpu(cfg, W, hidden, "resident", triage="gemm=simt")
    r = compare_routing(idx, w, ref["route"])
    assert r["passed"], r
    assert np.array_equal(xq, ref["xq"])
    assert np.array_equal(xs, ref["xs"])
    T, k, E = cfg.T, cfg.k, cfg.E
    pos, row_start, row_token = extra["pos"], extra["row_start"], extra["row_token"]
    assert counts.sum() == T * k
    assert np.array_equal(counts, np.bincount(idx.reshape(-1), minlength=E))
    assert (row_start[:E] % 128 == 0).all() and row_start[E] == 0
    assert np.array_equal(row_token[pos], np.repeat(np.arange(T)[:, None], k, axis=1))      # true inverse
    assert len(np.unique(pos)) == T * k
    _, offsets, perm, pos_ref = permutation(idx, E)                                            # O8 on the GPU's idx
    for e in range(E):
        rows = row_token[row_start[e]:row_start[e] + counts[e]]
        assert np.array_equal(rows, perm[offsets[e]:offsets[e + 1]])                           # ascending token id
        pad = row_token[row_start[e] + counts[e]:row_start[e] + (counts[e] + 127) // 128 * 128]
        assert (pad == -1).all()
    ee = idx
    assert np.array_equal(pos - row_start[ee], pos_ref - offsets[ee])


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("mode", ["resident", "streamed"])
def test_layer_parity_simt(name, mode):
    check(name, mode, triage="gemm=simt")


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("mode", ["resident", "streamed"])
def test_layer_parity_tcgen05(name, mode):
    """Default: the product path (tcgen05 / TMEM / TMA, one CTA per 128 x 256 tile, dynamic tile order)."""
    check(name, mode, triage=None)


@pytest.mark.parametrize("name", list(CASES))
def test_layer_parity_tcgen05_cta_pair(name):
    """triage "gemm=pair": the cta_group::2 variant (clusters of two CTAs, pairs of 128-row tiles, dummy
    tile for experts with an odd tile count)."""
    check(name, "resident", triage="gemm=pair")


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("mode", ["resident", "streamed"])
def test_layer_parity_tcgen05_static_tiles(name, mode):
    """triage "gemm=static": the one-CTA kernel with the static round-robin tile order."""
    check(name, mode, triage="gemm=static")


@pytest.mark.parametrize("T", [1, 127, 128, 129, 257])
@pytest.mark.parametrize("triage", [None, "gemm=pair", "gemm=static"])
def test_ragged_token_counts(T, triage):
    """Edge sizes: a single token, one row short of / exactly / one row past a 128-row tile."""
    cfg, W, hidden, _ = problem("mini_dsv3")
    sub = cfg.with_tokens(T)
    x = hidden[:T].contiguous()
    ref = moe_layer(inputs.hidden_as_bits(x), inputs.weights_as_numpy(W), top_k=cfg.k, n_group=cfg.G,
                    topk_group=cfg.Gk, scoring=cfg.scoring, norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
    for mode in ("resident", "streamed"):
        out, idx, w, counts, *_ = run_gpu(sub, W, x, mode, triage=triage)
        r = compare_routing(idx, w, ref["route"])
        o = compare_output(out, ref["out_f64"], r["members_equal"])
        assert r["passed"] and o["passed"], (T, mode, r, o)
        assert counts.sum() == T * cfg.k


@pytest.mark.parametrize("name", ["mini_dsv3_ragged", "mini_zipf", "mini_softmax"])
@pytest.mark.parametrize("triage", [None, "gemm=pair"])
def test_expert_intermediates_against_oracle(name, triage):
    """a5-a7 row by row: the requantised SwiGLU output (hq, hs) and the per-row expert output Y of the
    tcgen05 kernels against the oracle's expert_ffn on the same quantised rows.  The e4m3 codes are an
    integer decision taken in fp32 on both sides (Q12); they may differ only where fp32-vs-fp64
    accumulation noise moves h across a rounding boundary: at most 1e-4 of the codes, each by one
    e4m3 step, and the row scale by the ~1e-6 relative error of its fp32 amax element."""
    from oracle import expert_ffn, dequantize_rows_1x128, dequantize_weight_128x128
    from oracle import e4m3_decode as decode
    cfg, W, hidden, ref = problem(name)
    Wn = inputs.weights_as_numpy(W)
    layer = SlpMoeLayer(cfg, W, device=0, triage=triage)
    try:
        layer.set_residency("resident")
        layer.prefill(hidden.cuda())
        torch.cuda.synchronize()
        idx, w, counts = layer.debug_routing(cfg.T)
        xq, xs = layer.debug_quant_hidden(cfg.T)
        row_start = layer.debug_buffer("row_start", np.int32)
        row_token = layer.debug_buffer("row_token", np.int32)
        hs_stride = (cfg.I // 128 + 3) // 4 * 4
        hq = layer.debug_buffer("hq", np.uint8).reshape(-1, cfg.I)
        hs = layer.debug_buffer("hs", np.float32).reshape(-1, hs_stride)[:, :cfg.I // 128]
        n_rows = hq.shape[0]
        y = read_y_rows(layer, cfg, 0, n_rows)
    finally:
        layer.close()
    assert np.array_equal(xq, ref["xq"]) and np.array_equal(xs, ref["xs"])
    n_codes = n_flip = 0
    experts = [e for e in range(cfg.E) if counts[e] > 0][:6] + ([cfg.E] if cfg.n_shared else [])
    for e in experts:
        if e == cfg.E:
            r0, n, toks = 0, cfg.T, np.arange(cfg.T)
            keys = ("shared_gate_q", "shared_gate_s", "shared_up_q", "shared_up_s", "shared_down_q", "shared_down_s")
            ws = [Wn[k] for k in keys]
        else:
            r0, n = int(row_start[e]), int(counts[e])
            toks = row_token[r0:r0 + n]
            ws = [Wn[k][e] for k in ("gate_q", "gate_s", "up_q", "up_s", "down_q", "down_s")]
        y_ref, hq_ref, hs_ref = expert_ffn(xq[toks], xs[toks], *ws)
        g_hq, g_hs, g_y = hq[r0:r0 + n], hs[r0:r0 + n], y[r0:r0 + n]
        # scales = amax / 448: the amax element carries the fp32 accumulation + ex2/rcp.approx error (~1e-6)
        assert np.allclose(g_hs, hs_ref, rtol=3e-6, atol=0), (e, np.abs(g_hs / hs_ref - 1).max())
        diff = g_hq != hq_ref
        n_codes += diff.size
        n_flip += int(diff.sum())
        if diff.any():   # flipped codes are neighbours on the e4m3 grid
            a, b = decode(g_hq[diff]), decode(hq_ref[diff])
            step = np.maximum(np.abs(a), np.abs(b)) / 8 + 2.0 ** -9
            assert (np.abs(a - b) <= step * 1.0001).all(), e
        # Y rows (a7): the down GEMM on the GPU's OWN codes against the float64 product of the same codes,
        # so a flipped code upstream does not blur the check: only fp32 accumulation noise is left
        y_own = dequantize_rows_1x128(g_hq, g_hs) @ dequantize_weight_128x128(ws[4], ws[5]).T
        rms = np.sqrt((y_own ** 2).mean())
        assert (np.abs(g_y - y_own) <= y_tolerance(y_own, rms)).all(), (e, np.abs(g_y - y_own).max() / rms)
    print(name, triage, "codes", n_codes, "differ", n_flip)
    assert n_flip <= 1e-4 * n_codes   # observed: 4 of 718 848 (accumulation-order noise, SURVEY.md Q21 predicts ~2e-5)


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("triage", [None, "router=fp32"])
def test_router_logits_error(name, triage):
    """Router logits (SLP_BUF_LOGITS) against the fp64 product.  The tensor-core router splits the
    fp32 weights into bf16 hi + lo (kernels_router_tc.cuh); its logit error must stay a decade
    below the 1e-4 near-tie allowance on the selection scores (|d sigmoid| <= |d logit| / 4)."""
    cfg, W, hidden, ref = problem(name)
    layer = SlpMoeLayer(cfg, W, device=0, triage=triage)
    try:
        layer.set_residency("resident")
        layer.prefill(hidden.cuda())
        torch.cuda.synchronize()
        logits = layer.debug_buffer("logits", np.float32).reshape(cfg.T, cfg.E)
        idx, w, _ = layer.debug_routing(cfg.T)
    finally:
        layer.close()
    x = hidden.to(torch.float64).numpy()
    exact = x @ W["router_w"].to(torch.float64).numpy().T
    err = np.abs(logits - exact).max()
    print(name, "triage", triage, "max |logit error|", err)
    assert err < 4e-5, err
    r = compare_routing(idx, w, ref["route"])
    assert r["passed"], r


@pytest.mark.parametrize("kw", [dict(staging_slots=2, experts_per_launch=1),
                                dict(staging_slots=8, experts_per_launch=4),
                                dict(staging_slots=4, experts_per_launch=2, skip_empty_experts=True),
                                dict(skip_empty_experts=True)])
def test_streaming_ring_variants(kw):
    """Ring length 2 (the paper's ping-pong), partial rings, empty-expert skipping."""
    check("mini_zipf", "streamed", **kw)
    check("mini_dsv3_ragged", "streamed", **kw)


def test_run_to_run_bitwise_and_chunking():
    """Bitwise determinism, and Q20: chunked prefill == single pass, bit for bit."""
    cfg, W, hidden, ref = problem("mini_dsv3_ragged")
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        x = hidden.cuda()
        for mode in ("resident", "streamed"):
            layer.set_residency(mode)
            a = layer.prefill(x).clone()
            b = layer.prefill(x).clone()
            torch.cuda.synchronize()
            assert torch.equal(a.view(torch.int16), b.view(torch.int16))
            parts = []
            for r0 in range(0, cfg.T, 256):
                parts.append(layer.prefill(x[r0:r0 + 256].contiguous()).clone())
            torch.cuda.synchronize()
            assert torch.equal(torch.cat(parts).view(torch.int16), a.view(torch.int16))
    finally:
        layer.close()


def test_poisoned_unused_experts():
    """NaN bytes in the weights of experts that receive no token must not reach the output."""
    cfg, W, hidden, ref = problem("mini_zipf")
    unused = np.nonzero(ref["route"]["counts"] == 0)[0]
    assert len(unused) > 0
    Wp = {k: (v.clone().pin_memory() if isinstance(v, torch.Tensor) else v) for k, v in W.items()}
    for e in unused:
        for key in ("gate_q", "up_q", "down_q"):
            Wp[key][e].fill_(0x7F)
    for mode in ("resident", "streamed"):
        out, idx, w, *_ = run_gpu(cfg, Wp, hidden, mode)
        r = compare_routing(idx, w, ref["route"])
        o = compare_output(out, ref["out_f64"], r["members_equal"])
        assert o["finite"] and o["passed"], o


def test_host_entry_point_and_stats():
    cfg, W, hidden, ref = problem("mini_dsv3")
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        hin = hidden.pin_memory()
        hout = torch.empty_like(hin).pin_memory()
        layer.prefill_host(hin, hout)
        st = layer.stats()
        idx, w, _ = layer.debug_routing(cfg.T)
    finally:
        layer.close()
    r = compare_routing(idx, w, ref["route"])
    o = compare_output(inputs.hidden_as_bits(hout), ref["out_f64"], r["members_equal"])
    assert o["passed"], o
    assert st["experts_copied"] == cfg.E and st["bytes_copied"] == cfg.E * 3 * cfg.I * cfg.H
    assert st["gemm_launches"] > 0 and st["kernel_launches"] > st["gemm_launches"]


def test_error_paths():
    cfg, W, hidden, _ = problem("cfg0")
    bad = inputs.LayerConfig(**{**cfg.__dict__, "H": 200})
    with pytest.raises(SlpError) as ei:
        SlpMoeLayer(bad, W, device=0)
    assert ei.value.status == -2
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        x = hidden.cuda()
        with pytest.raises(SlpError):
            layer.prefill(torch.cat([x, x]))                      # T > max_tokens
        out = torch.full_like(x, 7.0)
        layer.prefill(x[:0], out[:0])                              # T == 0 touches nothing
        torch.cuda.synchronize()
        assert (out == 7.0).all()
    finally:
        layer.close()
