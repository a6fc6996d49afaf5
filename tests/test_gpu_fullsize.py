"""Full-size parity: the BASELINE configs in the launch configurations bench.py times.

  cfg 1 (T = 4096, DeepSeek-V3 shape, 11.27 GB of routed FP8 weights): streamed, default ring, ALL 4096
        tokens against the oracle; streamed == resident bit for bit; whole experts' hq / hs / Y row by row.
  cfg 2 (T = 32768): resident single pass, streamed single pass, 8 resident chunks and 8 streamed chunks,
        all bit-identical; >= 2048 tokens against the oracle; hq / hs / Y of whole >= 1000-row experts
        (many tiles per persistent CTA, weight-scale rotation at K block 32, Y staging reuse).
  cfg 3 (Zipf-skewed routing, T = 16384, streamed, empty experts skipped) and cfg 4 (128-expert softmax
        layer, T = 8192, resident and streamed): >= 2048 tokens each, whole experts' intermediates.

Token subsets follow SURVEY.md 8(d): the tile-boundary rows (first, 127, 128, last) of >= 8 experts, all
rows of the 4 least- and 4 most-loaded non-empty experts are compared at the Y level (row by row, each
against the oracle's expert_ffn on the same quantised rows), and the layer output is compared on the
boundary-row tokens plus a seeded random fill up to >= 2048 tokens the oracle computes one by one.
Routing, quantised hidden bytes and the permutation are checked for EVERY token.
"""

import time

import numpy as np
import pytest
import torch

from oracle import moe_layer, expert_ffn, dequantize_rows_1x128, dequantize_weight_128x128, bf16_bits_to_f64
from oracle import e4m3_decode as decode
from oracle.acceptance import compare_routing, compare_output
from paper_2606_10493_b200 import SlpMoeLayer, inputs
from gpu_util import read_y_rows, y_tolerance

pytestmark = pytest.mark.gpu

N_SUBSET = 2048


@pytest.fixture(scope="module")
def dsv3():
    """cfg 1 / cfg 2 share their weights (same seed, same shape)."""
    cfg = inputs.CONFIGS[1]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    return W, inputs.weights_as_numpy(W)


def oracle_layer(cfg, Wn, hidden, tokens):
    t0 = time.perf_counter()
    ref = moe_layer(inputs.hidden_as_bits(hidden), Wn, top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk, scoring=cfg.scoring,
                    norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale, tokens=tokens)
    print(f"{cfg.name}: oracle on {len(tokens)} of {cfg.T} tokens in {time.perf_counter() - t0:.1f} s")
    return ref


def expert_weights(Wn, cfg, e):
    if e == cfg.E:
        return [Wn[k] for k in ("shared_gate_q", "shared_gate_s", "shared_up_q", "shared_up_s", "shared_down_q", "shared_down_s")]
    return [Wn[k][e] for k in ("gate_q", "gate_s", "up_q", "up_s", "down_q", "down_s")]


def loaded_extremes(counts, n=4):
    nonempty = np.nonzero(counts > 0)[0]
    order = nonempty[np.argsort(counts[nonempty], kind="stable")]
    return [int(e) for e in order[:n]], [int(e) for e in order[-n:]]


def boundary_tokens(cfg, counts, row_start, row_token, n_experts=8, seed=0):
    """Tokens sitting on the tile-boundary rows (0, 127, 128, last) of `n_experts` experts: the least- and
    most-loaded ones plus a seeded pick of the rest."""
    rng = np.random.default_rng(seed)
    lo, hi = loaded_extremes(counts, 2)
    nonempty = np.nonzero(counts > 0)[0]
    rest = [int(e) for e in rng.permutation(nonempty) if e not in lo + hi][:max(0, n_experts - len(lo) - len(hi))]
    toks = set()
    for e in lo + hi + rest:
        n = int(counts[e])
        for r in (0, 127, 128, n - 1, n // 128 * 128 - 1, n // 128 * 128):
            if 0 <= r < n:
                toks.add(int(row_token[row_start[e] + r]))
    return toks, lo + hi + rest


def subset_tokens(cfg, counts, row_start, row_token, n_total=N_SUBSET, seed=0):
    toks, experts = boundary_tokens(cfg, counts, row_start, row_token, seed=seed)
    rng = np.random.default_rng(seed + 1)
    for t in rng.permutation(cfg.T):
        if len(toks) >= n_total:
            break
        toks.add(int(t))
    return np.array(sorted(toks)), experts


def check_layer_output(cfg, Wn, hidden, out, idx, w, tokens):
    ref = oracle_layer(cfg, Wn, hidden, tokens)
    r = compare_routing(idx, w, ref["route"])                       # every token
    print(cfg.name, "routing", {k: v for k, v in r.items() if k != "members_equal"})
    assert r["passed"], r
    o = compare_output(inputs.hidden_as_bits(out)[tokens], ref["out_f64"], r["members_equal"][tokens])
    print(cfg.name, "output on", len(tokens), "tokens:", o)
    assert o["passed"], o
    return ref, r, o


def check_expert_intermediates(cfg, Wn, layer, ref_xq, ref_xs, counts, row_start, row_token, experts, max_rows=None):
    """a5-a7 row by row at full size: hq / hs against the oracle's expert_ffn on the same quantised rows, Y
    against the float64 product of the GPU's OWN codes (so a legitimately flipped code upstream does not
    blur the check).  Same bars as the reduced-size test in test_gpu_parity.py."""
    hs_stride = (cfg.I // 128 + 3) // 4 * 4
    n_codes = n_flip = 0
    for e in experts:
        if e == cfg.E:
            r0, n = 0, cfg.T
        else:
            r0, n = int(row_start[e]), int(counts[e])
        if max_rows is not None and n > max_rows:                    # head and tail of a very long expert
            pick = np.r_[0:max_rows // 2, n - max_rows // 2:n]
        else:
            pick = np.arange(n)
        toks = np.arange(cfg.T)[pick] if e == cfg.E else row_token[r0:r0 + n][pick]
        ws = expert_weights(Wn, cfg, e)
        y_ref, hq_ref, hs_ref = expert_ffn(ref_xq[toks], ref_xs[toks], *ws)
        g_hq = layer.debug_rows("hq", np.uint8, r0, n, cfg.I)[pick]
        g_hs = layer.debug_rows("hs", np.float32, r0, n, hs_stride)[pick][:, :cfg.I // 128]
        g_y = read_y_rows(layer, cfg, r0, n)[pick]
        assert np.allclose(g_hs, hs_ref, rtol=3e-6, atol=0), (e, np.abs(g_hs / hs_ref - 1).max())
        diff = g_hq != hq_ref
        n_codes += diff.size
        n_flip += int(diff.sum())
        if diff.any():                                               # flipped codes are neighbours on the e4m3 grid
            a, b = decode(g_hq[diff]), decode(hq_ref[diff])
            step = np.maximum(np.abs(a), np.abs(b)) / 8 + 2.0 ** -9
            assert (np.abs(a - b) <= step * 1.0001).all(), e
        y_own = dequantize_rows_1x128(g_hq, g_hs) @ dequantize_weight_128x128(ws[4], ws[5]).T
        rms = np.sqrt((y_own ** 2).mean())
        tol = y_tolerance(y_own, rms)
        bad = np.abs(g_y - y_own) > tol
        assert not bad.any(), (e, float(np.abs(g_y - y_own).max() / rms), int(bad.sum()))
    print(cfg.name, "experts", experts, "codes", n_codes, "differ", n_flip)
    assert n_flip <= 1e-4 * n_codes
    return n_codes, n_flip


def run_layer(layer, hidden, T):
    out = layer.prefill(hidden).clone()
    torch.cuda.synchronize()
    idx, w, counts = layer.debug_routing(T)
    row_start = layer.debug_buffer("row_start", np.int32)
    row_token = layer.debug_buffer("row_token", np.int32)
    return out, idx, w, counts, row_start, row_token


def test_cfg1_all_tokens_streamed_and_resident(dsv3):
    """BASELINE config 1 in bench.py's launch configuration (streamed, default ring): EVERY token's output
    against the oracle, every token's routing and quantised hidden bytes, streamed == resident bitwise."""
    W, Wn = dsv3
    cfg = inputs.CONFIGS[1]
    hidden = inputs.make_hidden(cfg, device=torch.device("cuda", 0))
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out_s, idx, w, counts, row_start, row_token = run_layer(layer, hidden, cfg.T)
        out_s2 = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        st = layer.stats()
        xq, xs = layer.debug_quant_hidden(cfg.T)
        ref, r, o = check_layer_output(cfg, Wn, hidden, out_s, idx, w, np.arange(cfg.T))
        assert o["rows"] >= cfg.T - r["near_tie_tokens"]
        assert np.array_equal(xq, ref["xq"]) and np.array_equal(xs, ref["xs"])
        lo, hi = loaded_extremes(counts)
        check_expert_intermediates(cfg, Wn, layer, ref["xq"], ref["xs"], counts, row_start, row_token, lo + hi + [cfg.E])
        layer.set_residency("resident")
        out_r = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
    finally:
        layer.close()
    assert torch.equal(out_s.view(torch.int16), out_s2.view(torch.int16)), "streamed run-to-run differs"
    assert torch.equal(out_s.view(torch.int16), out_r.view(torch.int16)), "streamed != resident"
    assert st["experts_copied"] == cfg.E and st["bytes_copied"] == 11274289152


def test_cfg2_32k_resident_streamed_chunked(dsv3):
    """BASELINE config 2: one 32K-token pass resident (the launch bench.py times under resident_32k) and
    streamed (64-expert launch groups with ~1000 rows per expert), and 8 chunks of 4096 in both modes
    (Q20): all four bit-identical; >= 2048 tokens and whole >= 1000-row experts against the oracle."""
    W, Wn = dsv3
    cfg = inputs.CONFIGS[2]
    hidden = inputs.make_hidden(cfg, device=torch.device("cuda", 0))
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        layer.set_residency("resident")
        out, idx, w, counts, row_start, row_token = run_layer(layer, hidden, cfg.T)
        st = layer.stats()
        assert st["experts_copied"] == 0 and counts.sum() == cfg.T * cfg.k
        tokens, _ = subset_tokens(cfg, counts, row_start, row_token)
        assert len(tokens) >= N_SUBSET
        ref, r, o = check_layer_output(cfg, Wn, hidden, out, idx, w, tokens)
        lo, hi = loaded_extremes(counts)
        assert counts[hi[-1]] >= 1000
        check_expert_intermediates(cfg, Wn, layer, ref["xq"], ref["xs"], counts, row_start, row_token, lo + hi)
        check_expert_intermediates(cfg, Wn, layer, ref["xq"], ref["xs"], counts, row_start, row_token, [cfg.E], max_rows=1024)
        parts = [layer.prefill(hidden[r0:r0 + 4096].contiguous()).clone() for r0 in range(0, cfg.T, 4096)]
        torch.cuda.synchronize()
        assert torch.equal(torch.cat(parts).view(torch.int16), out.view(torch.int16)), "resident: chunked != single pass"
        layer.set_residency("streamed")
        out_s = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        st = layer.stats()
        assert st["experts_copied"] == cfg.E and st["bytes_copied"] == 11274289152
        assert torch.equal(out_s.view(torch.int16), out.view(torch.int16)), "streamed 32K pass != resident"
        parts = [layer.prefill(hidden[r0:r0 + 4096].contiguous()).clone() for r0 in range(0, cfg.T, 4096)]
        torch.cuda.synchronize()
        assert torch.equal(torch.cat(parts).view(torch.int16), out.view(torch.int16)), "streamed: chunked != single pass"
    finally:
        layer.close()


def test_cfg2_resident_soak_is_bitwise_stable(dsv3):
    """120 back-to-back resident 32K-token calls (the chip settles under its power cap, clocks move, CTAs take
    different tiles from the dynamic scheduler every time): every output equals the first bit for bit, the
    in-kernel watchdog never fires.  A hand-off race in the GEMM pipeline would show here as a flipped output."""
    W, _ = dsv3
    cfg = inputs.CONFIGS[2]
    hidden = inputs.make_hidden(cfg, device=torch.device("cuda", 0))
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        layer.set_residency("resident")
        first = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        out = torch.empty_like(first)
        for i in range(120):
            layer.prefill(hidden, out=out)
            if i % 10 == 9:
                torch.cuda.synchronize()
                assert torch.equal(out.view(torch.int16), first.view(torch.int16)), f"call {i} differs from the first"
        layer.stats()   # raises if a pipeline wait timed out
    finally:
        layer.close()


def test_cfg2_cta_pair_kernel_full_size(dsv3):
    """The cta_group::2 variant (triage "gemm=pair") at full size: resident 32K pass against the oracle on
    the tile-boundary tokens, and streamed with empty launch groups impossible here but 64-expert groups."""
    W, Wn = dsv3
    cfg = inputs.CONFIGS[2]
    hidden = inputs.make_hidden(cfg, device=torch.device("cuda", 0))
    layer = SlpMoeLayer(cfg, W, device=0, triage="gemm=pair")
    try:
        layer.set_residency("resident")
        out, idx, w, counts, row_start, row_token = run_layer(layer, hidden, cfg.T)
        toks, _ = boundary_tokens(cfg, counts, row_start, row_token, n_experts=8)
        tokens = np.array(sorted(toks))
        check_layer_output(cfg, Wn, hidden, out, idx, w, tokens)
    finally:
        layer.close()


def test_cfg3_zipf_streamed_skip_empty():
    """BASELINE config 3: skewed routing (several experts > 5 % of tokens, many with 0-3 rows), streamed,
    experts without tokens neither copied nor run; fixed-order streaming gives the same bits."""
    cfg = inputs.CONFIGS[3]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    Wn = inputs.weights_as_numpy(W)
    hidden = inputs.make_hidden(cfg, device=dev)
    layer = SlpMoeLayer(cfg, W, device=0, skip_empty_experts=True)
    try:
        out, idx, w, counts, row_start, row_token = run_layer(layer, hidden, cfg.T)
        st = layer.stats()
        n_empty = int((counts == 0).sum())
        print("cfg3 histogram: empty", n_empty, "<=3 rows", int((counts <= 3).sum()), "max share", counts.max() / cfg.T)
        assert n_empty >= 32 and (counts <= 3).sum() >= 64 and (counts > 0.05 * cfg.T).sum() >= 3
        assert st["experts_skipped"] == n_empty and st["experts_copied"] == cfg.E - n_empty
        tokens, _ = subset_tokens(cfg, counts, row_start, row_token)
        ref, r, o = check_layer_output(cfg, Wn, hidden, out, idx, w, tokens)
        lo, hi = loaded_extremes(counts)
        check_expert_intermediates(cfg, Wn, layer, ref["xq"], ref["xs"], counts, row_start, row_token, lo + hi, max_rows=1536)
    finally:
        layer.close()
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out_all = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
    finally:
        layer.close()
    assert torch.equal(out.view(torch.int16), out_all.view(torch.int16)), "skip_empty changes the output"


def test_cfg4_softmax_resident_and_streamed():
    """BASELINE config 4: 128 experts, softmax routing, no grouping, no shared expert, I = 1536."""
    cfg = inputs.CONFIGS[4]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    Wn = inputs.weights_as_numpy(W)
    hidden = inputs.make_hidden(cfg, device=dev)
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out_s = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        layer.set_residency("resident")
        out_r, idx, w, counts, row_start, row_token = run_layer(layer, hidden, cfg.T)
        tokens, _ = subset_tokens(cfg, counts, row_start, row_token)
        ref, r, o = check_layer_output(cfg, Wn, hidden, out_r, idx, w, tokens)
        lo, hi = loaded_extremes(counts)
        check_expert_intermediates(cfg, Wn, layer, ref["xq"], ref["xs"], counts, row_start, row_token, lo + hi)
    finally:
        layer.close()
    assert torch.equal(out_s.view(torch.int16), out_r.view(torch.int16)), "streamed != resident"


def test_cfg1_smallep_eight_emulated_ranks(dsv3):
    """SmallEP at full size: 8 handles over disjoint 32-expert ranges of the cfg 1 layer on one
    GPU.  Each streams 11.27 GB / 8 per pass (the point of expert sharding on a host-link-bound path), the fp32
    partial sums added in rank order and rounded once match the oracle on the tile-boundary tokens and the
    single-handle output to within one bf16 ulp."""
    from paper_2606_10493_b200 import finalize_partial, sharding, smallep
    W, Wn = dsv3
    cfg = inputs.CONFIGS[1]
    G = 8
    hidden = inputs.make_hidden(cfg, device=torch.device("cuda", 0))
    single = SlpMoeLayer(cfg, W, device=0)
    try:
        out_single, idx, w, counts, row_start, row_token = run_layer(single, hidden, cfg.T)
    finally:
        single.close()
    total = None
    for r in range(G):
        e0, e1 = smallep.expert_range(cfg.E, r, G)
        layer = SlpMoeLayer(cfg, W, device=0, expert_range=(e0, e1))
        try:
            p = layer.prefill_partial(hidden, shared_tokens=sharding.token_range(cfg.T, r, G))
            torch.cuda.synchronize()
            st = layer.stats()
        finally:
            layer.close()
        assert st["experts_copied"] == 32 and st["bytes_copied"] == 11274289152 // G
        total = p.clone() if total is None else total.add_(p)
    out = finalize_partial(total)
    toks, _ = boundary_tokens(cfg, counts, row_start, row_token, n_experts=8)
    rng = np.random.default_rng(5)
    tokens = np.array(sorted(toks | set(rng.choice(cfg.T, 64, replace=False).tolist())))
    check_layer_output(cfg, Wn, hidden, out, idx, w, tokens)
    from test_gpu_smallep import close_to_single_gpu
    ok, frac = close_to_single_gpu(out, out_single)
    print("smallep x8 vs single handle: within one bf16 step:", ok, "fraction differing", frac)
    assert ok and frac < 2e-2


def test_cfg5_kimi_k2_shape_streamed():
    """The paper's second model shape: 384 routed experts (16.9 GB of FP8 weights per layer),
    top-8 without expert groups, T = 4096, streamed.  384 / 32 = 12 experts per lane is not a power of two, so
    this runs the general top-k kernel; routing is checked for every token, the output on sampled tokens."""
    cfg = inputs.CONFIGS[5]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    Wn = inputs.weights_as_numpy(W)
    hidden = inputs.make_hidden(cfg, device=dev)
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out, idx, w, counts, row_start, row_token = run_layer(layer, hidden, cfg.T)
        st = layer.stats()
        out2 = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
    finally:
        layer.close()
    assert st["experts_copied"] == 384 and st["bytes_copied"] == 384 * 3 * 2048 * 7168       # 16.9 GB
    assert abs(st["bytes_copied"] / 1e9 - 16.9) < 0.05
    assert torch.equal(out.view(torch.int16), out2.view(torch.int16))
    toks, _ = boundary_tokens(cfg, counts, row_start, row_token, n_experts=4)
    rng = np.random.default_rng(9)
    tokens = np.array(sorted(toks | set(rng.choice(cfg.T, 16, replace=False).tolist())))
    check_layer_output(cfg, Wn, hidden, out, idx, w, tokens)
