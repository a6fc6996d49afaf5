"""Full-size parity: BASELINE config 1 (T = 4096, DeepSeek-V3 shape, 11.27 GB of routed FP8
weights) in the launch configuration bench.py times (streamed, default ring), plus resident mode
on the same weights; config 2 (T = 32768: single resident pass, and 8 chunks of 4096 == single pass
bit for bit); config 3 (Zipf-skewed routing, T = 16384, streamed, empty experts skipped); config 4
(128-expert softmax layer, T = 8192, resident and streamed).

The oracle cannot run the full layer in seconds, so:
  - routing, quantised hidden bytes and the permutation are checked for EVERY token;
  - the layer output is checked on sampled tokens the oracle computes one by one (all tokens of
    the least- and most-loaded experts' first rows plus a seeded random sample);
  - properties that hold at any size: run-to-run bitwise identity, streamed == resident bitwise.
"""

import numpy as np
import pytest
import torch

from oracle import moe_layer
from oracle.acceptance import compare_routing, compare_output
from paper_2606_10493_b200 import SlpMoeLayer, inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cfg1():
    cfg = inputs.CONFIGS[1]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    hidden = inputs.make_hidden(cfg, device=dev)
    return cfg, W, hidden


def test_cfg1_streamed_and_resident_sampled(cfg1):
    cfg, W, hidden = cfg1
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out_s = layer.prefill(hidden).clone()
        out_s2 = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        st = layer.stats()
        idx, w, counts = layer.debug_routing(cfg.T)
        xq, xs = layer.debug_quant_hidden(cfg.T)
        layer.set_residency("resident")
        out_r = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
    finally:
        layer.close()
    assert torch.equal(out_s.view(torch.int16), out_s2.view(torch.int16)), "streamed run-to-run differs"
    assert torch.equal(out_s.view(torch.int16), out_r.view(torch.int16)), "streamed != resident"
    assert st["experts_copied"] == cfg.E and st["bytes_copied"] == 11274289152

    hb = inputs.hidden_as_bits(hidden)
    rng = np.random.default_rng(0)
    order = np.argsort(counts)
    picks = set(rng.choice(cfg.T, 6, replace=False).tolist())
    for e in (order[0], order[-1]):                                 # least / most loaded expert
        toks = np.nonzero((idx == e).any(axis=1))[0]
        picks.update(toks[:2].tolist())
    tokens = np.array(sorted(picks))
    ref = moe_layer(hb, inputs.weights_as_numpy(W), top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk,
                    scoring=cfg.scoring, norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale, tokens=tokens)
    r = compare_routing(idx, w, ref["route"])
    print({k: v for k, v in r.items() if k != "members_equal"})
    assert r["passed"], r
    assert np.array_equal(xq, ref["xq"]) and np.array_equal(xs, ref["xs"])
    out_bits = inputs.hidden_as_bits(out_s)[tokens]
    o = compare_output(out_bits, ref["out_f64"], r["members_equal"][tokens])
    print(o, st)
    assert o["passed"], o


def _sampled_check(cfg, W, hidden, out, idx, w, counts, n_random=3, seed=0):
    """Routing for every token, output on a few tokens the oracle computes one by one."""
    hb = inputs.hidden_as_bits(hidden)
    rng = np.random.default_rng(seed)
    picks = set(rng.choice(cfg.T, n_random, replace=False).tolist())
    nonempty = np.nonzero(counts > 0)[0]
    e_small = nonempty[np.argmin(counts[nonempty])]                 # least-loaded non-empty expert
    picks.add(int(np.nonzero((idx == e_small).any(axis=1))[0][-1]))  # its last row: a ragged tile tail
    tokens = np.array(sorted(picks))
    ref = moe_layer(hb, inputs.weights_as_numpy(W), top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk,
                    scoring=cfg.scoring, norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale, tokens=tokens)
    r = compare_routing(idx, w, ref["route"])
    print(cfg.name, {k: v for k, v in r.items() if k != "members_equal"})
    assert r["passed"], r
    o = compare_output(inputs.hidden_as_bits(out)[tokens], ref["out_f64"], r["members_equal"][tokens])
    print(cfg.name, o)
    assert o["passed"], o
    return ref


def test_cfg2_32k_resident_single_pass_and_chunked(cfg1):
    """BASELINE config 2: one 32K-token resident pass (the launch bench.py times under resident_32k),
    and DESIGN.md Q20: 8 chunks of 4096 through the same handle equal the single pass bit for bit."""
    cfg1_, W, _ = cfg1
    cfg = inputs.CONFIGS[2]
    hidden = inputs.make_hidden(cfg, device=torch.device("cuda", 0))
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        layer.set_residency("resident")
        out = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        idx, w, counts = layer.debug_routing(cfg.T)
        st = layer.stats()
        parts = [layer.prefill(hidden[r0:r0 + 4096].contiguous()).clone() for r0 in range(0, cfg.T, 4096)]
        torch.cuda.synchronize()
    finally:
        layer.close()
    assert st["experts_copied"] == 0 and counts.sum() == cfg.T * cfg.k
    assert torch.equal(torch.cat(parts).view(torch.int16), out.view(torch.int16)), "chunked != single pass"
    _sampled_check(cfg, W, hidden, out, idx, w, counts)


def test_cfg3_zipf_streamed_skip_empty():
    """BASELINE config 3: skewed routing (several experts > 5 % of tokens, many with 0-3 rows),
    streamed, experts without tokens neither copied nor run; fixed-order streaming gives the same bits."""
    cfg = inputs.CONFIGS[3]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    hidden = inputs.make_hidden(cfg, device=dev)
    layer = SlpMoeLayer(cfg, W, device=0, skip_empty_experts=True)
    try:
        out = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        st = layer.stats()
        idx, w, counts = layer.debug_routing(cfg.T)
    finally:
        layer.close()
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out_all = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
    finally:
        layer.close()
    n_empty = int((counts == 0).sum())
    print("cfg3 histogram: empty", n_empty, "<=3 rows", int((counts <= 3).sum()), "max share", counts.max() / cfg.T)
    assert n_empty >= 32 and (counts <= 3).sum() >= 64 and (counts > 0.05 * cfg.T).sum() >= 3
    assert st["experts_skipped"] == n_empty and st["experts_copied"] == cfg.E - n_empty
    assert torch.equal(out.view(torch.int16), out_all.view(torch.int16)), "skip_empty changes the output"
    _sampled_check(cfg, W, hidden, out, idx, w, counts)


def test_cfg4_softmax_resident_and_streamed():
    """BASELINE config 4: 128 experts, softmax routing, no grouping, no shared expert, I = 1536."""
    cfg = inputs.CONFIGS[4]
    dev = torch.device("cuda", 0)
    W = inputs.make_weights(cfg, device=dev, pin=True)
    hidden = inputs.make_hidden(cfg, device=dev)
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        out_s = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        layer.set_residency("resident")
        out_r = layer.prefill(hidden).clone()
        torch.cuda.synchronize()
        idx, w, counts = layer.debug_routing(cfg.T)
    finally:
        layer.close()
    assert torch.equal(out_s.view(torch.int16), out_r.view(torch.int16)), "streamed != resident"
    _sampled_check(cfg, W, hidden, out_r, idx, w, counts)
