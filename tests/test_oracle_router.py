"""Pins for the oracle's router (O3) and permutation (O8).

Brute force here is a pure-Python, per-token restatement of the definition,
written with loops and Python's own sort; the G = 1 case is also checked against torch.topk.
"""

import math

import numpy as np
import pytest
import torch

from oracle import router, permutation, bf16_bits_to_f64


def rand_inputs(T, H, E, seed, bias_std=0.01):
    g = torch.Generator().manual_seed(seed)
    x = torch.randn(T, H, generator=g).to(torch.bfloat16)
    w = (torch.randn(E, H, generator=g) / math.sqrt(H)).float()
    b = (torch.randn(E, generator=g) * bias_std).float()
    bits = x.view(torch.int16).numpy().view(np.uint16)
    return bits, w.numpy(), b.numpy()


def brute_force_route(bits, w, b, k, G, Gk, scoring, norm, scale):
    """Per-token loops; returns list of (idx list, weight list)."""
    x = bf16_bits_to_f64(bits)
    T, H = x.shape
    E = w.shape[0]
    out = []
    for t in range(T):
        logit = [sum(float(x[t, h]) * float(w[e, h]) for h in range(H)) for e in range(E)]
        if scoring == "sigmoid_bias":
            s = [1.0 / (1.0 + math.exp(-l)) for l in logit]
            sel = [s[e] + (float(b[e]) if b is not None else 0.0) for e in range(E)]
        else:
            m = max(logit)
            ex = [math.exp(l - m) for l in logit]
            z = sum(ex)
            s = [v / z for v in ex]
            sel = list(s)
        allowed = set(range(E))
        if G > 1:
            gs = E // G
            gscore = []
            for g in range(G):
                members = sorted((sel[e] for e in range(g * gs, (g + 1) * gs)), reverse=True)
                gscore.append(members[0] + members[1] if gs >= 2 else members[0])
            best = sorted(range(G), key=lambda g: (-gscore[g], g))[:Gk]
            allowed = {e for e in range(E) if e // gs in best}
        cand = sorted(allowed, key=lambda e: (-sel[e], e))[:k]
        tot = sum(s[e] for e in cand) if norm else 1.0
        out.append((cand, [s[e] / tot * scale for e in cand]))
    return out


@pytest.mark.parametrize("E,k,G,Gk,scoring,norm,scale", [
    (8, 2, 1, 1, "sigmoid_bias", True, 2.5),
    (16, 4, 4, 2, "sigmoid_bias", True, 2.5),
    (32, 8, 8, 4, "sigmoid_bias", True, 2.5),
    (16, 3, 1, 1, "softmax", True, 1.0),
    (16, 3, 1, 1, "softmax", False, 1.0),
    (12, 2, 3, 1, "sigmoid_bias", False, 1.5),
])
def test_router_vs_brute_force(E, k, G, Gk, scoring, norm, scale):
    bits, w, b = rand_inputs(24, 64, E, seed=E * 31 + k)
    bias = b if scoring == "sigmoid_bias" else None
    r = router(bits, w, bias, top_k=k, n_group=G, topk_group=Gk, scoring=scoring,
               norm_topk=norm, routed_scale=scale)
    ref = brute_force_route(bits, w, bias, k, G, Gk, scoring, norm, scale)
    for t, (cand, wt) in enumerate(ref):
        assert list(r["idx"][t]) == cand
        assert np.allclose(r["w"][t], wt, rtol=1e-12, atol=0)


def test_router_invariants_dsv3_like():
    E, k, G, Gk = 64, 8, 8, 4
    bits, w, b = rand_inputs(500, 128, E, seed=5)
    r = router(bits, w, b, top_k=k, n_group=G, topk_group=Gk, scoring="sigmoid_bias",
               norm_topk=True, routed_scale=2.5)
    idx = r["idx"]
    assert np.allclose(r["w"].sum(axis=1), 2.5, atol=1e-6)                  # sum w = scale
    assert all(len(set(row)) == k for row in idx)                            # distinct
    assert all(len(set(row // (E // G))) <= Gk for row in idx)               # <= Gk groups
    assert r["counts"].sum() == 500 * k
    assert (r["expert_gap"] >= 0).all() and (r["group_gap"] >= 0).all()
    # weights use the UNBIASED score: w_j proportional to sigmoid(logit), not sigmoid + bias
    s = np.take_along_axis(r["score"], idx.astype(np.int64), axis=1)
    assert np.allclose(r["w"], 2.5 * s / s.sum(axis=1, keepdims=True), rtol=1e-12)


def test_router_g1_equals_torch_topk():
    E, k = 40, 6
    bits, w, b = rand_inputs(300, 96, E, seed=9)
    r = router(bits, w, b, top_k=k, n_group=1, topk_group=1, scoring="sigmoid_bias",
               norm_topk=True, routed_scale=1.0)
    x = torch.from_numpy(bf16_bits_to_f64(bits))
    sel = torch.sigmoid(x @ torch.from_numpy(w).double().T) + torch.from_numpy(b).double()
    ref = torch.topk(sel, k, dim=1).indices.numpy()
    assert np.array_equal(r["idx"], ref)


def test_router_k_equals_E_weights_proportional_to_scores():
    E = 8
    bits, w, _ = rand_inputs(50, 32, E, seed=11)
    r = router(bits, w, None, top_k=E, n_group=1, topk_group=1, scoring="sigmoid_bias",
               norm_topk=True, routed_scale=3.0)
    full = np.zeros((50, E))
    np.put_along_axis(full, r["idx"].astype(np.int64), r["w"], axis=1)
    assert np.allclose(full, 3.0 * r["score"] / r["score"].sum(axis=1, keepdims=True), rtol=1e-12)


def test_router_softmax_topk_then_softmax_equivalence():
    """Q7: softmax-then-top-k-then-renormalise == softmax over the selected logits."""
    E, k = 32, 4
    bits, w, _ = rand_inputs(100, 64, E, seed=13)
    r = router(bits, w, None, top_k=k, n_group=1, topk_group=1, scoring="softmax",
               norm_topk=True, routed_scale=1.0)
    lg = np.take_along_axis(r["logits"], r["idx"].astype(np.int64), axis=1)
    ref = torch.softmax(torch.from_numpy(lg), dim=1).numpy()
    assert np.allclose(r["w"], ref, rtol=1e-12)


def test_excluded_groups_never_picked_even_with_negative_bias():
    """Q2: exclusion is -inf, so a kept expert with sel < 0 still beats an excluded one."""
    E, k, G, Gk = 8, 4, 4, 2
    bits, w, _ = rand_inputs(200, 32, E, seed=17)
    b = np.array([0, 0, 0, 0, -2, -2, -2, -2], dtype=np.float32)            # groups 2,3 hopeless
    r = router(bits, w, b, top_k=k, n_group=G, topk_group=Gk, scoring="sigmoid_bias",
               norm_topk=True, routed_scale=1.0)
    assert (r["idx"] < 4).all()


def test_tie_break_lower_index():
    bits = np.zeros((3, 16), dtype=np.uint16)                                # x = 0 -> all logits 0
    w = np.ones((6, 16), dtype=np.float32)
    r = router(bits, w, None, top_k=2, n_group=3, topk_group=2, scoring="sigmoid_bias",
               norm_topk=True, routed_scale=1.0)
    assert (r["idx"] == np.array([0, 1])).all()


def test_permutation_roundtrip_and_order():
    rng = np.random.default_rng(0)
    T, k, E = 257, 4, 19
    idx = np.stack([rng.choice(E, k, replace=False) for _ in range(T)]).astype(np.int32)
    counts, offsets, perm, pos = permutation(idx, E)
    assert offsets[-1] == T * k and counts.sum() == T * k
    # gather-by-perm then scatter-by-pos is the identity on [T*k]
    payload = rng.normal(size=(T, k))
    gathered = np.empty(T * k)
    gathered[pos.reshape(-1)] = payload.reshape(-1)
    assert np.array_equal(gathered[pos], payload)
    assert np.array_equal(perm[pos], np.repeat(np.arange(T)[:, None], k, axis=1))
    for e in range(E):
        rows = perm[offsets[e]:offsets[e + 1]]
        assert (np.diff(rows) > 0).all()                                     # ascending token id
        assert all(e in idx[t] for t in rows)
    assert sorted(pos.reshape(-1).tolist()) == list(range(T * k))
