"""O2..O8 — the MoE layer of stream-loading prefill, step by step (TEST INFRASTRUCTURE ONLY).

What the hot path computes, in the paper's order (Fig. 2 steps 3-5: "tokens on each
rank are gated and sorted to form per-expert token lists (3) ... Local experts execute on those
tokens (4) ... A final weighted sum produces the per-token outputs (5)"), with the FP8 data
format of PAPER.md:108 ("FP8 weights and scales are loaded from VRAM, activations are quantized to
FP8, and ... native FP8 GEMM with FP32 accumulation") and the 128-element K scale blocks of
PAPER.md:235,255.  Where the paper is silent the readings Q1..Q21 of DESIGN.md §3.2 apply; each
is named where it is used.

Everything the definition calls "real arithmetic" is float64 here.  The only roundings are the
ones that are part of the definition: bf16 inputs, e4m3 codes, fp32 scales, and the fp32 division
inside the two activation quantisers (Q12).  Weight streaming moves bytes and
does not change values, so it has no counterpart here.

All arrays are numpy.  bf16 tensors are passed as uint16 bit patterns.
"""

import numpy as np

from .e4m3 import e4m3_decode, e4m3_encode_rne

BLOCK = 128  # scale-block length along K ("128 elements per block")


# ----------------------------------------------------------------------------------------------
# bf16 <-> float64
# ----------------------------------------------------------------------------------------------
def bf16_bits_to_f64(bits):
    """uint16 bf16 bit patterns -> float64 (exact)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def f64_to_bf16_bits(x):
    """float64 -> bf16 bit patterns, one round-to-nearest-even (no double rounding through fp32).

    Normal range only (the layer's outputs are O(1)); bf16 subnormals are not handled specially.
    """
    x = np.asarray(x, dtype=np.float64)
    m, ex = np.frexp(np.abs(x))                      # |x| = m * 2^ex, m in [0.5, 1)
    n = np.rint(m * 256.0)                           # 8 significant bits, ties to even
    val = np.ldexp(n, ex - 8)
    val = np.where(np.isfinite(x), np.copysign(val, x), x)
    return (val.astype(np.float32).view(np.uint32) >> 16).astype(np.uint16)


# ----------------------------------------------------------------------------------------------
# O4 — activation quantisation, 1 x 128 blocks (readings Q10, Q11, Q12)
# ----------------------------------------------------------------------------------------------
def quantize_rows_1x128(x_f32):
    """Per row, per 128 channels: amax -> s = amax / 448 (fp32) -> e4m3(x / s) (fp32 division).

    x_f32: [R, C] float32 (C multiple of 128).  Returns (q uint8 [R, C], s float32 [R, C/128]).
    amax == 0 gives s = 1 and codes 0 (Q11).
    """
    x = np.ascontiguousarray(x_f32, dtype=np.float32)
    R, C = x.shape
    assert C % BLOCK == 0
    xb = x.reshape(R, C // BLOCK, BLOCK)
    amax = np.abs(xb).max(axis=2)                                    # fp32, exact
    s = np.where(amax == 0, np.float32(1.0), amax / np.float32(448.0)).astype(np.float32)
    ratio = (xb / s[:, :, None]).astype(np.float32)                   # IEEE fp32 division (Q12)
    q = e4m3_encode_rne(ratio).reshape(R, C)
    return q, s


def dequantize_rows_1x128(q, s):
    """x_hat = decode(q) * s, in float64 (exact product)."""
    R, C = q.shape
    v = e4m3_decode(q).reshape(R, C // BLOCK, BLOCK)
    return (v * s.astype(np.float64)[:, :, None]).reshape(R, C)


# ----------------------------------------------------------------------------------------------
# O2 — weights are bytes + 128x128 block scales (readings Q8, Q9)
# ----------------------------------------------------------------------------------------------
def dequantize_weight_128x128(q, s):
    """w[n, k] = decode(q[n, k]) * s[n // 128, k // 128], float64 (exact product).

    q: [N, K] uint8, s: [N/128, K/128] float32.
    """
    q = np.asarray(q)
    N, K = q.shape
    assert N % BLOCK == 0 and K % BLOCK == 0
    v = e4m3_decode(q).reshape(N // BLOCK, BLOCK, K // BLOCK, BLOCK)
    sc = np.asarray(s, dtype=np.float64).reshape(N // BLOCK, 1, K // BLOCK, 1)
    return (v * sc).reshape(N, K)


# ----------------------------------------------------------------------------------------------
# O3 — router ("top-k or grouped top-k"; PAPER.md:92 step 3; readings Q1..Q7)
# ----------------------------------------------------------------------------------------------
def router(hidden_bits, router_w, router_bias, *, top_k, n_group, topk_group, scoring,
           norm_topk, routed_scale):
    """Group-limited top-k routing.

    scoring == "sigmoid_bias" (Q1):
        logits = x . W_r^T ; s = sigmoid(logits) ; sel = s + bias
        if n_group > 1: group score = sum of the 2 largest sel in each contiguous group of
        E / n_group experts; keep the topk_group best groups; all other experts are excluded
        (-inf, Q2); then the top_k largest sel among those kept.
        weights w_j = s[idx_j]  (unbiased score), / sum_j s[idx_j] if norm_topk, * routed_scale.
    scoring == "softmax" (Q7):
        p = softmax(logits) over all E; top_k by p; w_j = p[idx_j] (/ sum if norm_topk) * scale.
    Ties: lower expert index / lower group index wins (Q3).  Output order: descending sel.

    Returns a dict: idx [T,k] int32, w [T,k] float64, logits, score (s or p) [T,E],
    expert_gap [T] (k-th minus (k+1)-th kept sel), group_gap [T] (Gk-th minus (Gk+1)-th group
    score; +inf when no group is dropped), counts [E].
    """
    x = bf16_bits_to_f64(hidden_bits)
    W = np.asarray(router_w, dtype=np.float64)
    T, _ = x.shape
    E = W.shape[0]
    logits = x @ W.T
    if scoring == "sigmoid_bias":
        score = 1.0 / (1.0 + np.exp(-logits))
        sel = score.copy()
        if router_bias is not None:
            sel = sel + np.asarray(router_bias, dtype=np.float64)[None, :]
    elif scoring == "softmax":
        z = logits - logits.max(axis=1, keepdims=True)
        ez = np.exp(z)
        score = ez / ez.sum(axis=1, keepdims=True)
        sel = score.copy()
    else:
        raise ValueError(scoring)

    group_gap = np.full(T, np.inf)
    if n_group > 1:
        gs = E // n_group
        assert gs * n_group == E
        selg = sel.reshape(T, n_group, gs)
        if gs >= 2:
            top2 = np.sort(selg, axis=2)[:, :, -2:]
            gscore = top2.sum(axis=2)
        else:
            gscore = selg[:, :, 0]
        gorder = np.argsort(-gscore, axis=1, kind="stable")          # ties: lower group first
        keep = np.zeros((T, n_group), dtype=bool)
        np.put_along_axis(keep, gorder[:, :topk_group], True, axis=1)
        if topk_group < n_group:
            gsorted = np.take_along_axis(gscore, gorder, axis=1)
            group_gap = gsorted[:, topk_group - 1] - gsorted[:, topk_group]
        sel = np.where(np.repeat(keep, gs, axis=1), sel, -np.inf)

    order = np.argsort(-sel, axis=1, kind="stable")                  # ties: lower expert first
    idx = order[:, :top_k]
    sel_sorted = np.take_along_axis(sel, order, axis=1)
    if top_k < E:
        expert_gap = sel_sorted[:, top_k - 1] - sel_sorted[:, top_k]  # +inf if (k+1)-th excluded
    else:
        expert_gap = np.full(T, np.inf)
    picked = np.take_along_axis(score, idx, axis=1)
    w = picked / picked.sum(axis=1, keepdims=True) if norm_topk else picked.copy()
    w = w * float(routed_scale)
    counts = np.bincount(idx.reshape(-1), minlength=E).astype(np.int64)
    return dict(idx=idx.astype(np.int32), w=w, logits=logits, score=score,
                expert_gap=expert_gap, group_gap=group_gap, counts=counts)


# ----------------------------------------------------------------------------------------------
# O8 — permutation into per-expert token lists ("sorted to form per-expert token
# lists")
# ----------------------------------------------------------------------------------------------
def permutation(idx, n_experts):
    """Rows of expert e = the tokens with e in their top-k, ascending token id.

    Returns counts [E], offsets [E+1] (exclusive scan), perm [T*k] (token id of each permuted
    row), pos [T,k] (row of (t, j) in the permuted order) with perm[pos[t, j]] == t.
    """
    idx = np.asarray(idx)
    T, k = idx.shape
    counts = np.bincount(idx.reshape(-1), minlength=n_experts).astype(np.int64)
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    perm = np.empty(T * k, dtype=np.int64)
    pos = np.empty((T, k), dtype=np.int64)
    fill = offsets[:-1].copy()
    for t in range(T):                                   # ascending token id by construction
        for j in range(k):
            e = idx[t, j]
            perm[fill[e]] = t
            pos[t, j] = fill[e]
            fill[e] += 1
    return counts, offsets, perm, pos


# ----------------------------------------------------------------------------------------------
# O5 — one expert's FFN on a set of rows ("gate/up ... SiLU(.) (.) ... down";
# readings Q13, Q14, Q21)
# ----------------------------------------------------------------------------------------------
def expert_ffn(xq, xs, gate_q, gate_s, up_q, up_s, down_q, down_s):
    """y = down( requant( silu(gate(x_hat)) * up(x_hat) ) ) for rows given as (xq, xs).

    x_hat = decode(xq) * xs.  g, u in float64.  a = g / (1 + exp(-g)) * u in float64, no
    intermediate rounding (Q14).  a is requantised per row per 128 channels with the O4 rule
    (amax rounded to fp32, fp32 scale, fp32 division of fp32(a)).  y in float64.

    Returns (y [R, H] float64, hq [R, I] uint8, hs [R, I/128] float32).
    """
    x_hat = dequantize_rows_1x128(xq, xs)
    Wg = dequantize_weight_128x128(gate_q, gate_s)
    g = x_hat @ Wg.T
    del Wg
    Wu = dequantize_weight_128x128(up_q, up_s)
    u = x_hat @ Wu.T
    del Wu
    a = g / (1.0 + np.exp(-g)) * u
    hq, hs = quantize_rows_1x128(a.astype(np.float32))
    a_hat = dequantize_rows_1x128(hq, hs)
    Wd = dequantize_weight_128x128(down_q, down_s)
    y = a_hat @ Wd.T
    return y, hq, hs


# ----------------------------------------------------------------------------------------------
# O6, O7 — whole layer (PAPER.md:48 shared experts "always active"; PAPER.md:92 step 5 "final
# weighted sum"; "router-weighted accumulation"; readings Q15, Q16, Q17)
# ----------------------------------------------------------------------------------------------
def moe_layer(hidden_bits, weights, *, top_k, n_group, topk_group, scoring, norm_topk,
              routed_scale, tokens=None):
    """out[t] = sum_j w[t,j] * FFN_{idx[t,j]}(x_t) + FFN_shared(x_t).  No residual (Q17).

    `weights` is a mapping with router_w [E,H] f32, router_bias [E] f32 or None, and per-expert
    sequences gate_q/gate_s/up_q/up_s/down_q/down_s (index e -> array), plus optional
    shared_gate_q/.../shared_down_s (None when there is no shared expert).

    `tokens`: optional 1-D array of token ids; the FFN/combine is evaluated only for those rows
    (routing is always evaluated for every token).  Returns a dict with the routing dict `route`,
    xq/xs (all tokens), `tokens`, out_f64 [len(tokens), H] and out_bf16 bits.
    """
    hidden_bits = np.asarray(hidden_bits)
    T, H = hidden_bits.shape
    E = np.asarray(weights["router_w"]).shape[0]
    route = router(hidden_bits, weights["router_w"], weights.get("router_bias"),
                   top_k=top_k, n_group=n_group, topk_group=topk_group, scoring=scoring,
                   norm_topk=norm_topk, routed_scale=routed_scale)
    x32 = (np.ascontiguousarray(hidden_bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)
    xq, xs = quantize_rows_1x128(x32)

    tok = np.arange(T) if tokens is None else np.asarray(tokens, dtype=np.int64)
    out = np.zeros((len(tok), H), dtype=np.float64)
    idx_sub = route["idx"][tok]                       # [n, k]
    w_sub = route["w"][tok]
    for e in range(E):
        rows, slots = np.nonzero(idx_sub == e)        # which sampled tokens use expert e
        if len(rows) == 0:
            continue
        y, _, _ = expert_ffn(xq[tok[rows]], xs[tok[rows]],
                             weights["gate_q"][e], weights["gate_s"][e],
                             weights["up_q"][e], weights["up_s"][e],
                             weights["down_q"][e], weights["down_s"][e])
        out[rows] += w_sub[rows, slots][:, None] * y
    if weights.get("shared_gate_q") is not None:
        y, _, _ = expert_ffn(xq[tok], xs[tok],
                             weights["shared_gate_q"], weights["shared_gate_s"],
                             weights["shared_up_q"], weights["shared_up_s"],
                             weights["shared_down_q"], weights["shared_down_s"])
        out += y                                       # weight 1, not scaled (Q16)
    return dict(route=route, xq=xq, xs=xs, tokens=tok, out_f64=out,
                out_bf16=f64_to_bf16_bits(out))
