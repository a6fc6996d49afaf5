"""Pins for oracle/acceptance.py — the gate every parity claim passes through.

Negative controls: each plausible way a wrong CUDA result could slip through (a one-e4m3-step
error in one expert's contribution, a swapped expert, a membership flip outside the near-tie
window, a wrong routing weight, a NaN, an empty comparison) must FAIL; the legitimate
differences north_star allows (bf16 output rounding, order-only index differences, membership
flips inside the 1e-4 near-tie window) must PASS.  The bars themselves are north_star's
(BASELINE.json: "output relative L2 error <= 1e-2 and max abs error <= 3e-2 x output RMS";
"expert indices bit-exact, except tokens whose k-th/(k+1)-th score gap is below 1e-4").
"""

import numpy as np

from oracle import moe_layer, expert_ffn, f64_to_bf16_bits
from oracle.acceptance import compare_routing, compare_output, NEAR_TIE, REL_L2_BAR, MAX_ABS_BAR
from paper_2606_10493_b200 import inputs


def _layer(seed=21, T=48, E=8, k=2):
    cfg = inputs.LayerConfig(name="acc", T=T, H=256, E=E, k=k, G=1, Gk=1, I=128, n_shared=1,
                             scoring="sigmoid_bias", norm_topk=True, routed_scale=2.5, seed=seed,
                             bias="normal", mode="resident")
    W = inputs.weights_as_numpy(inputs.make_weights(cfg))
    hb = inputs.hidden_as_bits(inputs.make_hidden(cfg))
    ref = moe_layer(hb, W, top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk, scoring=cfg.scoring,
                    norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
    return cfg, W, hb, ref


def test_bars_are_north_stars():
    assert NEAR_TIE == 1e-4 and REL_L2_BAR == 1e-2 and MAX_ABS_BAR == 3e-2


def test_exact_and_bf16_rounded_outputs_pass():
    cfg, W, hb, ref = _layer()
    o = compare_output(ref["out_bf16"], ref["out_f64"])
    assert o["passed"] and o["rows"] == cfg.T
    assert o["rel_l2"] < 3e-3 and o["max_abs_over_rms"] < 2e-2      # half an ulp of bf16 at most
    r = compare_routing(ref["route"]["idx"].copy(), ref["route"]["w"].astype(np.float32), ref["route"])
    assert r["passed"] and r["membership_mismatch_bad"] == 0 and r["order_only_mismatch"] == 0


def test_one_e4m3_step_in_one_experts_output_fails():
    """One expert's contribution off by one e4m3 step (2^-3 relative) on its tokens: the kind of
    error a wrong scale index or a stale weight slot would produce.  Must break the max bar."""
    cfg, W, hb, ref = _layer()
    idx, w = ref["route"]["idx"], ref["route"]["w"]
    e = int(np.argmax(ref["route"]["counts"]))
    rows, slots = np.nonzero(idx == e)
    y, _, _ = expert_ffn(ref["xq"][rows], ref["xs"][rows], W["gate_q"][e], W["gate_s"][e], W["up_q"][e],
                         W["up_s"][e], W["down_q"][e], W["down_s"][e])
    bad = ref["out_f64"].copy()
    bad[rows] += 0.125 * w[rows, slots][:, None] * y
    o = compare_output(f64_to_bf16_bits(bad), ref["out_f64"])
    assert not o["passed"] and o["max_abs_over_rms"] > MAX_ABS_BAR


def test_swapped_expert_fails():
    """A token computed with a different expert than the one routed (same weight) must fail."""
    cfg, W, hb, ref = _layer()
    idx, w = ref["route"]["idx"], ref["route"]["w"]
    t = 5
    e_old, e_new = int(idx[t, 0]), int((idx[t, 0] + 1) % cfg.E)
    if e_new in idx[t]:
        e_new = int(next(x for x in range(cfg.E) if x not in idx[t]))
    args = lambda e: (W["gate_q"][e], W["gate_s"][e], W["up_q"][e], W["up_s"][e], W["down_q"][e], W["down_s"][e])
    y_old, _, _ = expert_ffn(ref["xq"][t:t + 1], ref["xs"][t:t + 1], *args(e_old))
    y_new, _, _ = expert_ffn(ref["xq"][t:t + 1], ref["xs"][t:t + 1], *args(e_new))
    bad = ref["out_f64"].copy()
    bad[t] += w[t, 0] * (y_new[0] - y_old[0])
    o = compare_output(f64_to_bf16_bits(bad), ref["out_f64"])
    assert not o["passed"]


def test_uniform_two_percent_error_fails_l2_bar():
    cfg, W, hb, ref = _layer()
    o = compare_output(f64_to_bf16_bits(ref["out_f64"] * 1.02), ref["out_f64"])
    assert not o["passed"] and o["rel_l2"] > REL_L2_BAR
    o = compare_output(f64_to_bf16_bits(ref["out_f64"] * 1.002), ref["out_f64"])
    assert o["passed"]                                                # 0.2 % stays inside both bars


def test_single_element_outlier_fails_max_bar_only():
    cfg, W, hb, ref = _layer()
    rms = np.sqrt(np.mean(ref["out_f64"] ** 2))
    bad = ref["out_f64"].copy()
    bad[3, 17] += 0.05 * rms
    o = compare_output(f64_to_bf16_bits(bad), ref["out_f64"])
    assert not o["passed"] and o["rel_l2"] < REL_L2_BAR and o["max_abs_over_rms"] > MAX_ABS_BAR


def test_nonfinite_output_fails():
    cfg, W, hb, ref = _layer()
    bits = ref["out_bf16"].copy()
    bits[0, 0] = 0x7FC0                                               # bf16 NaN
    o = compare_output(bits, ref["out_f64"])
    assert not o["passed"] and not o["finite"]
    bits[0, 0] = 0x7F80                                               # +inf
    assert not compare_output(bits, ref["out_f64"])["passed"]


def test_zero_valid_rows_does_not_pass_silently():
    cfg, W, hb, ref = _layer()
    o = compare_output(ref["out_bf16"], ref["out_f64"], np.zeros(cfg.T, bool))
    assert o["rows"] == 0 and not o["passed"]
    o = compare_output(ref["out_bf16"][:0], ref["out_f64"][:0])
    assert o["rows"] == 0 and not o["passed"]


def _route_with_gaps(ref, expert_gap=None, group_gap=None):
    route = dict(ref["route"])
    if expert_gap is not None:
        route["expert_gap"] = expert_gap
    if group_gap is not None:
        route["group_gap"] = group_gap
    return route


def test_membership_flip_outside_near_tie_fails_inside_passes():
    cfg, W, hb, ref = _layer()
    idx = ref["route"]["idx"].copy()
    w32 = ref["route"]["w"].astype(np.float32)
    t = 7
    outsider = int(next(x for x in range(cfg.E) if x not in idx[t]))
    idx[t, -1] = outsider
    wide = np.full(cfg.T, 1e-2)
    r = compare_routing(idx, w32, _route_with_gaps(ref, expert_gap=wide, group_gap=np.full(cfg.T, np.inf)))
    assert not r["passed"] and r["membership_mismatch_bad"] == 1 and not r["members_equal"][t]
    # exactly at the allowance (gap == 1e-4 is NOT below it): still a failure
    edge = wide.copy()
    edge[t] = NEAR_TIE
    r = compare_routing(idx, w32, _route_with_gaps(ref, expert_gap=edge, group_gap=np.full(cfg.T, np.inf)))
    assert not r["passed"]
    # inside the near-tie window of the expert gap: counted, reported, not a failure
    tie = wide.copy()
    tie[t] = 0.5 * NEAR_TIE
    r = compare_routing(idx, w32, _route_with_gaps(ref, expert_gap=tie, group_gap=np.full(cfg.T, np.inf)))
    assert r["passed"] and r["membership_mismatch_near_tie"] == 1 and r["membership_mismatch_bad"] == 0
    assert not r["members_equal"][t]                                  # ... and the token is excluded from the output metrics
    # inside the near-tie window of the GROUP gap (reading Q4)
    gtie = np.full(cfg.T, np.inf)
    gtie[t] = 0.5 * NEAR_TIE
    r = compare_routing(idx, w32, _route_with_gaps(ref, expert_gap=wide, group_gap=gtie))
    assert r["passed"] and r["membership_mismatch_near_tie"] == 1


def test_order_only_difference_passes_and_is_counted():
    cfg, W, hb, ref = _layer()
    idx = ref["route"]["idx"].copy()
    w32 = ref["route"]["w"].astype(np.float32)
    idx[4] = idx[4, ::-1]
    w32[4] = w32[4, ::-1]
    r = compare_routing(idx, w32, _route_with_gaps(ref, expert_gap=np.full(cfg.T, 1e-2)))
    assert r["passed"] and r["order_only_mismatch"] == 1 and r["membership_mismatch_bad"] == 0
    assert r["max_weight_err"] < 1e-6                                 # weights are compared per expert, not per slot


def test_wrong_routing_weight_fails():
    cfg, W, hb, ref = _layer()
    idx = ref["route"]["idx"].copy()
    w32 = ref["route"]["w"].astype(np.float32)
    w32[9, 0] *= 1.001                                                # 1e-3 relative on a weight of O(1)
    r = compare_routing(idx, w32, ref["route"])
    assert not r["passed"] and r["max_weight_err"] > 3e-5
    # weights attached to the wrong experts (swapped within the token) also fail
    w32 = ref["route"]["w"].astype(np.float32)
    if abs(w32[9, 0] - w32[9, 1]) > 1e-3:
        w32[9, 0], w32[9, 1] = w32[9, 1], w32[9, 0]
        assert not compare_routing(idx, w32, ref["route"])["passed"]


def test_mismatched_tokens_are_excluded_from_output_metrics():
    """A token whose membership legitimately differs (near-tie) may have any output: it must not
    count towards the L2 / max metrics, while the other rows still do."""
    cfg, W, hb, ref = _layer()
    valid = np.ones(cfg.T, bool)
    valid[11] = False
    bad = ref["out_f64"].copy()
    bad[11] *= 3.0
    o = compare_output(f64_to_bf16_bits(bad), ref["out_f64"], valid)
    assert o["passed"] and o["rows"] == cfg.T - 1
    assert not compare_output(f64_to_bf16_bits(bad), ref["out_f64"])["passed"]
