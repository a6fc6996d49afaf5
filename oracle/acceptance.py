"""Acceptance rule of BASELINE.json:north_star, applied to (CUDA result, oracle result).

Test infrastructure (see oracle/__init__.py).  Nothing here computes the layer; it only compares.

  - expert indices bit-exact, except tokens whose k-th/(k+1)-th selection-score gap (or, reading
    Q4, whose Gk-th/(Gk+1)-th group-score gap) is below 1e-4: those are counted and reported;
  - ordered lists are compared; a mismatch that is only a permutation of the same members is
    "order-only" and does not fail (Q5: the output does not depend on the order);
  - output: relative L2 error <= 1e-2 and max |delta| <= 3e-2 * RMS(oracle output), against the
    oracle's UNROUNDED float64 output, over tokens whose expert membership agrees.
"""

import numpy as np

from .moe_layer import bf16_bits_to_f64

NEAR_TIE = 1e-4
REL_L2_BAR = 1e-2
MAX_ABS_BAR = 3e-2


def compare_routing(idx_gpu, w_gpu, route):
    idx_ref = route["idx"]
    T, k = idx_ref.shape
    same_ordered = (idx_gpu == idx_ref).all(axis=1)
    same_members = np.array([set(a) == set(b) for a, b in zip(idx_gpu, idx_ref)]) if not same_ordered.all() \
        else np.ones(T, bool)
    near = (route["expert_gap"] < NEAR_TIE) | (route["group_gap"] < NEAR_TIE)
    bad = ~same_members & ~near
    # weights: compare per expert (order-insensitive) on tokens with equal membership
    w_err = 0.0
    ok = np.nonzero(same_members)[0]
    if len(ok):
        o_g = np.argsort(idx_gpu[ok], axis=1)
        o_r = np.argsort(idx_ref[ok], axis=1)
        wg = np.take_along_axis(w_gpu[ok].astype(np.float64), o_g, axis=1)
        wr = np.take_along_axis(route["w"][ok], o_r, axis=1)
        w_err = float(np.abs(wg - wr).max())
    return dict(tokens=T, near_tie_tokens=int(near.sum()), order_only_mismatch=int((~same_ordered & same_members).sum()),
                membership_mismatch_near_tie=int((~same_members & near).sum()),
                membership_mismatch_bad=int(bad.sum()), max_weight_err=w_err,
                members_equal=same_members, passed=bool(bad.sum() == 0 and w_err < 3e-5))


def compare_output(out_gpu_bits, out_ref_f64, valid_rows=None):
    """out_gpu_bits: uint16 bf16 [n, H]; out_ref_f64: float64 [n, H]; valid_rows: bool [n]."""
    g = bf16_bits_to_f64(out_gpu_bits)
    r = out_ref_f64
    if valid_rows is not None:
        g, r = g[valid_rows], r[valid_rows]
    if r.size == 0:   # nothing was compared: that is not a pass (pinned by tests/test_oracle_acceptance.py)
        return dict(rel_l2=float("nan"), max_abs_over_rms=float("nan"), rows=0, passed=False, finite=True)
    finite = bool(np.isfinite(g).all())
    d = g - r
    rms = float(np.sqrt(np.mean(r * r)))
    rel = float(np.linalg.norm(d) / max(np.linalg.norm(r), 1e-300))
    mx = float(np.abs(d).max() / max(rms, 1e-300))
    return dict(rel_l2=rel, max_abs_over_rms=mx, rows=int(r.shape[0]), finite=finite,
                passed=bool(finite and rel <= REL_L2_BAR and mx <= MAX_ABS_BAR))
