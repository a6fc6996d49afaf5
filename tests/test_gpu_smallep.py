"""SmallEP (expert-sharded streaming) on one GPU: G handles over disjoint expert ranges play the
G ranks.  Every handle routes all tokens, streams and runs only its own experts, and returns an fp32 partial sum;
the partials are added in rank order and rounded once.  The oracle for the result is the single-GPU layer
(SURVEY.md 4): the oracle itself under the acceptance rule, and the single-handle CUDA output to within one bf16
ulp (the fp32 additions associate differently, nothing else changes)."""

import numpy as np
import pytest
import torch

from oracle.acceptance import compare_routing, compare_output
from paper_2606_10493_b200 import SlpMoeLayer, SlpError, finalize_partial, inputs, sharding, smallep
from test_gpu_parity import problem, CASES, small_dsv3

# T = 1020 (Tpad = 1024) over 3 ranks: the last rank's shared-expert token range is [680, 1020), which neither starts
# on a 32-row boundary nor ends more than 31 rows before Tpad (the 32-row output groups of the down kernel)
CASES["mini_dsv3_1020"] = small_dsv3(name="mini_dsv3_1020", T=1020, seed=15)

pytestmark = pytest.mark.gpu


def close_to_single_gpu(out, out_single):
    """The expert-sharded result differs from the single-handle one only in how the fp32 additions associate, so
    after the one bf16 rounding the two agree to one bf16 step of the value (2^-7 relative); near zero, where a
    step is meaningless, to 1e-3 of the output RMS.  Returns (ok, fraction of elements that differ at all)."""
    a, b = out.float(), out_single.float()
    rms = float(b.pow(2).mean().sqrt())
    ok = bool(((a - b).abs() <= 2.0 ** -7 * b.abs() + 1e-3 * rms).all())
    return ok, float((a != b).float().mean())


@pytest.mark.parametrize("name,G", [(n, G) for n in ("mini_dsv3_ragged", "mini_zipf", "mini_softmax") for G in (2, 4)] +
                         [("mini_dsv3_1020", 3)])
@pytest.mark.parametrize("mode", ["resident", "streamed"])
def test_emulated_ranks_match_single_gpu(name, G, mode):
    cfg, W, hidden, ref = problem(name)
    x = hidden.cuda()
    single = SlpMoeLayer(cfg, W, device=0)
    try:
        single.set_residency(mode)
        out_single = single.prefill(x).clone()
        whole_f32 = single.prefill_partial(x, shared_tokens=(0, cfg.T)).clone()     # unsharded handle: the layer in fp32
        torch.cuda.synchronize()
    finally:
        single.close()
    assert torch.equal(finalize_partial(whole_f32).view(torch.int16), out_single.view(torch.int16))   # same FMA order, same rounding

    partials, copied = [], []
    for r in range(G):
        e0, e1 = smallep.expert_range(cfg.E, r, G)
        Wr = inputs.make_weights(cfg, device="cpu", pin=True, shard=(e0, e1))     # this rank's share only (same bytes)
        layer = SlpMoeLayer(cfg, Wr, device=0, expert_range=(e0, e1))
        try:
            layer.set_residency(mode)
            with pytest.raises(SlpError):
                layer.prefill(x)                                                   # a shard cannot produce the final output alone
            p = layer.prefill_partial(x, shared_tokens=sharding.token_range(cfg.T, r, G) if cfg.n_shared else (0, 0))
            torch.cuda.synchronize()
            st = layer.stats()
            idx, w, counts = layer.debug_routing(cfg.T)
            partials.append(p.clone())
            copied.append(st["bytes_copied"])
        finally:
            layer.close()
        rr = compare_routing(idx, w, ref["route"])                                 # every rank routes the full batch
        assert rr["passed"], rr
        assert copied[-1] == (0 if mode == "resident" else (e1 - e0) * 3 * cfg.I * cfg.H)
    if mode == "streamed":
        assert sum(copied) == cfg.E * 3 * cfg.I * cfg.H                            # the weight pass is split, not replicated
    out = finalize_partial(smallep.reduce_partials_in_rank_order(partials))
    o = compare_output(inputs.hidden_as_bits(out), ref["out_f64"], rr["members_equal"])
    assert o["passed"], o
    ok, frac = close_to_single_gpu(out, out_single)
    assert ok and frac < 2e-2, frac


@pytest.mark.parametrize("mode", ["resident", "streamed"])
@pytest.mark.parametrize("rng", [(997, 1020), (1, 1020), (33, 34), (680, 1020), (1019, 1020)])
def test_arbitrary_shared_token_range_on_an_unsharded_handle(mode, rng):
    """The shared expert over [t0, t1) for ranges that start anywhere: tokens inside get exactly the full layer's fp32
    sum, tokens outside exactly the routed-only sum (the routed rows next to the shared region stay intact)."""
    cfg, W, hidden, _ = problem("mini_dsv3_1020")
    x = hidden.cuda()
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        layer.set_residency(mode)
        whole = layer.prefill_partial(x, shared_tokens=(0, cfg.T)).clone()
        routed = layer.prefill_partial(x, shared_tokens=(0, 0)).clone()
        part = layer.prefill_partial(x, shared_tokens=rng).clone()
        torch.cuda.synchronize()
        row_start = layer.debug_buffer("row_start", np.int32)
    finally:
        layer.close()
    t0, t1 = rng
    assert torch.equal(part[t0:t1], whole[t0:t1])
    assert torch.equal(part[:t0], routed[:t0]) and torch.equal(part[t1:], routed[t1:])
    assert not torch.equal(whole[t0:t1], routed[t0:t1])
    assert row_start[cfg.E] == t0 // 32 * 32


def test_world_size_one_runner_equals_prefill():
    """SmallEpLayer with one rank: no collective, the partial path must reproduce slp_moe_prefill bit for bit."""
    cfg, W, hidden, ref = problem("mini_dsv3")
    x = hidden.cuda()
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        a = layer.prefill(x).clone()
        b = smallep.SmallEpLayer(layer, cfg, 0, 1).prefill(x).clone()
        torch.cuda.synchronize()
    finally:
        layer.close()
    assert torch.equal(a.view(torch.int16), b.view(torch.int16))


def test_bad_expert_ranges_are_rejected():
    cfg, W, hidden, _ = problem("mini_dsv3")
    for rng in ((5, 3), (0, cfg.E + 1), (-1, 4), (4, 0)):
        with pytest.raises(SlpError) as ei:
            SlpMoeLayer(cfg, W, device=0, expert_range=rng)
        assert ei.value.status == -1


def test_one_rank_nccl_group_runs_the_collectives():
    """The NCCL lines of SmallEpLayer (all_gather_into_tensor on bf16, reduce_scatter_tensor on fp32, then
    slp_moe_finalize_partial) executed on a real process group of one rank: with one rank they move the data unchanged,
    so the result must be slp_moe_prefill's bit for bit."""
    import socket
    import torch.distributed as dist
    cfg, W, hidden, ref = problem("mini_dsv3_ragged")
    x = hidden.cuda()
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1,
                            device_id=torch.device("cuda", 0))
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        a = layer.prefill(x).clone()
        runner = smallep.SmallEpLayer(layer, cfg, 0, 1, always_collective=True)
        assert runner.collective
        b = runner.prefill(x).clone()
        c = runner.prefill(x).clone()      # second call reuses the gathered / partial buffers
        torch.cuda.synchronize()
    finally:
        layer.close()
        dist.destroy_process_group()
    assert torch.equal(a.view(torch.int16), b.view(torch.int16)) and torch.equal(b.view(torch.int16), c.view(torch.int16))
