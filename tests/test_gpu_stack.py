"""Multi-layer stack with a cross-layer experts ring (Fig. 5) and one host weight copy shared by
two handles, on reduced layers.  A stack's layer l must give exactly what a single-layer handle on
the same weights gives (same kernels, same bytes: bitwise), while its expert copies are enqueued one layer ahead."""

import ctypes

import numpy as np
import pytest
import torch

from oracle.acceptance import compare_routing, compare_output
from paper_2606_10493_b200 import SlpMoeLayer, SlpError, inputs
from test_gpu_parity import small_dsv3, problem

pytestmark = pytest.mark.gpu

N_LAYERS = 3


@pytest.fixture(scope="module")
def layers():
    cfgs = [small_dsv3(name=f"stack_l{l}", T=700, seed=40 + l) for l in range(N_LAYERS)]
    Ws = [inputs.make_weights(c, device="cpu", pin=True) for c in cfgs]
    hidden = inputs.make_hidden(cfgs[0], device="cpu").cuda()
    singles = []
    for c, W in zip(cfgs, Ws):
        one = SlpMoeLayer(c, W, device=0)
        try:
            singles.append(one.prefill(hidden).clone())
            torch.cuda.synchronize()
        finally:
            one.close()
    return cfgs, Ws, hidden, singles


def test_stack_layers_equal_single_layer_handles_and_prefetch_accounting(layers):
    cfgs, Ws, hidden, singles = layers
    cfg = cfgs[0]
    per_layer = cfg.E * 3 * cfg.I * cfg.H
    stack = SlpMoeLayer(cfg, Ws, device=0)
    try:
        assert stack.n_layers == N_LAYERS
        for rnd in range(2):
            for l in range(N_LAYERS):
                out = stack.prefill(hidden, layer=l).clone()
                torch.cuda.synchronize()
                st = stack.stats()
                assert torch.equal(out.view(torch.int16), singles[l].view(torch.int16)), (rnd, l)
                assert st["layer"] == l
                first = rnd == 0 and l == 0
                # the very first call loads its own experts; every later call finds them prefetched by its predecessor
                assert st["experts_copied"] == (cfg.E if first else 0) and st["bytes_copied"] == (per_layer if first else 0)
                assert st["experts_from_prefetch"] == (0 if first else cfg.E)
                assert st["experts_prefetched"] == cfg.E and st["bytes_prefetched"] == per_layer   # next layer, wrapping to 0
        with pytest.raises(SlpError) as ei:
            stack.set_residency("resident")
        assert ei.value.status == -2
        with pytest.raises(SlpError):
            stack.prefill(hidden, layer=N_LAYERS)
    finally:
        stack.close()


def test_long_calls_launch_the_last_group_in_pieces():
    """A call with >= 256 rows per expert copies and launches its LAST launch group in 8-expert pieces (the call then
    ends a piece's compute, not a group's, after the last copy).  Same bytes, same kernels, same result as the resident
    pass; in a stack the pieces apply to the layer the call loads itself, prefetched layers arrive whole."""
    cfgs = [small_dsv3(name=f"tail_l{l}", T=2100, seed=60 + l) for l in range(2)]     # 2100 * 4 >= 256 * 32
    Ws = [inputs.make_weights(c, device="cpu", pin=True) for c in cfgs]
    hidden = inputs.make_hidden(cfgs[0], device="cpu").cuda()
    cfg = cfgs[0]
    resident = []
    for c, W in zip(cfgs, Ws):
        one = SlpMoeLayer(c, W, device=0)
        try:
            out_s = one.prefill(hidden).clone()
            torch.cuda.synchronize()
            st = one.stats()
            # 1 shared-expert pair + the single 32-expert group as 4 pieces of 8
            assert st["gemm_launches"] == 2 * (1 + 4), st
            assert st["experts_copied"] == cfg.E and st["bytes_copied"] == cfg.E * 3 * cfg.I * cfg.H
            one.set_residency("resident")
            out_r = one.prefill(hidden).clone()
            torch.cuda.synchronize()
            assert one.stats()["gemm_launches"] == 2
            assert torch.equal(out_s.view(torch.int16), out_r.view(torch.int16))
            resident.append(out_r)
        finally:
            one.close()
    stack = SlpMoeLayer(cfg, Ws, device=0)
    try:
        for rnd in range(2):
            for l in range(2):
                out = stack.prefill(hidden, layer=l).clone()
                torch.cuda.synchronize()
                st = stack.stats()
                assert torch.equal(out.view(torch.int16), resident[l].view(torch.int16)), (rnd, l)
                first = rnd == 0 and l == 0
                assert st["gemm_launches"] == (2 * (1 + 4) if first else 2 * (1 + 1)), st   # prefetched layers: one whole group
    finally:
        stack.close()


def test_stack_out_of_order_and_explicit_prefetch(layers):
    cfgs, Ws, hidden, singles = layers
    cfg = cfgs[0]
    stack = SlpMoeLayer(cfg, Ws, device=0)
    try:
        a = stack.prefill(hidden, layer=0).clone()            # prefetches layer 1 ...
        b = stack.prefill(hidden, layer=2).clone()            # ... but layer 2 runs next: the prefetch is overwritten
        torch.cuda.synchronize()
        st = stack.stats()
        assert st["experts_from_prefetch"] == 0 and st["experts_copied"] == cfg.E
        stack.prefetch(1)                                     # explicit loader run-ahead (layer 0 is already prefetched: ring full)
        c = stack.prefill(hidden, layer=1).clone()
        torch.cuda.synchronize()
        st1 = stack.stats()
        d = stack.prefill(hidden, layer=0).clone()
        torch.cuda.synchronize()
    finally:
        stack.close()
    for got, l in ((a, 0), (b, 2), (c, 1), (d, 0)):
        assert torch.equal(got.view(torch.int16), singles[l].view(torch.int16)), l
    assert st1["experts_from_prefetch"] + st1["experts_copied"] == cfg.E


@pytest.mark.parametrize("kw", [dict(staging_slots=8, experts_per_launch=4), dict(staging_slots=2, experts_per_launch=1),
                                dict(staging_slots=16, experts_per_launch=8, skip_empty_experts=True)])
def test_stack_with_a_ring_shorter_than_a_layer(layers, kw):
    """Ring length below the number of experts of a layer (down to 2, ping-pong): only the first ring
    pass of the next layer can be prefetched, the rest streams during the call."""
    cfgs, Ws, hidden, singles = layers
    cfg = cfgs[0]
    stack = SlpMoeLayer(cfg, Ws, device=0, **kw)
    try:
        for l in (0, 1, 2, 0):
            out = stack.prefill(hidden, layer=l).clone()
            torch.cuda.synchronize()
            st = stack.stats()
            assert torch.equal(out.view(torch.int16), singles[l].view(torch.int16)), (kw, l)
            assert st["experts_prefetched"] == kw["staging_slots"]
            assert st["experts_from_prefetch"] + st["experts_copied"] + st["experts_skipped"] == cfg.E
    finally:
        stack.close()


def test_stack_against_oracle(layers):
    from oracle import moe_layer
    cfgs, Ws, hidden, singles = layers
    cfg = cfgs[1]
    ref = moe_layer(inputs.hidden_as_bits(hidden), inputs.weights_as_numpy(Ws[1]), top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk,
                    scoring=cfg.scoring, norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
    stack = SlpMoeLayer(cfg, Ws, device=0)
    try:
        stack.prefill(hidden, layer=0)
        out = stack.prefill(hidden, layer=1).clone()
        torch.cuda.synchronize()
        idx, w, _ = stack.debug_routing(cfg.T)
    finally:
        stack.close()
    r = compare_routing(idx, w, ref["route"])
    o = compare_output(inputs.hidden_as_bits(out), ref["out_f64"], r["members_equal"])
    assert r["passed"] and o["passed"], (r, o)


def test_two_handles_share_one_pageable_host_copy():
    """one resident DRAM copy of the weights serves two consumers.  Two handles borrow the same
    PAGEABLE host tensors: the library page-locks each range once, counts its users, and keeps it locked until the
    last handle goes away."""
    cfg, _, hidden, ref = problem("mini_dsv3")
    W = inputs.make_weights(cfg, device="cpu", pin=False)
    x = hidden.cuda()
    cudart = ctypes.CDLL("libcudart.so.12")
    ptr, nbytes = W["gate_q"].data_ptr(), W["gate_q"].numel()

    def still_registered():
        rc = cudart.cudaHostRegister(ctypes.c_void_p(ptr), ctypes.c_size_t(nbytes), 0)
        if rc == 0:                                    # it was NOT registered any more: undo and report
            cudart.cudaHostUnregister(ctypes.c_void_p(ptr))
            return False
        cudart.cudaGetLastError()
        return True

    a = SlpMoeLayer(cfg, W, device=0)
    b = SlpMoeLayer(cfg, W, device=0, staging_slots=4, experts_per_launch=2)
    try:
        oa = a.prefill(x).clone()
        ob = b.prefill(x).clone()
        torch.cuda.synchronize()
        assert torch.equal(oa.view(torch.int16), ob.view(torch.int16))
        a.close()
        assert still_registered(), "destroying the first handle unpinned memory the second one still streams from"
        ob2 = b.prefill(x).clone()
        torch.cuda.synchronize()
        assert torch.equal(ob2.view(torch.int16), oa.view(torch.int16))
    finally:
        a.close()
        b.close()
    assert not still_registered(), "the last handle must release the registration"
    with pytest.raises(SlpError) as ei:
        SlpMoeLayer(cfg, W, device=0, require_pinned=True)
    assert ei.value.status == -5


def test_longer_range_at_a_registered_pointer_is_not_taken_for_pinned():
    """A shard handle page-locks experts [0, E/2) of a pageable stack; a second handle over all E experts starts at
    the SAME host pointer but needs twice the bytes.  It must not ride on the shorter registration: either create
    refuses (NOT_PINNED: the range is not page-locked end to end) or the whole range is page-locked afterwards."""
    cfg, _, hidden, _ = problem("mini_dsv3")
    W = inputs.make_weights(cfg, device="cpu", pin=False)
    cudart = ctypes.CDLL("libcudart.so.12")
    g = W["gate_q"]
    tail_ptr, tail_bytes = g[cfg.E - 1].data_ptr(), g[cfg.E - 1].numel()

    def tail_is_registered():
        rc = cudart.cudaHostRegister(ctypes.c_void_p(tail_ptr), ctypes.c_size_t(tail_bytes), 0)
        if rc == 0:
            cudart.cudaHostUnregister(ctypes.c_void_p(tail_ptr))
            return False
        cudart.cudaGetLastError()
        return True

    a = SlpMoeLayer(cfg, W, device=0, expert_range=(0, cfg.E // 2))
    try:
        assert not tail_is_registered()
        try:
            b = SlpMoeLayer(cfg, W, device=0)
        except SlpError as e:
            assert e.status == -5 and "page-locked end to end" in str(e)
        else:
            try:
                assert tail_is_registered(), "create accepted a range whose tail is pageable"
            finally:
                b.close()
    finally:
        a.close()
    assert not tail_is_registered()
    full = SlpMoeLayer(cfg, W, device=0)     # with the shard gone the full stack registers normally
    try:
        assert tail_is_registered()
        out = full.prefill(hidden.cuda())
        torch.cuda.synchronize()
        assert torch.isfinite(out.float()).all()
    finally:
        full.close()


def test_a_later_prefetch_replaces_an_unconsumed_one(layers):
    """Run-ahead for layer 2 that nobody consumes must not block the ring: a following prefetch of layer 1 overwrites
    it, and the call on layer 1 then finds all its experts loaded ahead (and computes the right thing)."""
    cfgs, Ws, hidden, singles = layers
    cfg = cfgs[0]
    stack = SlpMoeLayer(cfg, Ws, device=0)
    try:
        stack.prefetch(2)
        stack.prefetch(1)
        stack.prefetch(1)                                  # same groups again: kept, not copied twice
        out = stack.prefill(hidden, layer=1).clone()
        torch.cuda.synchronize()
        st = stack.stats()
        assert st["experts_from_prefetch"] == cfg.E and st["experts_copied"] == 0, st
        assert torch.equal(out.view(torch.int16), singles[1].view(torch.int16))
        out0 = stack.prefill(hidden, layer=0).clone()      # out of order: layer 2 was prefetched behind layer 1, layer 0 is asked for
        torch.cuda.synchronize()
        assert stack.stats()["experts_copied"] == cfg.E
        assert torch.equal(out0.view(torch.int16), singles[0].view(torch.int16))
    finally:
        stack.close()


def test_partial_sums_address_the_layers_of_a_stack(layers):
    """slp_moe_stack_prefill_partial: the fp32 partial path on layer l of a stack.  Unsharded, rounded once, it is
    slp_moe_prefill of that layer bit for bit; over two expert-sharded stacks the partial sums add up to it (to the
    bf16 step the different association of the fp32 additions allows)."""
    from paper_2606_10493_b200 import finalize_partial, smallep
    cfgs, Ws, hidden, singles = layers
    cfg = cfgs[0]
    stack = SlpMoeLayer(cfg, Ws, device=0)
    try:
        for l in (2, 0, 1):
            p = stack.prefill_partial(hidden, shared_tokens=(0, cfg.T), layer=l)
            torch.cuda.synchronize()
            assert stack.stats()["layer"] == l
            assert torch.equal(finalize_partial(p).view(torch.int16), singles[l].view(torch.int16)), l
        with pytest.raises(SlpError) as ei:
            stack.prefill_partial(hidden, shared_tokens=(0, cfg.T), layer=N_LAYERS)
        assert ei.value.status == -1
    finally:
        stack.close()
    G = 2
    shards = [SlpMoeLayer(cfg, Ws, device=0, expert_range=smallep.expert_range(cfg.E, r, G)) for r in range(G)]
    try:
        for l in range(N_LAYERS):
            total = None
            for r, sh in enumerate(shards):
                t0, t1 = r * cfg.T // G, (r + 1) * cfg.T // G
                p = sh.prefill_partial(hidden, shared_tokens=(t0, t1), layer=l)
                torch.cuda.synchronize()
                total = p.clone() if total is None else total + p
            out = finalize_partial(total)
            a, b = out.float(), singles[l].float()
            rms = float(b.pow(2).mean().sqrt())
            assert bool(((a - b).abs() <= 2.0 ** -7 * b.abs() + 1e-3 * rms).all()), l
    finally:
        for sh in shards:
            sh.close()
