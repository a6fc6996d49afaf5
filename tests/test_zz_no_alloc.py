"""slp_moe_permute_static: the histogram / scan / permute step for callers that cannot allocate.

Some users of this library run where device memory cannot be requested: a serving process that gave
all of HBM to its own pool at start-up, or a plugin called from a loop in which the host forbids
cudaMalloc because it stalls the GPU.  For them the library keeps the step's scratch in a fixed
616 KiB array inside libslpmoe.so; the caller passes every input and output.  These tests check that
this entry point writes exactly what the handle-based path (slp_moe_prefill, read back through the
debug exports) writes for the same routing, twice in a row with different shapes, so that whatever the
first call left in the shared array would show up in the second if the call relied on it.

The file name sorts after every other test file on purpose: `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests.  The GPU test makes no assumption about what ran
before it in the process (it passes alone in a fresh process and after the whole suite).
"""

import numpy as np
import pytest
import torch

import __graft_entry__ as entry
from paper_2606_10493_b200 import SlpMoeLayer, SlpError, inputs, permute_static, permute_static_rows


def _cfg(**kw):
    base = dict(name="no_alloc", T=1000, H=256, E=64, k=8, G=8, Gk=4, I=128, n_shared=1, scoring="sigmoid_bias",
                norm_topk=True, routed_scale=2.5, seed=31, bias="normal", mode="resident")
    base.update(kw)
    return inputs.LayerConfig(**base)


def _existing_path(cfg):
    """Routing and permutation tables of the handle-based path for cfg's seeded inputs."""
    W = inputs.make_weights(cfg, device="cpu", pin=True)
    hidden = inputs.make_hidden(cfg, device="cpu")
    layer = SlpMoeLayer(cfg, W, device=0)
    try:
        layer.set_residency("resident")
        layer.prefill(hidden.cuda())
        torch.cuda.synchronize()
        idx, _, counts = layer.debug_routing(cfg.T)
        ref = dict(idx=idx, counts=counts, row_start=layer.debug_buffer("row_start", np.int32),
                   pos=layer.debug_buffer("pos", np.int32).reshape(cfg.T, cfg.k),
                   row_token=layer.debug_buffer("row_token", np.int32))
    finally:
        layer.close()
    return ref


def _static_path(cfg, idx, bufs, check_driver_memory):
    """One slp_moe_permute_static call into buffers that were allocated before the call.  `check_driver_memory`: also
    require that the device's free memory as the driver reports it did not move (not on the first call of a process,
    where loading the kernels' module may take device memory)."""
    counts, row_start, pos, row_token = bufs
    for b in bufs:
        b.fill_(-7)   # stale caller memory must not leak into the result either
    d_idx = torch.from_numpy(idx).cuda()
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    permute_static(d_idx, cfg.E, counts, row_start, pos[:cfg.T * cfg.k].view(cfg.T, cfg.k), row_token)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    if check_driver_memory:
        assert torch.cuda.mem_get_info()[0] == free_before
    return dict(counts=counts[:cfg.E].cpu().numpy(), row_start=row_start[:cfg.E + 2].cpu().numpy(),
                pos=pos[:cfg.T * cfg.k].view(cfg.T, cfg.k).cpu().numpy(), row_token=row_token.cpu().numpy())


@pytest.mark.gpu
def test_static_scratch_permute_matches_the_handle_path_on_consecutive_calls():
    entry.build()
    torch.cuda.set_device(0)
    # different T, E and k per call: the second call is smaller than the first (stale histograms and tile tables of
    # a larger problem stay in the array), the third is the largest, the fourth repeats the first
    cases = [_cfg(), _cfg(T=513, E=16, k=4, G=1, Gk=1, n_shared=0, scoring="softmax", routed_scale=1.0, bias="none", seed=32),
             _cfg(T=2048, bias="zipf", seed=33), _cfg()]
    refs = [_existing_path(c) for c in cases]
    cap = max(permute_static_rows(c.T, c.k, c.E) for c in cases)
    bufs = (torch.empty(512, dtype=torch.int32, device="cuda"), torch.empty(514, dtype=torch.int32, device="cuda"),
            torch.empty(max(c.T * c.k for c in cases), dtype=torch.int32, device="cuda"),
            torch.empty(cap, dtype=torch.int32, device="cuda"))
    for n, (c, ref) in enumerate(zip(cases, refs)):   # back to back, nothing of the existing path in between
        got = _static_path(c, ref["idx"], bufs, check_driver_memory=n > 0)
        rows = int(got["row_start"][c.E + 1])   # rows in use
        # integer work: bit-exact, as in the parity tests of the handle path
        assert np.array_equal(got["counts"], ref["counts"]), c.name
        assert np.array_equal(got["row_start"][:c.E + 1], ref["row_start"]), c.name
        assert np.array_equal(got["pos"], ref["pos"]), c.name
        assert rows == ref["row_token"].size and rows <= permute_static_rows(c.T, c.k, c.E)
        assert np.array_equal(got["row_token"][:rows], ref["row_token"]), c.name
        bound = permute_static_rows(c.T, c.k, c.E)
        assert (got["row_token"][rows:bound] == -1).all() and (got["row_token"][bound:] == -7).all()
        # and it is a permutation: every assignment has its own row, whose token is t
        t_of = got["row_token"][got["pos"].reshape(-1)]
        assert np.array_equal(t_of, np.repeat(np.arange(c.T, dtype=np.int32), c.k))
        assert np.unique(got["pos"]).size == c.T * c.k


def test_static_scratch_limits_are_reported_before_any_device_use():
    """Sizes beyond the fixed array are refused with a message that names the limit (checked before the device is
    touched, so this runs without a GPU)."""
    entry.build()
    from paper_2606_10493_b200 import binding
    L = binding.lib()
    assert permute_static_rows(1000, 8, 64) == 1024 + 16128   # roundup128(T) + roundup128(T * k + 127 * E)
    assert permute_static_rows(-1, 8, 64) == -1
    for T, k, E, word in ((32769, 8, 256, "tokens"), (32768, 9, 256, "assignments"), (128, 8, 512, "n_experts"),
                          (128, 33, 256, "top_k"), (128, 0, 256, "top_k")):
        st = L.slp_moe_permute_static(0, None, T, k, E, None, None, None, None, 0, None)
        assert st == -2, (T, k, E)
        assert word in L.slp_last_error().decode()
    assert L.slp_moe_permute_static(0, None, 0, 8, 256, None, None, None, None, 0, None) == 0     # T == 0: nothing to do
    assert L.slp_moe_permute_static(0, None, 128, 8, 256, None, None, None, None, 0, None) == -1  # NULL buffers
    with pytest.raises(SlpError):
        binding._check(L.slp_moe_permute_static(0, None, 128, 8, 256, None, None, None, None, 0, None))
