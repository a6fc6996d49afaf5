"""Memory-safety evidence without compute-sanitizer (closed on the GPU pool): with triage "guards" every workspace
buffer of a handle sits between two 4 KB canary bands; slp_moe_get_stats and slp_moe_layer_destroy fail if a kernel
wrote into one.  Reduced layers in every kernel variant and residency, ragged token counts, and the full-size
DeepSeek-V3-shaped layer (cfg 1 streamed, T = 4096: every tile of every expert is ragged; cfg 2's first 16K tokens
resident: >= 500 rows per expert, many tiles per CTA)."""

import pytest
import torch

from paper_2606_10493_b200 import SlpMoeLayer, SlpError, inputs
from test_gpu_parity import CASES, problem

pytestmark = pytest.mark.gpu


def run_guarded(cfg, W, hidden, mode, triage):
    layer = SlpMoeLayer(cfg, W, device=0, triage=triage)
    try:
        layer.set_residency(mode)
        for _ in range(2):
            out = layer.prefill(hidden)
            torch.cuda.synchronize()
            layer.stats()          # raises SlpError if a canary band was written
        assert torch.isfinite(out.float()).all()
    finally:
        layer.close()              # checks the bands once more


@pytest.mark.parametrize("name", sorted(CASES))
@pytest.mark.parametrize("mode", ["resident", "streamed"])
@pytest.mark.parametrize("triage", ["guards", "guards,gemm=pair", "guards,gemm=static", "guards,gemm=simt"])
def test_reduced_layers_leave_the_canary_bands_alone(name, mode, triage):
    cfg, W, hidden, _ = problem(name)
    if "pair" in triage and mode == "streamed":
        pytest.skip("the pair variant is exercised in resident mode")
    run_guarded(cfg, W, hidden.cuda(), mode, triage)


@pytest.mark.parametrize("T", [1, 127, 129, 257])
def test_ragged_token_counts_leave_the_canary_bands_alone(T):
    cfg, W, hidden, _ = problem("mini_dsv3_ragged")
    layer = SlpMoeLayer(cfg, W, device=0, triage="guards")
    try:
        out = layer.prefill(hidden[:T].contiguous().cuda())
        torch.cuda.synchronize()
        layer.stats()
        assert out.shape[0] == T
    finally:
        layer.close()


def test_full_size_layer_leaves_the_canary_bands_alone():
    cfg = inputs.CONFIGS[1]
    W = inputs.make_weights(cfg, device="cuda", pin=True)
    hidden = inputs.make_hidden(cfg, device="cuda")
    run_guarded(cfg, W, hidden, "streamed", "guards")
    cfg2 = inputs.CONFIGS[2]
    hidden2 = inputs.make_hidden(cfg2, device="cuda")[:16384].contiguous()
    layer = SlpMoeLayer(cfg2, W, device=0, triage="guards")
    try:
        layer.set_residency("resident")
        layer.prefill(hidden2)
        torch.cuda.synchronize()
        layer.stats()
    finally:
        layer.close()


def test_a_damaged_canary_band_is_reported():
    """Negative control: guards=selftest makes create write one byte behind the counts buffer."""
    cfg, W, hidden, _ = problem("mini_dsv3")
    layer = SlpMoeLayer(cfg, W, device=0, triage="guards=selftest")
    try:
        layer.prefill(hidden.cuda())
        torch.cuda.synchronize()
        with pytest.raises(SlpError) as ei:
            layer.stats()
        assert "d_counts" in str(ei.value) and "overrun" in str(ei.value)
    finally:
        with pytest.raises(SlpError):
            layer.close()
