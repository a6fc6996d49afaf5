"""CPU-side checks of the C-ABI library: it builds, loads without a GPU, exports every symbol
include/slp_moe.h declares, and refuses work loudly when no CUDA device is present."""

import ctypes
import os
import re

import pytest
import torch

import __graft_entry__ as entry
from paper_2606_10493_b200 import binding, inputs, SlpMoeLayer, SlpError

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    entry.build()
    return binding.lib()


def test_exports_every_declared_symbol(built):
    header = open(os.path.join(ROOT, "include", "slp_moe.h")).read()
    body = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(slp_[a-z0-9_]+)\s*\(", body))
    assert declared == set(binding.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(built, name), name
    assert built.slp_version().startswith(b"slpmoe")


def test_struct_sizes_match_header(built):
    # 21 four-byte fields / 14 pointers / see header
    assert ctypes.sizeof(binding._Cfg) == 21 * 4
    header = open(os.path.join(ROOT, "include", "slp_moe.h")).read()
    assert int(re.search(r"#define SLP_MOE_ABI_VERSION (\d+)u", header).group(1)) == binding.ABI_VERSION
    assert f"abi {binding.ABI_VERSION})".encode() in built.slp_version()
    assert ctypes.sizeof(binding._HostWeights) == 14 * 8
    assert ctypes.sizeof(binding.Stats) == 120  # ... + experts_from_prefetch, experts_prefetched, layer, (pad), bytes_prefetched, ms_gateup_shared, ms_down_shared


def test_invalid_arguments_are_reported(built):
    out = ctypes.c_void_p()
    assert built.slp_moe_layer_create(None, None, ctypes.byref(out)) == -1
    assert b"NULL" in built.slp_last_error()
    cfg = binding._Cfg(struct_size=4)
    hw = binding._HostWeights()
    assert built.slp_moe_layer_create(ctypes.byref(cfg), ctypes.byref(hw), ctypes.byref(out)) == -1
    assert b"struct_size" in built.slp_last_error()
    # a caller built against the previous header (20 fields, gemm_impl / router_impl where the expert range is now)
    stale = binding._Cfg(struct_size=80)
    assert built.slp_moe_layer_create(ctypes.byref(stale), ctypes.byref(hw), ctypes.byref(out)) == -1
    assert b"another slp_moe.h" in built.slp_last_error()
    wrong = binding._make_cfg(inputs.CONFIGS[0])
    wrong.abi_version = 2
    plan = binding.Plan(struct_size=ctypes.sizeof(binding.Plan))
    assert built.slp_moe_query_plan(ctypes.byref(wrong), ctypes.byref(plan)) == -1
    assert b"abi_version 2" in built.slp_last_error()
    assert built.slp_moe_prefill(None, None, 1, None, None) == -1
    assert built.slp_moe_layer_destroy(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_gpu_fails_loudly(built):
    cfg = inputs.CONFIGS[0]
    W = inputs.make_weights(cfg)
    with pytest.raises(SlpError) as ei:
        SlpMoeLayer(cfg, W)
    assert ei.value.status == -3 and "no CPU path" in str(ei.value)
    with pytest.raises(SlpError):
        binding.measure_h2d_gbs()


def test_shape_validation_precedes_device_use(built):
    cfg = inputs.CONFIGS[0]
    W = inputs.make_weights(cfg)
    for bad in (dict(H=200), dict(k=40), dict(G=3), dict(E=0)):
        with pytest.raises(SlpError) as ei:
            SlpMoeLayer(inputs.LayerConfig(**{**cfg.__dict__, **bad}), W)
        assert ei.value.status == -2, bad


# ---- host logic reachable without a GPU: slp_moe_query_plan (same validation as create) ----------

def _cfg(**kw):
    from paper_2606_10493_b200 import inputs
    return inputs.LayerConfig(**{**inputs.CONFIGS[1].__dict__, **kw})


def test_query_plan_byte_accounting_matches_the_paper(built):
    """PAPER.md:412 "11.3 GB" of routed FP8 weights per DeepSeek-V3 layer; PAPER.md:140 one ring slot
    = one expert's three FP8 linears (44.5 K tensors = 58 x 256 x 3)."""
    from paper_2606_10493_b200 import inputs
    p = binding.query_plan(inputs.CONFIGS[1])
    assert p["expert_slot_bytes"] == 3 * 2048 * 7168 == 44040192
    assert p["routed_bytes_per_pass"] == 11274289152 and round(p["routed_bytes_per_pass"] / 1e9, 1) == 11.3
    assert p["staging_slots"] == 256 and p["pool_bytes_streamed"] == 257 * 44040192 == p["pool_bytes_resident"]
    assert p["experts_per_launch"] == 64 and p["launch_pairs_streamed"] == 4 + 1        # T = 4096: 128 rows per expert, whole groups
    p32 = binding.query_plan(inputs.CONFIGS[2])                                         # T = 32768: the last group goes in 8-expert pieces
    assert p32["experts_per_launch"] == 64 and p32["launch_pairs_streamed"] == 3 + 8 + 1
    assert p["scale_bytes"] == 257 * 3 * 16 * 56 * 4
    assert p["fp8_flops_per_token"] == 2 * 3 * 2048 * 7168 * 9 == inputs.fp8_flops_per_token(inputs.CONFIGS[1])
    assert p["workspace_rows"] == 4096 + (4096 * 8 + 256 * 127 + 127) // 128 * 128
    assert max(p["gemm_smem_bytes_gateup"], p["gemm_smem_bytes_down"]) <= 227 * 1024
    k2 = binding.query_plan(_cfg(E=384, G=8, Gk=4))            # Kimi-K2-like expert count: "16.9 GB"
    assert round(k2["routed_bytes_per_pass"] / 1e9, 1) == 16.9


def test_query_plan_ring_defaults(built):
    from paper_2606_10493_b200 import inputs
    cfg = inputs.CONFIGS[1]
    assert binding.query_plan(cfg, staging_slots=2)["experts_per_launch"] == 1          # ping-pong
    p = binding.query_plan(cfg, staging_slots=96)
    assert p["staging_slots"] == 96 and p["experts_per_launch"] == 32 and p["pool_bytes_streamed"] == 97 * 44040192
    assert binding.query_plan(cfg, staging_slots=100)["experts_per_launch"] == 25      # largest divisor <= min(32, n/2)
    assert binding.query_plan(cfg, staging_slots=8, experts_per_launch=4)["launch_pairs_streamed"] == 64 + 1
    assert binding.query_plan(inputs.CONFIGS[0])["experts_per_launch"] == 8             # whole tiny layer in one launch


@pytest.mark.parametrize("kw, status", [
    (dict(H=7000), -2), (dict(I=100), -2), (dict(E=600), -2), (dict(E=250), -2),        # shapes
    (dict(G=3), -2), (dict(Gk=9), -2), (dict(k=33), -2), (dict(k=200), -2), (dict(G=8, Gk=1, k=40), -2),
    (dict(n_shared=2), -2),
])
def test_query_plan_rejects_unsupported_shapes(built, kw, status):
    with pytest.raises(binding.SlpError) as ei:
        binding.query_plan(_cfg(**kw))
    assert ei.value.status == status and str(ei.value)


def test_query_plan_rejects_bad_options(built):
    from paper_2606_10493_b200 import inputs
    cfg = inputs.CONFIGS[1]
    for kw in (dict(staging_slots=1), dict(staging_slots=8, experts_per_launch=8), dict(staging_slots=9, experts_per_launch=2),
               dict(max_tokens=-5)):
        with pytest.raises(binding.SlpError) as ei:
            binding.query_plan(cfg, **kw)
        assert ei.value.status == -1, kw


def test_triage_is_a_thread_local_debug_call_not_an_environment_variable(built):
    assert built.slp_moe_debug_set_triage(b"gemm=pair,router=fp32,guards") == 0
    assert built.slp_moe_debug_set_triage(b"gemm=fast") == -1
    assert b"gemm=fast" in built.slp_last_error()
    assert built.slp_moe_debug_set_triage(None) == 0          # back to the product path
    blob = open(binding.library_path(), "rb").read()
    assert b"SLP_TRIAGE" not in blob      # (getenv itself stays imported: the static CUDA runtime uses it)
