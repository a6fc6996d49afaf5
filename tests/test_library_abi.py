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
    # 20 four-byte fields / 14 pointers / see header
    assert ctypes.sizeof(binding._Cfg) == 20 * 4
    assert ctypes.sizeof(binding._HostWeights) == 14 * 8
    assert ctypes.sizeof(binding.Stats) == 88  # 80 + sm_mhz_gateup, sm_mhz_down


def test_invalid_arguments_are_reported(built):
    out = ctypes.c_void_p()
    assert built.slp_moe_layer_create(None, None, ctypes.byref(out)) == -1
    assert b"NULL" in built.slp_last_error()
    cfg = binding._Cfg(struct_size=4)
    hw = binding._HostWeights()
    assert built.slp_moe_layer_create(ctypes.byref(cfg), ctypes.byref(hw), ctypes.byref(out)) == -1
    assert b"struct_size" in built.slp_last_error()
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
