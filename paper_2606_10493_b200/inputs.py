"""Seeded synthetic inputs for the SLP MoE layer (shared by tests, bench and the oracle's callers).

This module holds NONE of the method's arithmetic: it only draws random tensors with torch's
generators and stores weights in the e4m3 + 128x128-block-scale byte format using torch's own
float8_e4m3fn conversion (a library routine, independent of both the CUDA kernels and the
oracle's codec).  The bytes it returns are the ground truth for both sides.

Recipe (stand-ins for the real DeepSeek-V3 / Qwen3-style checkpoints the paper
measures on, which are not available here):
  hidden    bf16(N(0,1))                                  [T, H]
  router_w  fp32 N(0, 1/sqrt(H))                          [E, H]
  bias      fp32 N(0, 0.01)  | none | zipf (cfg 3)        [E]
  experts   N(0, 0.02) fp32 -> per 128x128 block s = amax/448 (fp32), q = e4m3_rne(w / s)
Every tensor has its own generator seeded from (cfg.seed, tensor id, expert/chunk index), so
any expert or any 4096-row hidden chunk can be regenerated alone, and cfg 2's first 4096 hidden
rows equal cfg 1's (same seed).
The stream a seed produces depends on the device the generator lives on (CPU Mersenne vs CUDA
Philox); whichever produced the bytes, the host copies are what both sides consume.
"""

from dataclasses import dataclass, replace
import math

import numpy as np
import torch

BLOCK = 128
HIDDEN_CHUNK = 4096


@dataclass(frozen=True)
class LayerConfig:
    name: str
    T: int                    # tokens per call
    H: int                    # hidden
    E: int                    # routed experts
    k: int                    # top-k
    G: int                    # n_group
    Gk: int                   # topk_group
    I: int                    # moe_intermediate
    n_shared: int             # shared experts (intermediate = I each)
    scoring: str              # "sigmoid_bias" | "softmax"
    norm_topk: bool
    routed_scale: float
    seed: int
    bias: str                 # "normal" | "none" | "zipf"
    mode: str                 # default residency the config is quoted in

    def with_tokens(self, T):
        return replace(self, T=T)


# BASELINE.json:configs, in order.
CONFIGS = [
    LayerConfig("cfg0_tiny", 64, 256, 8, 2, 1, 1, 128, 0, "sigmoid_bias", True, 2.5, 0, "normal", "resident"),
    LayerConfig("cfg1_dsv3_T4096", 4096, 7168, 256, 8, 8, 4, 2048, 1, "sigmoid_bias", True, 2.5, 1, "normal", "streamed"),
    LayerConfig("cfg2_dsv3_T32768", 32768, 7168, 256, 8, 8, 4, 2048, 1, "sigmoid_bias", True, 2.5, 1, "normal", "streamed"),
    LayerConfig("cfg3_dsv3_zipf_T16384", 16384, 7168, 256, 8, 8, 4, 2048, 1, "sigmoid_bias", True, 2.5, 2, "zipf", "streamed"),
    LayerConfig("cfg4_softmax128_T8192", 8192, 4096, 128, 8, 1, 1, 1536, 0, "softmax", True, 1.0, 3, "none", "resident"),
    # not a BASELINE config: the 384-expert Kimi-K2-shaped layer the paper also serves (16.9 GB of
    # routed FP8 weights per layer): top-8 of 384, no expert groups, one shared expert.
    LayerConfig("cfg5_k2_T4096", 4096, 7168, 384, 8, 1, 1, 2048, 1, "sigmoid_bias", True, 2.827, 4, "normal", "streamed"),
]

_TENSOR_IDS = dict(hidden=1, router_w=2, bias=3, gate=4, up=5, down=6,
                   shared_gate=7, shared_up=8, shared_down=9, zipf_perm=10)


def _gen(cfg_seed, tensor, index, device):
    g = torch.Generator(device=device)
    g.manual_seed((cfg_seed * 1000003 + _TENSOR_IDS[tensor]) * 7919 + index)
    return g


def make_hidden(cfg, device="cpu", T=None, first_chunk=0):
    """bf16 N(0,1) hidden states [T, H], generated in independent 4096-row chunks.  `first_chunk`
    offsets the chunk index: rank r of a token-sharded run takes chunks [r * n, (r + 1) * n)."""
    T = cfg.T if T is None else T
    out = torch.empty((T, cfg.H), dtype=torch.bfloat16, device=device)
    for c in range((T + HIDDEN_CHUNK - 1) // HIDDEN_CHUNK):
        r0 = c * HIDDEN_CHUNK
        n = min(HIDDEN_CHUNK, T - r0)
        x = torch.randn((HIDDEN_CHUNK, cfg.H), generator=_gen(cfg.seed, "hidden", first_chunk + c, device),
                        device=device, dtype=torch.float32)
        out[r0:r0 + n] = x[:n].to(torch.bfloat16)
    return out


def _zipf_bias(cfg, device):
    """Correction bias giving Zipf(1.2) expert popularity over a random expert permutation,
    with an explicit near-empty and empty tail (cfg 3).

    Closed form, no routing arithmetic: with logits ~ N(0,1), an expert with bias b is selected
    roughly when sigmoid(z) + b > tau, i.e. with probability p = 1 - Phi(logit(tau - b)); so for a
    target p the bias is b = tau - sigmoid(Phi^-1(1 - p)).  tau is arbitrary (only differences
    matter); it is set so the median bias is 0.
    """
    E, T, k = cfg.E, cfg.T, cfg.k
    perm = torch.randperm(E, generator=_gen(cfg.seed, "zipf_perm", 0, "cpu"))
    rank = torch.empty(E, dtype=torch.long)
    rank[perm] = torch.arange(1, E + 1)
    r = rank.double()
    n_head, n_ragged = E // 2, E // 4
    zipf = r.pow(-1.2)
    p = k * zipf / zipf[rank <= E].sum()
    p = p.clamp(max=0.6)
    ragged = (rank > n_head) & (rank <= n_head + n_ragged)
    rows = (3 - ((rank - n_head - 1) % 3)).double()           # 3, 2, 1, 3, 2, 1 ...
    p = torch.where(ragged, rows / T, p)
    theta = torch.sigmoid(torch.special.ndtri(1.0 - p))
    tau = theta[rank <= n_head].median()
    bias = tau - theta
    bias = torch.where(rank > n_head + n_ragged, torch.full_like(bias, -1.0), bias)
    return bias.float().to(device)


def make_router(cfg, device="cpu"):
    w = torch.randn((cfg.E, cfg.H), generator=_gen(cfg.seed, "router_w", 0, device),
                    device=device, dtype=torch.float32) / math.sqrt(cfg.H)
    if cfg.bias == "normal":
        b = torch.randn((cfg.E,), generator=_gen(cfg.seed, "bias", 0, device),
                        device=device, dtype=torch.float32) * 0.01
    elif cfg.bias == "zipf":
        b = _zipf_bias(cfg, device)
    else:
        b = None
    return w, b


def quantize_weight_128x128(w):
    """fp32 [N, K] -> (uint8 e4m3 codes [N, K], fp32 scales [N/128, K/128]); w ~= q * s."""
    N, K = w.shape
    wb = w.reshape(N // BLOCK, BLOCK, K // BLOCK, BLOCK)
    amax = wb.abs().amax(dim=(1, 3))
    s = torch.where(amax == 0, torch.ones_like(amax), amax / 448.0)
    q = (wb / s[:, None, :, None]).clamp(-448.0, 448.0).to(torch.float8_e4m3fn)
    return q.reshape(N, K).view(torch.uint8), s


def _make_matrix(cfg, tensor, index, N, K, device):
    w = torch.randn((N, K), generator=_gen(cfg.seed, tensor, index, device),
                    device=device, dtype=torch.float32) * 0.02
    return quantize_weight_128x128(w)


def make_weights(cfg, device="cpu", pin=False, experts=None, shard=None):
    """All layer weights as HOST tensors (pinned if `pin`), generated on `device`.

    Returns a dict of torch tensors:
      router_w [E,H] f32, router_bias [E] f32 | None,
      gate_q/up_q [E,I,H] u8, gate_s/up_s [E,I/128,H/128] f32,
      down_q [E,H,I] u8, down_s [E,H/128,I/128] f32,
      shared_* (same shapes without the E axis) | None.
    `experts`: optional iterable restricting which experts are generated (others left zero);
    used by sampled full-size checks to save time.
    `shard` = (e0, e1): allocate and generate only experts e0 .. e1 - 1 (an expert-parallel rank's share,
    same bytes as the full layer's); the per-expert tensors then have e1 - e0 entries and the dict carries
    "expert_offset" = e0.
    """
    E, H, I = cfg.E, cfg.H, cfg.I
    e_off = 0
    if shard is not None:
        e_off, E = shard[0], shard[1] - shard[0]
        experts = None

    def host(shape, dtype):
        return torch.empty(shape, dtype=dtype, pin_memory=pin)

    out = {}
    rw, rb = make_router(cfg, device)
    out["router_w"] = rw.cpu()
    out["router_bias"] = None if rb is None else rb.cpu()
    out["gate_q"], out["gate_s"] = host((E, I, H), torch.uint8), host((E, I // BLOCK, H // BLOCK), torch.float32)
    out["up_q"], out["up_s"] = host((E, I, H), torch.uint8), host((E, I // BLOCK, H // BLOCK), torch.float32)
    out["down_q"], out["down_s"] = host((E, H, I), torch.uint8), host((E, H // BLOCK, I // BLOCK), torch.float32)
    todo = range(E) if experts is None else experts
    if experts is not None:
        for key in ("gate_q", "up_q", "down_q"):
            out[key].zero_()
        for key in ("gate_s", "up_s", "down_s"):
            out[key].fill_(1.0)
    if shard is not None:
        out["expert_offset"] = e_off
    for e in todo:
        for name, N, K in (("gate", I, H), ("up", I, H), ("down", H, I)):
            q, s = _make_matrix(cfg, name, e_off + e, N, K, device)
            out[name + "_q"][e].copy_(q)
            out[name + "_s"][e].copy_(s)
    for name, N, K in (("shared_gate", I, H), ("shared_up", I, H), ("shared_down", H, I)):
        if cfg.n_shared:
            assert cfg.n_shared == 1
            q, s = _make_matrix(cfg, name, 0, N, K, device)
            hq, hs = host(q.shape, torch.uint8), host(s.shape, torch.float32)
            hq.copy_(q)
            hs.copy_(s)
            out[name + "_q"], out[name + "_s"] = hq, hs
        else:
            out[name + "_q"], out[name + "_s"] = None, None
    return out


def weights_as_numpy(weights):
    """Zero-copy numpy views of `make_weights` output, in the mapping the oracle takes."""
    return {k: (v if v is None or isinstance(v, int) else v.numpy()) for k, v in weights.items()}


def hidden_as_bits(hidden):
    """torch bf16 [T,H] (any device) -> numpy uint16 bit patterns on the host."""
    return hidden.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def routed_bytes_per_expert(cfg):
    return 3 * cfg.I * cfg.H


def fp8_flops_per_token(cfg):
    """FP8 FLOPs per token: 2*3*H*I per (token, expert) pair, k routed + n_shared shared."""
    return 2 * 3 * cfg.H * cfg.I * (cfg.k + cfg.n_shared)
