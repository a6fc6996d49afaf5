"""Host-side logic of the multi-GPU path.

The layer is token-wise (every output row depends on its own input row only), so N GPUs shard the
prompt by tokens with no data-path collective: rank r owns a contiguous token range, runs it
through its own layer replica (weights replicated, each rank streaming over its own host link), and
the only communication is the timing reduction of the bench (max over ranks).  This module holds
that plumbing; it contains none of the method's arithmetic and works on any torch.distributed
backend (`nccl` on GPUs, `gloo` in the CPU tests).
"""

import torch
import torch.distributed as dist

from .inputs import HIDDEN_CHUNK


def token_range(total_tokens, rank, world):
    """Contiguous, balanced split of `total_tokens` rows: the first (total % world) ranks get one more."""
    if world <= 0 or not 0 <= rank < world:
        raise ValueError(f"rank {rank} outside world of {world}")
    base, rem = divmod(total_tokens, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def weak_scaling_first_chunk(tokens_per_rank, rank):
    """Index of the first 4096-row hidden chunk of `rank` when every rank processes its own
    `tokens_per_rank` synthetic tokens (weak scaling): ranks never generate the same rows."""
    return rank * ((tokens_per_rank + HIDDEN_CHUNK - 1) // HIDDEN_CHUNK)


def max_over_ranks(value, device="cpu", group=None):
    """Max of a Python float over all ranks (the bench's device-time reduction)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def whole_job_tokens_per_s(tokens_this_rank, ms_this_rank, device="cpu", group=None):
    """Aggregate throughput: tokens processed by all ranks / the slowest rank's time."""
    ms = max_over_ranks(ms_this_rank, device, group)
    if dist.is_available() and dist.is_initialized():
        t = torch.tensor([float(tokens_this_rank)], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        total = float(t.item())
    else:
        total = float(tokens_this_rank)
    return total / (ms * 1e-3), ms
