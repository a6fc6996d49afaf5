"""SmallEP: expert-sharded stream-loading prefill of one MoE layer over N GPUs (Fig. 6b).

The paper's steps, per layer: (1) all-gather the unsorted tokens, (2) every rank gates and sorts the full batch
locally and keeps only the tokens of its own experts, (3) runs its local experts and forms a partial weighted
sum of shape [N, D], (4) exchanges the partial sums and reduces locally.  Steps 2-3 are one C-ABI call
(`slp_moe_prefill_partial`, hand-written kernels); steps 1 and 4 are NCCL collectives over NVLink / NVSwitch
issued through torch.distributed (all_gather_into_tensor, reduce_scatter_tensor - the paper's all-to-all +
local reduction is a reduce-scatter), and the single bf16 rounding happens after the reduction
(`slp_moe_finalize_partial`).  What this buys on a host-link-bound path: every rank streams only E / N experts
over ITS OWN host link per layer, so the link-bound weight pass shrinks by N.

This module is plumbing: rank arithmetic and the order of the calls.  It holds none of the method's arithmetic.
The shared expert is token-sharded: rank r adds it for its own token range only (PAPER.md:179 argues the load
balance; the shared expert's cost is uniform per token).
"""

import torch
import torch.distributed as dist

from .binding import finalize_partial
from .sharding import token_range


def expert_range(n_experts, rank, world):
    """Contiguous, balanced expert ranges (the first n_experts % world ranks own one more)."""
    return token_range(n_experts, rank, world)


class SmallEpLayer:
    """Drives one expert-sharded SlpMoeLayer handle per rank.  `layer` must have been created with
    expert_range=expert_range(E, rank, world)."""

    def __init__(self, layer, cfg, rank, world, group=None, always_collective=False):
        """`always_collective`: issue the all-gather and the reduce-scatter for world == 1 too (a one-rank process
        group must then exist).  They are copies there, but they are the very calls the multi-rank path makes, so
        a single GPU can execute and time them."""
        self.layer, self.cfg, self.rank, self.world, self.group = layer, cfg, rank, world, group
        self.collective = world > 1 or always_collective
        self._all = None
        self._partial = None
        self._mine = None

    def prefill(self, hidden_shard, out_shard=None):
        """hidden_shard: this rank's [T / world, H] bf16 tokens (equal shards).  Returns its [T / world, H] bf16 output."""
        n, H = hidden_shard.shape
        T = n * self.world
        if self._all is None or self._all.shape[0] != T:
            self._all = torch.empty((T, H), dtype=torch.bfloat16, device=hidden_shard.device)
            self._partial = torch.empty((T, H), dtype=torch.float32, device=hidden_shard.device)
            self._mine = torch.empty((n, H), dtype=torch.float32, device=hidden_shard.device)
        if self.collective:
            dist.all_gather_into_tensor(self._all, hidden_shard, group=self.group)                       # step 1
        else:
            self._all.copy_(hidden_shard)
        t0 = self.rank * n
        self.layer.prefill_partial(self._all, self._partial, shared_tokens=(t0, t0 + n))                 # steps 2-3
        if self.collective:
            dist.reduce_scatter_tensor(self._mine, self._partial, op=dist.ReduceOp.SUM, group=self.group)  # step 4
        else:
            self._mine.copy_(self._partial)
        return finalize_partial(self._mine, out_shard)


def reduce_partials_in_rank_order(partials):
    """Reference reduction used by the single-GPU emulation test: partial sums added in rank order."""
    total = partials[0].clone()
    for p in partials[1:]:
        total += p
    return total
