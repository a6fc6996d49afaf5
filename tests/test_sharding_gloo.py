"""The N > 1 path on CPU: world_size-2 `gloo` processes exercise the token sharding and the
max-over-ranks / whole-job reductions bench.py uses under torchrun (the layer
shards by tokens with no data-path collective)."""

import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_10493_b200 import inputs, sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = inputs.CONFIGS[0]
        # weak scaling: every rank generates its own tokens
        h = inputs.make_hidden(cfg, device="cpu", first_chunk=sharding.weak_scaling_first_chunk(cfg.T, rank))
        gathered = [torch.empty_like(h) for _ in range(world)]
        dist.all_gather(gathered, h)
        distinct = not torch.equal(gathered[0], gathered[1])
        # strong split of one prompt: ranges tile [0, T) exactly
        lo, hi = sharding.token_range(1001, rank, world)
        ranges = [None] * world
        dist.all_gather_object(ranges, (lo, hi))
        ms = 10.0 + 5.0 * rank                    # rank 1 is the slow one
        value, ms_max = sharding.whole_job_tokens_per_s(hi - lo, ms)
        q.put((rank, distinct, ranges, value, ms_max, sharding.max_over_ranks(float(rank))))
    finally:
        dist.destroy_process_group()


def test_two_rank_token_sharding_and_reductions():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, distinct, ranges, value, ms_max, mx in res:
        assert distinct
        assert ranges == [(0, 501), (501, 1001)]
        assert ms_max == 15.0 and mx == 1.0
        assert value == pytest.approx(1001 / 15e-3)


def test_token_range_properties():
    for total in (0, 1, 7, 4096, 32768, 1001):
        for world in (1, 2, 3, 8):
            r = [sharding.token_range(total, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == total
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.token_range(10, 2, 2)


def test_first_chunk_offsets_do_not_overlap():
    cfg = inputs.CONFIGS[0]
    a = inputs.make_hidden(cfg, first_chunk=sharding.weak_scaling_first_chunk(cfg.T, 0))
    b = inputs.make_hidden(cfg, first_chunk=sharding.weak_scaling_first_chunk(cfg.T, 1))
    assert torch.equal(a, inputs.make_hidden(cfg)) and not torch.equal(a, b)


# --------------------------------------------------------------------------------------------------
# SmallEP plumbing: all-gather -> local partial sums -> reduce-scatter, on CPU tensors
# --------------------------------------------------------------------------------------------------
class _FakeShardLayer:
    """Stands in for an expert-sharded SlpMoeLayer: 'expert' e multiplies the hidden row by (e + 1), every
    token uses all experts with weight 1, the 'shared expert' adds 1000 * hidden for the given token range.
    Enough to check which rank computes what, and that the reduction puts the pieces together."""

    def __init__(self, e0, e1):
        self.e0, self.e1 = e0, e1
        self.calls = []

    def prefill_partial(self, hidden_all, partial, shared_tokens=(0, 0)):
        x = hidden_all.float()
        partial.copy_(x * float(sum(e + 1 for e in range(self.e0, self.e1))))
        t0, t1 = shared_tokens
        partial[t0:t1] += 1000.0 * x[t0:t1]
        self.calls.append((tuple(hidden_all.shape), shared_tokens))
        return partial


def _smallep_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_10493_b200 import smallep
        smallep.finalize_partial = lambda s, out=None: s.to(torch.bfloat16)   # the CUDA rounding kernel is not available on CPU
        E, n, H = 7, 6, 8
        e0, e1 = smallep.expert_range(E, rank, world)
        full = torch.arange(world * n * H, dtype=torch.float32).reshape(world * n, H).div(64).bfloat16()
        layer = _FakeShardLayer(e0, e1)
        runner = smallep.SmallEpLayer(layer, None, rank, world)
        out = runner.prefill(full[rank * n:(rank + 1) * n].contiguous())
        want = (full.float() * (sum(range(1, E + 1)) + 1000.0))[rank * n:(rank + 1) * n].to(torch.bfloat16)
        q.put((rank, (e0, e1), layer.calls, torch.equal(out, want)))
    finally:
        dist.destroy_process_group()


def test_two_rank_smallep_plumbing():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_smallep_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [(0, 4), (4, 7)]                         # balanced contiguous expert ranges
    for rank, _, calls, ok in res:
        assert calls == [((12, 8), (rank * 6, rank * 6 + 6))]              # all-gathered batch, own token shard for the shared expert
        assert ok                                                          # reduce-scatter returns the complete sum of this rank's tokens


def test_bench_gpus_2_dry_run_reaches_the_reduction():
    """`python bench.py --gpus 2` outside torchrun starts two ranks itself; --dry-run swaps the GPU work for fixed
    per-rank numbers and gloo, so launch, rendezvous, max-over-ranks and the rank-0 JSON line are covered here."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    for par, scaling, tokens in (("token", "weak", 2 * 4096), ("smallep", "strong", 4096)):
        res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-run", "--parallelism", par],
                             capture_output=True, text=True, timeout=300, env=env, cwd=root)
        assert res.returncode == 0, res.stderr[-2000:]
        lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
        assert len(lines) == 1, res.stdout                                  # rank 0 alone prints
        d = json.loads(lines[0])
        assert d["n_gpus"] == 2 and d["scaling"] == scaling and d["dry_run"]
        assert d["ms_per_step"] == 110.0                                    # the slower rank (100 + 10 * rank)
        assert d["value"] == pytest.approx(tokens / 0.110)
