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
