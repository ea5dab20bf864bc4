"""N > 1 path on CPU: world_size-2 gloo processes exercise the head sharding and the max-over-ranks timing reduction that
bench.py uses under torchrun (heads shard, no collective inside the operator)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_03012_b200 import sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        heads = sharding.shard_heads(24, rank, world)
        ms = sharding.max_over_ranks(10.0 + 5.0 * rank)          # rank 1 is the slow one
        gathered = [None] * world
        dist.all_gather_object(gathered, heads)
        q.put((rank, heads, ms, gathered))
    finally:
        dist.destroy_process_group()


def test_head_sharding_and_timing_reduction_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, heads, ms, gathered in out:
        assert ms == 15.0                                         # max over ranks on every rank
        assert heads == gathered[rank] == list(range(rank, 24, world))
    all_heads = sorted(h for _, heads, _, _ in out for h in heads)
    assert all_heads == list(range(24))                           # a partition: every head exactly once
    assert sharding.whole_job_value(15.0, world) == 7.5


def test_shard_heads_uneven_and_single():
    assert sharding.shard_heads(24, 0, 1) == list(range(24))
    parts = [sharding.shard_heads(10, r, 4) for r in range(4)]
    assert sorted(sum(parts, [])) == list(range(10)) and max(map(len, parts)) - min(map(len, parts)) <= 1
    assert sharding.max_over_ranks(3.5) == 3.5                    # no process group: identity
