"""The N > 1 host logic (replicas / independent-problem sharding, max-over-ranks timing) on CPU with the
gloo backend, world_size 2 (the graded path runs on one GPU)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2309_04623_b200 import sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_problems, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = sharding.shard_problems(n_problems, rank, world)
    gathered = [None] * world
    dist.all_gather_object(gathered, mine)
    t = 1.0 + rank                      # rank 1 is the slow one
    tmax = sharding.max_over_ranks(t)
    rate = sharding.aggregate_rate(10.0, t)
    q.put((rank, mine, gathered, tmax, rate, sharding.replica_seed(3003, rank)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n_problems", [64, 7, 1])
def test_two_ranks_partition_and_max_time(n_problems):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_problems, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    owned = [i for _, mine, _, _, _, _ in out for i in mine]
    assert sorted(owned) == list(range(n_problems))              # every problem exactly once
    assert abs(len(out[0][1]) - len(out[1][1])) <= 1             # balanced
    for rank, mine, gathered, tmax, rate, seed in out:
        assert gathered[rank] == mine and gathered[0] == out[0][1]
        assert tmax == 2.0                                       # max over ranks, not this rank's time
        assert rate == pytest.approx(2 * 10.0 / 2.0)             # units of all ranks / slowest rank
    assert out[0][5] == 3003 and out[1][5] != out[0][5]


def test_single_process_identity_and_errors():
    assert sharding.max_over_ranks(3.5) == 3.5
    assert sharding.aggregate_rate(5.0, 2.0) == 2.5
    assert sharding.shard_problems(5, 0, 1) == [0, 1, 2, 3, 4]
    with pytest.raises(ValueError):
        sharding.shard_problems(4, 2, 2)
