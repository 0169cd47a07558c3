"""World-size-2 CPU test (gloo) of the benchmark's multi-rank plumbing: beam sharding with no
data-path collective and the max-over-ranks timing reduction."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1401_8258_b200 import sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        beams = sharding.beams_of_rank(rank, world, 3)
        gathered = [None] * world
        dist.all_gather_object(gathered, beams)
        slowest = sharding.max_over_ranks(1.0 + rank, dist)        # rank 1 is slower
        out[rank] = (gathered, slowest, sharding.whole_job_rate(10, world, slowest))
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_beams_and_reduce_the_timing():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        gathered, slowest, rate = res[rank]
        flat = [b for part in gathered for b in part]
        assert sorted(flat) == list(range(6)) and len(set(flat)) == 6      # disjoint cover
        assert gathered[rank] == sharding.beams_of_rank(rank, world, 3)
        assert slowest == 2.0                                              # max over ranks
        assert rate == 10 * 2 / 2.0


def test_single_process_is_the_identity():
    assert sharding.max_over_ranks(3.5) == 3.5
    assert sharding.beams_of_rank(0, 1, 4) == [0, 1, 2, 3]
    with pytest.raises(ValueError):
        sharding.beams_of_rank(2, 2, 1)
