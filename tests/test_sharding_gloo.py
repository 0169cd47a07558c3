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


def _bench_rank(out):
    # what bench.run_ours does around its timed region, with a stubbed step time: process group from the
    # environment bench.launch_ranks set, max-over-ranks reduction, whole-job rate
    import bench
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    assert os.environ["MASTER_ADDR"] == "127.0.0.1" and int(os.environ["LOCAL_RANK"]) == rank
    dist.init_process_group("gloo")
    try:
        total_ms = 100.0 * (1 + rank)                                   # rank 1 took twice as long
        out[rank] = bench.finish_timing(total_ms, 10, 1000, world, dist, None)
    finally:
        dist.destroy_process_group()


def test_bench_launches_its_own_ranks_and_reduces_over_them():
    # `python bench.py --gpus 2` without torchrun goes through bench.launch_ranks
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    import bench
    with mp.Manager() as m:
        out = m.dict()
        bench.launch_ranks(2, _bench_rank, (out,))
        res = dict(out)
    assert sorted(res) == [0, 1]
    for rank in (0, 1):
        ms_per_step, value = res[rank]
        assert ms_per_step == 20.0                                          # slowest rank: 200 ms / 10 steps
        assert value == 1000 * 2 / 0.020 / 1e9                              # both ranks' units over that time


def test_single_process_is_the_identity():
    assert sharding.max_over_ranks(3.5) == 3.5
    assert sharding.beams_of_rank(0, 1, 4) == [0, 1, 2, 3]
    with pytest.raises(ValueError):
        sharding.beams_of_rank(2, 2, 1)
