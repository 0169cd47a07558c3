"""Multi-GPU plumbing of the benchmark: the path shards by beam with no exchange step
(beams are split across GPUs, one host thread each), so every rank
dedisperses its own beams and the only collective is the reduction of the timings.

No arithmetic of the method lives here.
"""
from __future__ import annotations


def beams_of_rank(rank: int, world: int, beams_per_rank: int) -> list[int]:
    """Global beam ids (= input seeds) handled by `rank`: a disjoint cover of
    range(world * beams_per_rank), contiguous per rank."""
    if not (0 <= rank < world) or beams_per_rank < 1:
        raise ValueError("bad rank / world / beams_per_rank")
    return list(range(rank * beams_per_rank, (rank + 1) * beams_per_rank))


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """Max of a per-rank scalar over the process group (identity without a group)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: int, world: int, seconds_max_over_ranks: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return units_per_rank * world / seconds_max_over_ranks
