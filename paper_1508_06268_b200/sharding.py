"""Rank sharding of the benchmark / batch drivers: independent disorder realisations per rank.

No method arithmetic lives here.  One process per GPU; rank r of W takes the realisations whose seeds are
`rank_seeds(base_seeds, r)`; there is no data-path collective, only the reduction of timings (max over ranks)
and, for drivers that want them, a gather of per-realisation observables.
"""
from typing import Sequence

import torch
import torch.distributed as dist


def rank_seeds(base_seeds: Sequence[int], rank: int):
    """Seeds of the realisations rank `rank` runs: every rank gets its own disorder, same workload shape."""
    return [int(s) + int(rank) for s in base_seeds]


def max_over_ranks(values: Sequence[float], device="cpu"):
    """Element-wise MAX of `values` over all ranks (identity when torch.distributed is not initialised)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_rate(units_per_rank: float, world: int, max_ms: float) -> float:
    """Whole-job throughput in units/ns: all ranks' units over the slowest rank's time."""
    return units_per_rank * world / (max_ms * 1e6)


def gather_by_rank(x: torch.Tensor):
    """all_gather of equally shaped per-rank observables -> list indexed by rank (list of one without a group)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [x]
    out = [torch.empty_like(x) for _ in range(dist.get_world_size())]
    dist.all_gather(out, x)
    return out
