"""Host-side sharding of the path over ranks (one process per GPU).

The filter shards over vectors with no data-path collective (the paper's one-Monte-Carlo-sample-per-GPU
layout): rank r owns the global vectors [r*nvec, (r+1)*nvec), which makes the white-noise
vectors independent of the number of ranks (sgw_random_vectors takes first_vec).  The only collectives are
the timing ones bench.py needs: a barrier and a MAX over ranks of the device time.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def first_vector(rank: int, nvec_per_rank: int) -> int:
    """Global index of the first stochastic vector owned by `rank` (weak scaling: fixed work per rank)."""
    if rank < 0 or nvec_per_rank < 0:
        raise ValueError("rank and nvec_per_rank must be non-negative")
    return rank * nvec_per_rank


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a per-rank scalar (device time in ms); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, world: int, steps: int, ms_max: float) -> float:
    """Aggregate throughput over all ranks: units all ranks processed / slowest rank's time."""
    return units_per_rank * world * steps / (ms_max * 1e-3)
