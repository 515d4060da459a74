"""Multi-GPU plumbing: the path shards by coarse channel (PAPER.md L115, L141 — one coarse channel per server, the
corner turn done by the network), so ranks exchange no data.  The only communication is the max-over-ranks of the
elapsed time that bench.py reports.  Host logic only; torch.distributed supplies the process group."""
from __future__ import annotations

import torch
import torch.distributed as dist


def coarse_channels_for_rank(n_coarse: int, rank: int, world: int) -> list[int]:
    """Coarse channels owned by `rank`: round-robin, so consecutive channels land on different GPUs."""
    if not (0 <= rank < world) or n_coarse < 0:
        raise ValueError("bad rank/world/n_coarse")
    return list(range(rank, n_coarse, world))


def max_over_ranks(value: float, device: str | torch.device = "cpu") -> float:
    """MAX all-reduce of a scalar (the slowest rank defines the step time); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, world: int, seconds_max: float) -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's time."""
    return units_per_rank * world / seconds_max
