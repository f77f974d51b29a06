"""Host-side sharding of a batch over ranks.

Systems are independent, so the batch is partitioned along the system axis i:
rank r owns a contiguous block of systems as its OWN interleaved (N x m_r) array and factors the
shared 5N-value matrix locally.  There is no data-path collective; the only collectives are the
barrier around the timed region and the MAX of the per-rank device times.
"""
from __future__ import annotations


def shard_columns(M_total: int, rank: int, world: int) -> tuple[int, int]:
    """(col0, m): rank `rank` of `world` owns systems [col0, col0+m) of a batch of M_total.
    Blocks are contiguous, cover 0..M_total-1 exactly once and differ in size by at most 1."""
    if world < 1 or not (0 <= rank < world) or M_total < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(M_total, world)
    col0 = rank * base + min(rank, rem)
    return col0, base + (1 if rank < rem else 0)


def max_over_ranks(seconds: float, device=None) -> float:
    """MAX over ranks of a per-rank duration (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: int, world: int, seconds_max: float) -> float:
    """Whole-job throughput under weak scaling: every rank processed `units_per_rank` units."""
    return world * units_per_rank / seconds_max
