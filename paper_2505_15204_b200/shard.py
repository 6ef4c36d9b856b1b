"""Host-side sharding helpers for multi-GPU runs (no imaging arithmetic).

The path has no exchange step: images are independent, so ranks either image
independent batches (weak scaling, what bench.py does) or disjoint timestep ranges of one batch.
The only cross-rank operation is the max over ranks of the measured time.
"""
from __future__ import annotations

from typing import Optional, Tuple


def rank_seed(config: int, rank: int) -> Optional[int]:
    """Seed of the independent batch a rank images: rank 0 keeps the config's own seed."""
    return None if rank == 0 else 1000 + config + 100 * rank


def timestep_range(T: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced [t0, t1) slice of T timesteps for `rank` (first T % world ranks get one more)."""
    base, extra = divmod(T, world)
    t0 = rank * base + min(rank, extra)
    return t0, t0 + base + (1 if rank < extra else 0)


def max_over_ranks(value_ms: float, device="cpu") -> float:
    """Slowest rank's time; identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value_ms)
    t = torch.tensor([float(value_ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: int, world: int, ms_max: float) -> float:
    """Whole-job units/s when every rank processed units_per_rank in ms_max (max over ranks)."""
    return world * units_per_rank / (ms_max * 1e-3)
