"""Host-side logic of the multi-GPU path: points are independent
(PAPER.md:83), so ranks own disjoint batches or slabs and the data path has no collective.
The only communication is the reduction of the step time (max over ranks).  No arithmetic of
the method lives here."""
from __future__ import annotations

import torch
import torch.distributed as dist


def rank_state_seed(cfg: int, rank: int) -> int:
    """Weak scaling: every rank draws its own full-size batch of states."""
    return 2000 + cfg + 100 * rank


def rank_slab(n_total: int, rank: int, world: int, align: int = 32):
    """Strong sharding of one field of n_total points: contiguous slabs, multiples of `align`
    points (a warp's chunk) except the last.  Returns (first, count)."""
    chunks = (n_total + align - 1) // align
    lo = (chunks * rank) // world * align
    hi = (chunks * (rank + 1)) // world * align
    lo, hi = min(lo, n_total), min(hi, n_total)
    return lo, hi - lo


def max_over_ranks(value: float, device=None) -> float:
    """A time-like number reduced with MAX over the process group (identity without one)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(points_per_rank: int, world: int, step_ms_max: float) -> float:
    """Whole-job points/s: the units all ranks processed over the slowest rank's time."""
    return world * points_per_rank / (step_ms_max * 1e-3)
