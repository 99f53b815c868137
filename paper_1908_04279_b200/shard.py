"""Host-side logic of the multi-GPU path: one process per GPU, configurations partitioned over
ranks, NO data-path collective -- configurations c = (x, y, theta) never interact during substeps ("easily
parallelized over r0"; the paper splits its outer array "by rows, which are contiguous in memory",
PAPER.md:245).  The only collective is the MAX over ranks of the device-timed milliseconds that bench.py reports.
Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests); holds no method arithmetic.
"""
from __future__ import annotations

from typing import Tuple


def config_range(nc: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block [begin, end) of configurations owned by `rank` when ONE grid of nc configurations is split
    over `world` ranks (strong scaling; block sizes differ by at most one, earlier ranks take the larger blocks)."""
    if world < 1 or not (0 <= rank < world) or nc < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, nc >= 0")
    base, rem = divmod(nc, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Weak scaling: rank r runs its own copy of the workload grid -- the r-th slab of a world-times-larger periodic
    domain -- drawn from seed + r, so the ranks' inputs differ and the per-GPU work is fixed."""
    return int(seed) + int(rank)


def max_over_ranks(ms: float, device=None) -> float:
    """MAX over ranks of a device-timed duration (the bench contract).  Identity when no process group is up."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_step: float, steps: int, world: int, ms_max: float) -> float:
    """Units all ranks processed divided by the slowest rank's time (units/s)."""
    return units_per_rank_step * world * steps / (ms_max * 1e-3)
