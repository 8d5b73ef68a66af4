"""Multi-GPU plumbing of the hot path: one process per GPU, views sharded across ranks.

Views are independent in `forward`, `forward_pose_grad` and `backproject_pose_grad` (Eq.18-22: every
projection / per-view 6-vector depends on its own pose only), so the path shards by views with NO data-path
collective; only the bookkeeping below (unit counts, max-over-ranks timing) crosses ranks.  A view-sharded
`backproject` yields per-rank partial volumes whose sum is the result (Eq.21 is a sum over views): that one
exchange is `allreduce_volume`.  Everything here works on any torch.distributed backend (NCCL on GPUs, gloo
in the CPU tests).
"""
from typing import Optional, Tuple

import torch


def shard_range(n_items: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced [lo, hi) slice of `n_items` for `rank`: sizes differ by at most one, the slices
    of ranks 0..world-1 tile [0, n_items) in order, and empty slices only occur when world > n_items."""
    if world <= 0 or not (0 <= rank < world) or n_items < 0:
        raise ValueError(f"bad shard request: n_items={n_items} rank={rank} world={world}")
    base, extra = divmod(n_items, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def _dist(group=None):
    import torch.distributed as dist
    return dist if (dist.is_available() and dist.is_initialized()) else None


def max_over_ranks(t: torch.Tensor, group=None) -> torch.Tensor:
    """Element-wise MAX over ranks (timings: a multi-GPU time is the slowest rank's)."""
    d = _dist()
    if d is not None and d.get_world_size(group) > 1:
        d.all_reduce(t, op=d.ReduceOp.MAX, group=group)
    return t


def sum_over_ranks(t: torch.Tensor, group=None) -> torch.Tensor:
    """Element-wise SUM over ranks (unit counts: ray-steps, voxel-views)."""
    d = _dist()
    if d is not None and d.get_world_size(group) > 1:
        d.all_reduce(t, op=d.ReduceOp.SUM, group=group)
    return t


def allreduce_volume(partial: torch.Tensor, group=None) -> torch.Tensor:
    """Sum of the per-rank partial back-projections of a view-sharded `backproject` (in place)."""
    return sum_over_ranks(partial, group)


def gather_view_results(local: torch.Tensor, n_total: int, group=None) -> Optional[torch.Tensor]:
    """All-gather per-view results ([n_local, ...] on each rank, sharded by `shard_range`) into
    [n_total, ...] in view order, on every rank."""
    d = _dist()
    if d is None or d.get_world_size(group) == 1:
        assert local.shape[0] == n_total
        return local
    world = d.get_world_size(group)
    sizes = [shard_range(n_total, r, world) for r in range(world)]
    biggest = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros((biggest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[:local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    d.all_gather(parts, pad, group=group)
    return torch.cat([p[:hi - lo] for p, (lo, hi) in zip(parts, sizes)], dim=0)


def job_throughput(units_local: float, seconds_local: float, group=None, device="cpu") -> Tuple[float, float, float]:
    """Whole-job rate = (units summed over ranks) / (seconds, max over ranks).  Returns (rate, units, seconds)."""
    u = sum_over_ranks(torch.tensor([float(units_local)], dtype=torch.float64, device=device), group)
    s = max_over_ranks(torch.tensor([float(seconds_local)], dtype=torch.float64, device=device), group)
    return float(u[0]) / float(s[0]), float(u[0]), float(s[0])
