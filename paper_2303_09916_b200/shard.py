"""Host-side sharding helpers for N > 1 ranks.

The path shards by independent units (poses for scoring, copies or systems for the search) with no
exchange during the work.  These helpers hold the only multi-rank logic there is: which units a rank
owns, the MAX-over-ranks reduction of a device time, and the all-gather of each rank's k candidates
(energy + pose row) that a multi-GPU screening run re-clusters with dock_topk.  They work on any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import Tuple


def shard_range(n_units: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [begin, end) of the units rank `rank` owns; sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_units, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def max_over_ranks(x: float, device="cpu") -> float:
    """MAX of a per-rank scalar (a device time); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_candidates(energy, poses):
    """All-gather every rank's candidates: energy [k], poses [k, row] -> ([world*k], [world*k, row]) sorted by
    energy ascending, ties to the lower (rank, index) -- the order dock_topk expects.  k must be equal on all ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        order = torch.argsort(energy, stable=True)
        return energy[order], poses[order]
    world = dist.get_world_size()
    es = [torch.empty_like(energy) for _ in range(world)]
    ps = [torch.empty_like(poses) for _ in range(world)]
    dist.all_gather(es, energy.contiguous())
    dist.all_gather(ps, poses.contiguous())
    e, p = torch.cat(es), torch.cat(ps)
    order = torch.argsort(e, stable=True)
    return e[order], p[order]
