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


def merge_shards(mode: str, parts, topk_fn, n_systems: int):
    """Merge the per-rank results of a sharded search (rank order).  "systems": concatenate along the system axis.
    "copies": concatenate along the copy axis and re-run top-k + RMSD clustering (A8) on the complete list of copies."""
    import torch
    if mode == "systems":
        return {k: torch.cat([p[k] for p in parts], dim=0) for k in ("best_pose", "best_e", "topk_idx", "topk_e", "topk_count")}
    if mode != "copies":
        raise ValueError("mode must be 'systems' or 'copies'")
    pose = torch.cat([p["best_pose"] for p in parts], dim=1).contiguous()
    en = torch.cat([p["best_e"] for p in parts], dim=1).contiguous()
    idx, te, cnt = [], [], []
    for s in range(n_systems):
        i, c = topk_fn(s, pose[s], en[s])
        idx.append(i)
        cnt.append(c.reshape(1))
        safe = i.clamp(min=0).long()
        te.append(torch.where(i >= 0, en[s][safe], torch.zeros_like(en[s][safe])))
    return dict(best_pose=pose, best_e=en, topk_idx=torch.stack(idx), topk_e=torch.stack(te), topk_count=torch.cat(cnt))


def dock_search_sharded(search_fn, topk_fn, n_systems: int, copies: int, mode: str, rank: int, world: int):
    """NEXT-4 ("independently and asynchronously"): one many-copy search split over `world`
    ranks with NO exchange during the search and ONE all-gather at the end.

    mode "systems" (screening batches, BASELINE.json configs[3]): rank r searches systems [b, e) = shard_range(n_systems)
        with system_base = b; every system is complete on its rank (top-k included); the per-system results are
        all-gathered in system order.
    mode "copies" (one large system, configs[4]): rank r runs copies [b, e) of every system with copy_base = b and no
        top-k; the copies' best poses and energies are all-gathered in copy order and top-k + RMSD clustering (A8) is
        re-run on the complete list -- exactly the unsharded result, because the Philox streams of a copy depend on its
        global index only (dock.h: system_base / copy_base).  (Gathering only each rank's k candidates, as SURVEY.md
        8(e) sketches, is cheaper but not exact: a pose dropped on its rank for being near a better one may survive
        globally when that better one is itself dropped.  copies x (8+T) floats per system is small enough to send.)

    search_fn(sys_begin, sys_end, copy_begin, copy_end, want_topk) -> dict with best_pose [ns, nc, row], best_e [ns, nc]
        and, if want_topk, topk_idx [ns, k], topk_e [ns, k], topk_count [ns];
    topk_fn(system, poses [copies, row], e [copies]) -> (idx [k], count).
    Returns a dict with best_pose [n_systems, copies, row], best_e, topk_idx, topk_e, topk_count -- the same on every rank."""
    import torch
    import torch.distributed as dist
    multi = dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1

    def gather(t):
        """all-gather of per-rank tensors whose leading size differs by at most one -> list in rank order"""
        if not multi:
            return [t]
        n = torch.tensor([t.shape[0]], dtype=torch.int64, device=t.device)
        ns = [torch.zeros_like(n) for _ in range(world)]
        dist.all_gather(ns, n)
        m = int(max(int(x) for x in ns))
        pad = torch.zeros((m,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        pad[: t.shape[0]] = t
        out = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(out, pad)
        return [o[: int(k)] for o, k in zip(out, ns)]

    if mode == "systems":
        b, e = shard_range(n_systems, rank, world)
        r = search_fn(b, e, 0, copies, True)
        keys = ("best_pose", "best_e", "topk_idx", "topk_e", "topk_count")
        cols = {k: gather(r[k].contiguous()) for k in keys}
        parts = [{k: cols[k][q] for k in keys} for q in range(len(cols["best_e"]))]
        return merge_shards(mode, parts, topk_fn, n_systems)
    if mode != "copies":
        raise ValueError("mode must be 'systems' or 'copies'")
    b, e = shard_range(copies, rank, world)
    r = search_fn(0, n_systems, b, e, False)
    # the copy axis is the one that is split: move it to the front for the variable-length all-gather
    gp = gather(r["best_pose"].transpose(0, 1).contiguous())
    ge = gather(r["best_e"].transpose(0, 1).contiguous())
    parts = [dict(best_pose=a.transpose(0, 1), best_e=c.transpose(0, 1)) for a, c in zip(gp, ge)]
    return merge_shards(mode, parts, topk_fn, n_systems)
