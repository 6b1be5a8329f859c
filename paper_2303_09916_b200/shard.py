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


def dock_search_sharded(search_fn, topk_fn, n_systems: int, copies: int, mode: str, rank: int, world: int, device=None):
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
    Pose rows: a rank's best_pose is 7 + T_max of its OWN systems wide; the gather pads every rank's rows with zeros to
    the widest, which is the unsharded run's row.  A rank that owns no unit (world > units) calls neither function and
    only takes part in the gather; `device` is where it builds its empty contribution (default: the current CUDA device
    under nccl, else the CPU).
    Kernel choice: with params.search_kernel = 0 the library picks the search kernel from the size of EACH call, so a
    shard may run the CTA kernel where the unsharded run took the warp kernel.  For BFGS the two are bit-identical; for
    Barzilai-Borwein they agree to round-off only, so pin search_kernel (1 or 2) when a BB run must reproduce across
    shardings.
    Returns a dict with best_pose [n_systems, copies, row], best_e, topk_idx, topk_e, topk_count -- the same on every rank."""
    import torch
    import torch.distributed as dist
    multi = dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if multi and dist.get_backend() == "nccl" else torch.device("cpu")

    def gather(t):
        """all-gather of per-rank tensors -> list in rank order.  The leading size may differ from rank to rank (also 0:
        `t` is None on a rank that owns no unit), and so may the trailing ones: a rank's pose rows are 7 + T_max of ITS
        systems wide.  Every rank pads with zeros to the element-wise MAX shape (the unsharded run's "unused tail 0",
        dock.h), sends that, and the leading padding is cut off again on arrival."""
        if not multi:
            return [t] if t is not None else []
        metas = [None] * world
        dist.all_gather_object(metas, None if t is None else (tuple(t.shape), str(t.dtype).split(".")[-1]))
        ref = next((m for m in metas if m is not None), None)
        if ref is None:
            raise ValueError("no rank holds any unit")
        shapes = [m[0] if m is not None else (0,) + tuple(ref[0][1:]) for m in metas]
        full = tuple(max(sh[d] for sh in shapes) for d in range(len(ref[0])))
        dev = t.device if t is not None else device
        pad = torch.zeros(full, dtype=getattr(torch, ref[1]), device=dev)
        if t is not None:
            pad[tuple(slice(0, n) for n in t.shape)] = t
        out = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(out, pad)
        return [o[: sh[0]] for o, sh in zip(out, shapes) if sh[0] > 0]

    if mode == "systems":
        b, e = shard_range(n_systems, rank, world)
        r = search_fn(b, e, 0, copies, True) if e > b else None         # world > n_systems: this rank only takes part in the gather
        keys = ("best_pose", "best_e", "topk_idx", "topk_e", "topk_count")
        cols = {k: gather(r[k].contiguous() if r is not None else None) for k in keys}
        parts = [{k: cols[k][q] for k in keys} for q in range(len(cols["best_e"]))]
        return merge_shards(mode, parts, topk_fn, n_systems)
    if mode != "copies":
        raise ValueError("mode must be 'systems' or 'copies'")
    b, e = shard_range(copies, rank, world)
    r = search_fn(0, n_systems, b, e, False) if e > b else None
    # the copy axis is the one that is split: move it to the front for the variable-length all-gather
    gp = gather(r["best_pose"].transpose(0, 1).contiguous() if r is not None else None)
    ge = gather(r["best_e"].transpose(0, 1).contiguous() if r is not None else None)
    parts = [dict(best_pose=a.transpose(0, 1), best_e=c.transpose(0, 1)) for a, c in zip(gp, ge)]
    return merge_shards(mode, parts, topk_fn, n_systems)
