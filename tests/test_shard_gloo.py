"""World-size-2 gloo test of the N > 1 host logic (shard ownership, MAX reduction, candidate gather)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2303_09916_b200.shard import dock_search_sharded, gather_candidates, max_over_ranks, merge_shards, shard_range


def test_shard_ranges_partition_the_units():
    for n in (0, 1, 7, 384, 1_048_576, 1_048_577):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [e - b for b, e in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


# ---- stand-ins for the CUDA calls (host logic only is under test here: who runs what, gather order, re-clustering) ----
_NS, _NC, _ROW, _K = 5, 37, 11, 4


def _fake_search(sb, se, cb, ce, want_topk):
    """Deterministic function of the GLOBAL (system, copy) index, like a search whose Philox streams depend on them only."""
    s_idx = torch.arange(sb, se, dtype=torch.float64)[:, None]
    c_idx = torch.arange(cb, ce, dtype=torch.float64)[None, :]
    e = torch.sin(12.9898 * s_idx + 78.233 * c_idx) * 43758.5453
    e = e - torch.floor(e)                                             # pseudo-random in [0, 1)
    pose = torch.stack([e * (k + 1) + s_idx for k in range(_ROW)], dim=-1)
    out = dict(best_pose=pose, best_e=e)
    if want_topk:
        idx, cnt = zip(*[_fake_topk(s, pose[s - sb], e[s - sb]) for s in range(sb, se)])
        out.update(topk_idx=torch.stack(idx), topk_count=torch.cat([c.reshape(1) for c in cnt]),
                   topk_e=torch.stack([e[k][i.long()] for k, i in enumerate(idx)]))
    return out


def _fake_topk(system, poses, e):
    """rank by energy (ties to the lower index), keep a pose iff its first coordinate is >= 0.05 from every kept one"""
    order = torch.argsort(e, stable=True)
    kept = []
    for i in order.tolist():
        if all(abs(float(poses[i, 0] - poses[j, 0])) >= 0.05 for j in kept):
            kept.append(i)
        if len(kept) == _K:
            break
    idx = torch.full((_K,), -1, dtype=torch.int32)
    idx[: len(kept)] = torch.tensor(kept, dtype=torch.int32)
    return idx, torch.tensor(len(kept), dtype=torch.int32)


def test_merge_of_shards_equals_the_unsharded_run():
    whole = _fake_search(0, _NS, 0, _NC, True)
    for world in (1, 2, 3):
        for mode, n_units in (("systems", _NS), ("copies", _NC)):
            parts = []
            for r in range(world):
                b, e = shard_range(n_units, r, world)
                parts.append(_fake_search(b, e, 0, _NC, True) if mode == "systems" else _fake_search(0, _NS, b, e, False))
            m = merge_shards(mode, parts, _fake_topk, _NS)
            for k in ("best_pose", "best_e", "topk_idx", "topk_e", "topk_count"):
                assert torch.equal(m[k], whole[k]), (world, mode, k)


_T = [2, 4, 3, 0, 1]                       # torsions per system: the pose rows a rank returns are 7 + max(T of ITS systems) wide


def _ragged_search(sb, se, cb, ce, want_topk):
    """_fake_search with the row convention of dock_search: 7 + T_max of the systems of THIS call, unused tail 0."""
    r = _fake_search(sb, se, cb, ce, want_topk)
    row = 7 + max(_T[sb:se])
    pose = torch.zeros(se - sb, ce - cb, row, dtype=torch.float64)
    for s in range(sb, se):
        pose[s - sb, :, : 7 + _T[s]] = r["best_pose"][s - sb, :, : 7 + _T[s]]
    r["best_pose"] = pose
    return r


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n, k, row = 1001, 5, 9
        b, e = shard_range(n, rank, world)
        rng = np.random.default_rng(7)                      # same stream on every rank: the global problem
        energy_all = torch.from_numpy(rng.normal(size=n))
        poses_all = torch.from_numpy(rng.normal(size=(n, row)))
        loc = torch.argsort(energy_all[b:e], stable=True)[:k] + b          # this rank's k best
        ge, gp = gather_candidates(energy_all[loc], poses_all[loc])
        t = max_over_ranks(1.0 + rank)
        sh = {m: dock_search_sharded(_fake_search, _fake_topk, _NS, _NC, m, rank, world) for m in ("systems", "copies")}
        sh["ragged"] = dock_search_sharded(_ragged_search, _fake_topk, _NS, _NC, "systems", rank, world)
        torch.save({"e": ge, "p": gp, "t": t, "span": (b, e), "sharded": sh}, os.path.join(out_dir, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [torch.load(os.path.join(tmp_path, f"r{i}.pt")) for i in range(world)]
    assert r[0]["t"] == r[1]["t"] == 2.0                                  # MAX over ranks
    assert torch.equal(r[0]["e"], r[1]["e"]) and torch.equal(r[0]["p"], r[1]["p"])
    # the gathered list is sorted and contains the global k best
    e = r[0]["e"]
    assert torch.all(e[1:] >= e[:-1]) and e.numel() == 2 * 5
    rng = np.random.default_rng(7)
    energy_all = np.sort(rng.normal(size=1001))
    assert np.isclose(float(e[0]), energy_all[0])
    assert r[0]["span"][1] == r[1]["span"][0]
    # NEXT-4 end to end (host logic): both ranks hold the unsharded result, whether systems or copies were split
    whole = _fake_search(0, _NS, 0, _NC, True)
    for rank in range(world):
        for mode in ("systems", "copies"):
            for k in ("best_pose", "best_e", "topk_idx", "topk_e", "topk_count"):
                assert torch.equal(r[rank]["sharded"][mode][k], whole[k]), (rank, mode, k)
    # ranks whose systems have different T_max return pose rows of different widths (7 + 4 and 7 + 1 here): the driver
    # pads them to the unsharded row instead of handing mismatched shapes to all_gather
    ragged = _ragged_search(0, _NS, 0, _NC, True)
    assert _ragged_search(0, 3, 0, _NC, True)["best_pose"].shape[-1] != _ragged_search(3, _NS, 0, _NC, True)["best_pose"].shape[-1]
    for rank in range(world):
        for k in ("best_pose", "best_e", "topk_idx", "topk_e", "topk_count"):
            assert torch.equal(r[rank]["sharded"]["ragged"][k], ragged[k]), (rank, k)


def _worker_more_ranks_than_units(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        calls = []

        def search(sb, se, cb, ce, want_topk):
            assert se > sb and ce > cb, "an empty shard must not reach the search call (dock_search rejects n_systems = 0)"
            calls.append((sb, se, cb, ce))
            return _ragged_search(sb, se, cb, ce, want_topk)

        sh = {m: dock_search_sharded(search, _fake_topk, 2, 2, m, rank, world) for m in ("systems", "copies")}
        torch.save({"sharded": sh, "calls": calls}, os.path.join(out_dir, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_more_ranks_than_units_gloo(tmp_path):
    """world 3, two systems x two copies: the third rank owns nothing in either mode, skips the search and still
    ends up with the full result."""
    world = 3
    mp.spawn(_worker_more_ranks_than_units, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [torch.load(os.path.join(tmp_path, f"r{i}.pt")) for i in range(world)]
    whole = _ragged_search(0, 2, 0, 2, True)
    assert r[2]["calls"] == [] and len(r[0]["calls"]) == len(r[1]["calls"]) == 2
    used = whole["topk_idx"] >= 0                            # two copies, k = 4: the unused slots' energies are unspecified
    for rank in range(world):
        for mode in ("systems", "copies"):
            got = r[rank]["sharded"][mode]
            for k in ("best_pose", "best_e", "topk_idx", "topk_count"):
                assert torch.equal(got[k], whole[k]), (rank, mode, k)
            assert torch.equal(got["topk_e"][used], whole["topk_e"][used]), (rank, mode)
