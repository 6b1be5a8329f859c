"""World-size-2 gloo test of the N > 1 host logic (shard ownership, MAX reduction, candidate gather)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2303_09916_b200.shard import gather_candidates, max_over_ranks, shard_range


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
        torch.save({"e": ge, "p": gp, "t": t, "span": (b, e)}, os.path.join(out_dir, f"r{rank}.pt"))
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
