"""dock_topk_fixed: the top-k + RMSD clustering call for callers that cannot allocate device memory.

Who that is: code that was handed device pointers but no allocator (a plug-in inside someone else's engine), code
running where cudaMalloc / cudaFree are not allowed or would stall the GPU, a loop with a fixed latency budget.  Such a
caller cannot give dock_topk the workspace it asks for, so dock_topk_fixed keeps the kernel's tables in an array built
into the library (DOCK_TOPK_FIXED_BYTES per GPU) and takes inputs and outputs only.

The checks: same indices and count as dock_topk (integer outputs: bit-exact, like every index comparison in this
suite) on calls made back to back with DIFFERENT ligands and inputs, so that tables left over from the previous call
would show; the ligand too large for the array is refused up front; the driver's free-memory figure does not move.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (first call = set-up call) and after the rest of the suite."""
import ctypes as C

import numpy as np
import pytest

from dock_synth import make_system, random_poses
from tests.parity import gpu_side


def _pack():
    import paper_2303_09916_b200 as dk
    dk.load_library()
    return dk


def _big_ligand(dk, n_atoms, n_tors):
    import dock_synth
    from dock_synth.generators import LIG_TYPES_FULL
    return dk.LigandHandle(dock_synth.make_ligand(np.random.default_rng(228), n_atoms, n_tors, LIG_TYPES_FULL))


def test_ligand_beyond_the_built_in_scratch_is_refused_before_any_device_work():
    """Host-side check, needs no GPU: the size test comes before the first CUDA call."""
    from paper_2303_09916_b200 import binding as B
    dk = _pack()
    lib, p = dk.load_library(), dk.dock_default_params()
    for n_atoms, n_tors in [(128, 32), (100, 20)]:
        lig = _big_ligand(dk, n_atoms, n_tors)
        need = C.c_size_t(0)
        rc = lib.dock_topk_fixed(C.byref(p), C.byref(lig.c), 10, None, None, None, None, C.byref(need), None)
        assert rc == B.DOCK_ECAPACITY and need.value > B.DOCK_TOPK_FIXED_BYTES
        # the figure is the one dock_topk reports for its caller-allocated workspace
        need2 = C.c_size_t(0)
        assert lib.dock_topk(C.byref(p), C.byref(lig.c), 10, None, None, None, None, None, C.c_size_t(0), C.byref(need2),
                             None) == B.DOCK_EWORKSPACE
        assert need2.value == need.value
    # a ligand that fits gets past the size test and is then stopped by its null outputs, still before any device work
    lig = dk.LigandHandle(make_system(4, seed=0).ligand)
    need = C.c_size_t(0)
    assert lib.dock_topk_fixed(C.byref(p), C.byref(lig.c), 10, None, None, None, None, C.byref(need), None) == B.DOCK_EINVAL
    assert 0 < need.value <= B.DOCK_TOPK_FIXED_BYTES


@pytest.mark.gpu
def test_topk_fixed_equals_topk_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "run GPU tests on a CUDA box"
    dk = _pack()
    rng = np.random.default_rng(77)
    # three ligands of different table sizes (2.8 KB, 26 KB, 8.7 KB): every call finds another ligand's tables in the array
    cases = []
    for cfg, n in [(0, 333), (4, 1024), (2, 50), (0, 7)]:
        s = make_system(cfg, seed=0)
        p, _, _, lig = gpu_side(dk, s, build_grid=False)
        centers = rng.normal(size=(8, 3)) * 3 + s.box_center
        poses = np.stack([random_poses(rng, 1, centers[rng.integers(8)], [1.0, 1.0, 1.0], lig.T)[0] for _ in range(n)])
        e = rng.normal(size=n).round(1).astype(np.float32)            # ties on purpose
        cases.append((p, lig, torch.from_numpy(poses).cuda(), torch.from_numpy(e).cuda()))
    k = int(cases[0][0].topk)
    # the existing path first (it allocates its workspace through torch), then everything the new calls write into
    want = [tuple(t.clone() for t in dk.dock_topk(p, lig, poses, e)) for p, lig, poses, e in cases]
    outs = [(torch.full((k,), -7, dtype=torch.int32, device="cuda"), torch.full((1,), -7, dtype=torch.int32, device="cuda"))
            for _ in range(2 * len(cases))]
    torch.cuda.synchronize()
    # first call on this device = the set-up call (address look-up); from the second on nothing may move the free-memory figure
    dk.dock_topk_fixed(*cases[0], *outs[0])
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    reserved_before = torch.cuda.memory_reserved()
    launches = dk.launch_count()
    for i in range(1, len(outs)):
        dk.dock_topk_fixed(*cases[i % len(cases)], *outs[i])          # back to back on one stream, no sync in between
    torch.cuda.synchronize()
    assert dk.launch_count() - launches == len(outs) - 1
    assert torch.cuda.memory_reserved() == reserved_before
    assert torch.cuda.mem_get_info()[0] >= free_before
    for i, (idx, cnt) in enumerate(outs):
        w_idx, w_cnt = want[i % len(cases)]
        assert int(cnt[0]) == int(w_cnt[0]) and int(cnt[0]) >= 1
        assert torch.equal(idx, w_idx), (i, idx.tolist(), w_idx.tolist())
    # too large for the array: refused, outputs untouched; the same ligand goes through dock_topk
    big = _big_ligand(dk, 128, 32)
    p = cases[0][0]
    poses = torch.from_numpy(random_poses(rng, 20, make_system(0, seed=0).box_center, [1.0, 1.0, 1.0], 32)).cuda()
    e = torch.arange(20, dtype=torch.float32, device="cuda")
    idx, cnt = outs[0][0].clone(), outs[0][1].clone()
    with pytest.raises(dk.DockError, match="DOCK_ECAPACITY"):
        dk.dock_topk_fixed(p, big, poses, e, idx, cnt)
    torch.cuda.synchronize()
    assert torch.equal(idx, outs[0][0]) and torch.equal(cnt, outs[0][1])
    assert int(dk.dock_topk(p, big, poses, e)[1][0]) >= 1
