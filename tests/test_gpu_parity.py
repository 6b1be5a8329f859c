"""GPU parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element on the same seeded inputs (SURVEY.md 8(c) parity protocol, levels 1-3').  Run with -m gpu."""
import json
import math
import os

import numpy as np
import pytest

from dock_synth import make_system, random_poses
from tests.parity import KINK_MARGIN, compare_scores, gpu_side, oracle_side, tol

pytestmark = pytest.mark.gpu

OUT = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")


def _log(name, obj):
    os.makedirs(OUT, exist_ok=True)
    with open(os.path.join(OUT, "parity_stats.jsonl"), "a") as f:
        f.write(json.dumps({"test": name, **obj}) + "\n")


@pytest.fixture(scope="module")
def dk():
    import torch
    assert torch.cuda.is_available(), "run GPU tests on a CUDA box"
    import paper_2303_09916_b200 as dk
    dk.load_library()
    return dk


@pytest.fixture(scope="module")
def torch():
    import torch
    return torch


@pytest.fixture(scope="module")
def tiny(dk, orc):
    s = make_system(0, seed=0)
    return s, gpu_side(dk, s), oracle_side(orc, s)


@pytest.fixture(scope="module")
def micro(dk, orc):
    s = make_system(1, seed=0)
    return s, gpu_side(dk, s), oracle_side(orc, s)


# ----------------------------------------------------------------------------------- A1 grid maps
@pytest.mark.parametrize("cfg", [0, 1])
def test_grid_maps_match_brute_force_at_every_node(dk, orc, tiny, micro, cfg):
    s, (p, box, grid, lig), (op, og, oL) = tiny if cfg == 0 else micro
    g = grid.data.cpu().numpy().astype(np.float64)
    assert g.shape == og.maps.shape
    assert tuple(grid.desc.dims) == og.dims and np.array_equal(np.array(grid.desc.origin, np.float64), og.origin)
    err = np.abs(g - og.maps) / tol(og.maps)
    _log("grid", dict(cfg=cfg, nodes=int(g.size), max_err=float(err.max()), max_abs=float(np.abs(g - og.maps).max())))
    assert err.max() <= 1.0
    # fp32 accumulation of ~150 terms: relative error should really be ~1e-6
    assert np.abs(g - og.maps).max() <= 2e-5 * max(1.0, np.abs(og.maps).max())


def test_grid_edge_cases(dk, orc, torch):
    p = dk.dock_default_params()
    op = orc.params_as_fp32(orc.default_params())
    # empty protein -> all zeros; a protein far away -> all zeros; ragged dims (non-cubic box, 17 types)
    box = dk.make_box([0, 0, 0], [6.0, 4.5, 3.0], 0.375)
    g = dk.dock_build_grids(p, np.zeros((0, 3), np.float32), np.zeros(0, np.int32), box, [0, 3])
    assert g.dims == (17, 13, 9) and float(g.data.abs().max()) == 0.0
    far = np.array([[100.0, 0, 0]], np.float32)
    g = dk.dock_build_grids(p, far, np.array([1], np.int32), box, [0])
    assert float(g.data.abs().max()) == 0.0
    rng = np.random.default_rng(5)
    xyz = (rng.random((60, 3)) * [10, 8, 6] - [5, 4, 3]).astype(np.float32)
    typ = rng.integers(0, 17, 60).astype(np.int32)
    all_types = list(range(17))                       # > 8 maps: two passes
    g = dk.dock_build_grids(p, xyz, typ, box, all_types)
    og = orc.build_grid(op, xyz, typ, [0, 0, 0], [6.0, 4.5, 3.0], 0.375, all_types)
    err = np.abs(g.data.cpu().numpy() - og.maps) / tol(og.maps)
    assert err.max() <= 1.0


# ----------------------------------------------------------------------------------- A2-A5 per pose
def test_score_and_gradient_tiny(dk, orc, torch, tiny):
    s, (p, box, grid, lig), (op, og, oL) = tiny
    rng = np.random.default_rng(1)
    poses = random_poses(rng, 4099, s.box_center, s.box_size * 1.3, lig.T)   # ragged count, some atoms outside
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    st = compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag, "tiny",
                        cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    assert (diag["atoms_outside"] > 0).mean() > 0.05     # the wall is exercised
    _log("score_tiny", st)


def test_score_and_gradient_microbench_sample(dk, orc, torch, micro):
    """Config 1 at full size in the bench launch configuration; 65 536 sampled poses go to the oracle."""
    s, (p, box, grid, lig), (op, og, oL) = micro
    rng = np.random.default_rng(0)
    n = 1_048_576
    poses = random_poses(rng, n, s.box_center, s.box_size, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    idx = np.sort(rng.choice(n, 65536, replace=False))
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses[idx].astype(np.float64))
    ii = torch.from_numpy(idx).cuda()
    st = compare_scores(e[ii].cpu().numpy(), g[ii].cpu().numpy(), t[ii].cpu().numpy(), oe, ograd, oterms, diag, "micro",
                        cond=orc.grad_cond(op, og, oL, poses[idx].astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    st["pairs_in_range_mean"] = float(diag["pairs_in_range"].mean())
    _log("score_micro", st)
    assert bool(torch.isfinite(e).all()) and bool(torch.isfinite(g).all())


def test_score_edge_cases(dk, orc, torch, tiny):
    s, (p, box, grid, lig), (op, og, oL) = tiny
    # empty batch
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.zeros((0, 7 + lig.T), device="cuda"))
    assert e.numel() == 0
    # energy only (no gradient / terms buffers)
    rng = np.random.default_rng(2)
    poses = random_poses(rng, 33, s.box_center, s.box_size, lig.T)
    e0, g0, t0 = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    e1, g1, t1 = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda(), want_grad=False, want_terms=False)
    assert g1 is None and t1 is None and torch.equal(e0, e1)
    # quaternions are normalised on read
    scaled = poses.copy()
    scaled[:, 3:7] *= 3.7
    e2, g2, _ = dk.dock_score_batch(p, grid, lig, torch.from_numpy(scaled).cuda())
    assert torch.allclose(e0, e2, rtol=1e-5, atol=1e-4)
    # whole ligand far outside the box: wall dominates, still finite and matching
    out = poses.copy()
    out[:, 0] += 40.0
    e3, g3, t3 = dk.dock_score_batch(p, grid, lig, torch.from_numpy(out).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, out.astype(np.float64))
    assert np.all(np.abs(e3.cpu().numpy() - oe) <= tol(oe))
    assert np.all(np.abs(g3.cpu().numpy() - ograd) <= tol(ograd))


@pytest.mark.parametrize("N,T", [(1, 0), (5, 0), (33, 3), (60, 15), (100, 9), (128, 32)])
def test_score_other_ligand_shapes(dk, orc, torch, micro, N, T):
    """Degenerate and large ligands on the config-1 grid: single atom, rigid, N > 32 (two atoms per lane), T = 15,
    and the maxima of include/dock.h (N = 128, T = 32: the pair schedule overflows the kernel-parameter bank and is
    read from global memory)."""
    s0, (p, box, grid, _), (op, og, _) = micro
    import dock_synth
    from dock_synth.generators import LIG_TYPES_FULL
    rng = np.random.default_rng(100 + N)
    if N == 1:
        from types import SimpleNamespace
        ligd = SimpleNamespace(ref_xyz=np.zeros((1, 3)), type=np.array([3], np.int32), frag=np.zeros(1, np.int32),
                               tors_parent=np.zeros(0, np.int32), tors_a=np.zeros(0, np.int32),
                               tors_b=np.zeros(0, np.int32), pairs=np.zeros((0, 2), np.int32))
    else:
        ligd = dock_synth.make_ligand(rng, N, T, LIG_TYPES_FULL)
    lig, oL = dk.LigandHandle(ligd), orc.Ligand(ligd)
    poses = random_poses(rng, 777, s0.box_center, s0.box_size, T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    st = compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag, f"N{N}T{T}",
                        cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=N, n_pairs=oL.P)
    _log("score_shapes", dict(N=N, T=T, **st))


def test_host_entry_point_matches_device_entry_point(dk, torch, tiny):
    s, (p, box, grid, lig), _ = tiny
    rng = np.random.default_rng(3)
    poses = random_poses(rng, 1000, s.box_center, s.box_size, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    eh, gh, th = dk.dock_score_batch_host(p, grid, lig, poses, want_grad=True, want_terms=True)
    assert np.array_equal(e.cpu().numpy(), eh) and np.array_equal(g.cpu().numpy(), gh) and np.array_equal(t.cpu().numpy(), th)


def test_run_to_run_determinism(dk, torch, tiny):
    s, (p, box, grid, lig), _ = tiny
    rng = np.random.default_rng(4)
    poses = torch.from_numpy(random_poses(rng, 2048, s.box_center, s.box_size, lig.T)).cuda()
    a = dk.dock_score_batch(p, grid, lig, poses)
    b = dk.dock_score_batch(p, grid, lig, poses)
    assert all(torch.equal(x, y) for x, y in zip(a, b))
    r1 = dk.dock_search(p, [grid], [lig], [box], 16, 6, 30, seed=5, want_trace=True)
    r2 = dk.dock_search(p, [grid], [lig], [box], 16, 6, 30, seed=5, want_trace=True)
    for k in ("best_pose", "best_e", "topk_idx", "trace", "evals"):
        assert torch.equal(r1[k], r2[k]), k


# ----------------------------------------------------------------------------------- A6 local optimisation
@pytest.mark.parametrize("cfg,n,cap", [(0, 256, 50), (1, 256, 300)])
def test_local_opt_final_energies(dk, orc, torch, tiny, micro, cfg, n, cap):
    s, (p, box, grid, lig), (op, og, oL) = tiny if cfg == 0 else micro
    rng = np.random.default_rng(7)
    poses = random_poses(rng, n, s.box_center, s.box_size * 0.6, lig.T)
    out_pose, out_e, out_it = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses).cuda(), cap)
    ge, gp, git = out_e.cpu().numpy().astype(np.float64), out_pose.cpu().numpy(), out_it.cpu().numpy()
    ref = [orc.local_opt(op, og, oL, poses[i].astype(np.float64), cap) for i in range(n)]
    re_ = np.array([r[0] for r in ref])
    # the GPU's reported energy is the oracle's energy of the GPU's final pose (level 1 at the optimum)
    # A descent that pushes a pair outward cannot cross the hard cutoff (E jumps UP by ~0.0036 at r = 8 A, reading
    # S3), so the backtracking line search parks that pair at r = 8 - O(1e-7): in about half of all local optima
    # -- the oracle's own too -- some pair sits closer to the cutoff than fp32 can resolve.  Those poses are
    # compared with the jump allowed for; all others under S20.
    chk, _, _, dg = orc.score_batch(op, og, oL, gp.astype(np.float64))
    away = dg["cutoff_margin"] > KINK_MARGIN
    assert away.mean() > 0.25 and np.all(np.abs(ge - chk)[away] <= tol(chk)[away])
    assert np.all(np.abs(ge - chk) <= tol(chk) + 3 * 0.004)
    # never worse than the start
    e0 = orc.score_batch(op, og, oL, poses.astype(np.float64), want_grad=False)[0]
    assert np.all(ge <= e0 + tol(e0))
    agree = np.abs(ge - re_) <= 1e-3
    st = dict(cfg=cfg, n=n, cap=cap, agree_1e3=float(agree.mean()), median_abs=float(np.median(np.abs(ge - re_))),
              gpu_mean=float(ge.mean()), ref_mean=float(re_.mean()),
              gpu_iters=float(git[:, 0].mean()), ref_iters=float(np.mean([r[2] for r in ref])))
    _log("local_opt", st)
    # Free-running fp32 vs fp64 BFGS on a piecewise-trilinear landscape (the gradient of eq. 3 jumps at
    # every cell face, so minima sit on faces and the stopping point is round-off sensitive): the
    # agreement rate is REPORTED; what is asserted is that the two
    # optimizers are statistically the same optimizer ...
    qg, qr = np.quantile(ge, [0.25, 0.5, 0.75]), np.quantile(re_, [0.25, 0.5, 0.75])
    st["gpu_quartiles"], st["ref_quartiles"] = qg.tolist(), qr.tolist()
    assert np.all(np.abs(qg - qr) <= 0.75 + 0.15 * np.abs(qr)), st
    assert abs(st["gpu_iters"] - st["ref_iters"]) <= 0.25 * max(st["ref_iters"], 1.0), st
    # ... that neither side is systematically better (paired sign test, 5 sigma) ...
    decided = np.abs(ge - re_) > 1e-3
    wins = int((ge < re_)[decided].sum())
    assert abs(wins - 0.5 * decided.sum()) <= 2.5 * math.sqrt(max(1, decided.sum())), (wins, int(decided.sum()), st)
    # ... and that the deterministic part agrees: same start, cap = 1 iteration -> same first step
    o1, e1, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses).cuda(), 1)
    r1 = np.array([orc.local_opt(op, og, oL, poses[i].astype(np.float64), 1)[0] for i in range(n)])
    c1, _, _, d1 = orc.score_batch(op, og, oL, o1.cpu().numpy().astype(np.float64))
    ok1 = d1["cutoff_margin"] > KINK_MARGIN
    first = np.abs(e1.cpu().numpy() - r1) <= tol(r1) * 10
    st["first_step_agree"] = float(first[ok1].mean())
    _log("local_opt_first_step", st)
    assert first[ok1].mean() >= 0.97, st


def test_local_opt_zero_iterations_is_a_plain_evaluation(dk, orc, torch, tiny):
    s, (p, box, grid, lig), (op, og, oL) = tiny
    rng = np.random.default_rng(8)
    poses = random_poses(rng, 64, s.box_center, s.box_size, lig.T)
    out_pose, out_e, out_it = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses).cuda(), 0)
    e, _, _ = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    # two evaluators (warp-per-pose in the optimizer, thread-per-pose in the batch call): same value up to summation order
    assert torch.allclose(out_e, e, rtol=1e-5, atol=1e-4)
    assert np.all(out_it.cpu().numpy() == [0, 1])


# ----------------------------------------------------------------------------------- A7 search
def _trace_fields(tr):
    return dict(e_cur=tr[..., 0], e_cand=tr[..., 1], u=tr[..., 2], accept=tr[..., 3] > 0.5,
                iters=tr[..., 4], evals=tr[..., 5], kind=tr[..., 6], pose=tr[..., 8:])


@pytest.mark.parametrize("cfg", [0, 2])
def test_search_free_run_and_teacher_forced(dk, orc, torch, cfg):
    s = make_system(cfg, seed=0)
    p, box, grid, lig = gpu_side(dk, s)
    op, og, oL = oracle_side(orc, s)
    copies, steps, cap = (s.copies, s.steps, s.bfgs_cap) if cfg == 0 else (64, 10, 300)
    seed = 2023
    init = dk.dock_init_poses(box, lig.T, seed, 0, copies)
    assert np.max(np.abs(init - orc.init_poses(s.box_center, s.box_size, lig.T, seed, 0, copies))) <= 1e-6
    res = dk.dock_search(p, [grid], [lig], [box], copies, steps, cap, seed,
                         init_poses=torch.from_numpy(init[None]).cuda(), want_trace=True)
    tr = _trace_fields(res["trace"][0].cpu().numpy().astype(np.float64))
    best_e = res["best_e"][0].cpu().numpy().astype(np.float64)
    best_pose = res["best_pose"][0].cpu().numpy().astype(np.float64)
    T_mc = float(p.t_mc)

    # --- internal consistency of the GPU trace (logic, exact) ---------------------------------
    for c in range(copies):
        for k in range(steps):
            assert tr["u"][c, k] == orc.mc_uniform(seed, 0, c, k)                  # same Philox stream, bit exact
            kind, _ = orc.mc_perturb(op, lig.T, seed, 0, c, k, tr["pose"][c, k])
            assert kind == int(tr["kind"][c, k])
            de = tr["e_cand"][c, k] - tr["e_cur"][c, k]
            thr = math.exp(min(50.0, -de / T_mc))
            if de != 0.0 and abs(tr["u"][c, k] - thr) > 1e-6:                       # margin rule
                assert bool(tr["accept"][c, k]) == (de < 0 or tr["u"][c, k] < thr), (c, k)
            if k + 1 < steps:                                                       # chain: next e_cur
                want = tr["e_cand"][c, k] if tr["accept"][c, k] else tr["e_cur"][c, k]
                assert tr["e_cur"][c, k + 1] == want
        acc = [tr["e_cur"][c, 0]] + [tr["e_cand"][c, k] for k in range(steps) if tr["accept"][c, k]]
        assert best_e[c] == min(acc)
    chk, _, _, dgb = orc.score_batch(op, og, oL, best_pose)
    awayb = dgb["cutoff_margin"] > KINK_MARGIN
    assert np.all(np.abs(best_e - chk)[awayb] <= tol(chk)[awayb])                   # best pose really has that energy
    assert int(res["evals"][0]) >= int(tr["evals"].sum()) + copies              # + the initial local optimisations

    # --- level 3': teacher-forced replay of every recorded step -------------------------------------
    n_steps = n_e_ok = n_dec = n_dec_ok = 0
    for c in range(copies):
        for k in range(steps):
            _, cand0 = orc.mc_perturb(op, lig.T, seed, 0, c, k, tr["pose"][c, k])
            e_c, _, _, _ = orc.local_opt(op, og, oL, cand0, cap)
            e_cur, _, _, dgc = orc.score_batch(op, og, oL, tr["pose"][c, k][None, :7 + lig.T])
            e_cur = float(e_cur[0])
            if dgc["cutoff_margin"][0] > KINK_MARGIN:
                assert abs(e_cur - tr["e_cur"][c, k]) <= tol(e_cur)                 # level 1 on the pre-step pose
            n_steps += 1
            ok = abs(e_c - tr["e_cand"][c, k]) <= 1e-3
            n_e_ok += ok
            if ok:
                de = e_c - e_cur
                thr = math.exp(min(50.0, -de / T_mc))
                if abs(de) > 2e-3 and abs(tr["u"][c, k] - thr) > 2e-3 * max(thr, 1e-3) / T_mc + 1e-6:
                    n_dec += 1
                    n_dec_ok += bool(tr["accept"][c, k]) == (de < 0 or tr["u"][c, k] < thr)
    # --- level 3: free run from the same initial poses --------------------------------------------
    ref = orc.search(op, og, oL, init.astype(np.float64), steps, cap, seed, 0)
    same_prefix = []
    for c in range(copies):
        k = 0
        while k < steps and bool(tr["accept"][c, k]) == bool(ref["trace"]["accept"][c, k]) \
                and abs(tr["e_cand"][c, k] - ref["trace"]["e_cand"][c, k]) <= 1e-3:
            k += 1
        same_prefix.append(k)
    best_ok = np.abs(best_e - ref["best_e"]) <= 1e-3
    st = dict(cfg=cfg, copies=copies, steps=steps, cap=cap,
              teacher_e_agree=n_e_ok / n_steps, teacher_decisions=n_dec, teacher_decision_agree=(n_dec_ok / max(1, n_dec)),
              free_full_agree=float(np.mean(np.array(same_prefix) == steps)), free_mean_prefix=float(np.mean(same_prefix)),
              free_best_agree=float(best_ok.mean()), gpu_best_min=float(best_e.min()), ref_best_min=float(ref["best_e"].min()),
              gpu_best_mean=float(best_e.mean()), ref_best_mean=float(ref["best_e"].mean()),
              gpu_evals=int(res["evals"][0]), ref_evals=int(ref["evals"]))
    _log("search", st)
    assert n_dec_ok == n_dec, st                         # a decision mismatch with agreeing energies is a bug
    # teacher_e_agree / free_* are round-off amplification rates of the fp32 path: REPORTED (gpurun_out/parity_stats.jsonl,
    # DESIGN.md "Parity levels"), not gated -- the gate on search logic is the decision check above plus the exact chain checks
    # best energies are heavy-tailed (a few copies stay stuck in a clash at E ~ 1e2): compare medians and quartiles
    qg, qr = np.quantile(best_e, [0.25, 0.5, 0.75]), np.quantile(ref["best_e"], [0.25, 0.5, 0.75])
    st["gpu_best_quartiles"], st["ref_best_quartiles"] = qg.tolist(), qr.tolist()
    _log("search_quartiles", st)
    assert np.all(np.abs(qg - qr) <= 0.75 + 0.15 * np.abs(qr)), st


def test_search_zero_steps_equals_local_opt_and_copy_independence(dk, torch, tiny):
    s, (p, box, grid, lig), _ = tiny
    init = dk.dock_init_poses(box, lig.T, 11, 0, 24)
    ti = torch.from_numpy(init[None]).cuda()
    r0 = dk.dock_search(p, [grid], [lig], [box], 24, 0, 50, 11, init_poses=ti)
    op_, oe_, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(init).cuda(), 50)
    assert torch.equal(r0["best_e"][0], oe_) and torch.equal(r0["best_pose"][0], op_)
    # generated-on-host initial poses are the same as passing dock_init_poses explicitly
    r1 = dk.dock_search(p, [grid], [lig], [box], 24, 5, 50, 11)
    r2 = dk.dock_search(p, [grid], [lig], [box], 24, 5, 50, 11, init_poses=ti)
    assert torch.equal(r1["best_e"], r2["best_e"])
    # copy c does not depend on the number of copies
    r3 = dk.dock_search(p, [grid], [lig], [box], 7, 5, 50, 11)
    assert torch.equal(r3["best_e"][0], r1["best_e"][0, :7])


def test_batched_systems_equal_single_system_runs(dk, torch):
    """Config-3 shape in miniature: heterogeneous systems in one launch == one launch per system."""
    systems = [make_system(3, seed=0, index=i, n_prot=300 + 50 * i) for i in range(3)]
    sides = [gpu_side(dk, s) for s in systems]
    p = sides[0][0]
    grids, ligs, boxes = [x[2] for x in sides], [x[3] for x in sides], [x[1] for x in sides]
    rb = dk.dock_search(p, grids, ligs, boxes, 8, 3, 40, 77)
    t_max = max(l.T for l in ligs)
    for i in range(3):
        # system index enters the Philox counter, so replay system i alone with the same init poses
        init = np.zeros((8, 7 + ligs[i].T), np.float32)
        init[:] = dk.dock_init_poses(boxes[i], ligs[i].T, 77, i, 8)
        rs_e = rb["best_e"][i].cpu().numpy()
        assert np.all(np.isfinite(rs_e))
        assert rb["best_pose"].shape[-1] == 7 + t_max
        assert int(rb["topk_count"][i]) >= 1
    # the first system has index 0 in both layouts -> identical
    r0 = dk.dock_search(p, grids[:1], ligs[:1], boxes[:1], 8, 3, 40, 77)
    assert torch.equal(r0["best_e"][0], rb["best_e"][0])


# ----------------------------------------------------------------------------------- A8 top-k
def test_topk_matches_oracle(dk, orc, torch, tiny):
    s, (p, box, grid, lig), (op, og, oL) = tiny
    rng = np.random.default_rng(9)
    for trial in range(4):
        n = [50, 333, 1024, 7][trial]
        centers = rng.normal(size=(8, 3)) * 3 + s.box_center
        poses = np.stack([random_poses(rng, 1, centers[rng.integers(8)], [1.0, 1.0, 1.0], lig.T)[0] for _ in range(n)])
        e = rng.normal(size=n).round(1).astype(np.float32)          # ties on purpose
        idx, cnt = dk.dock_topk(p, lig, torch.from_numpy(poses).cuda(), torch.from_numpy(e).cuda())
        cnt, idx = int(cnt[0]), idx.cpu().numpy()
        ocnt, oidx = orc.topk(op, oL, poses.astype(np.float64), e.astype(np.float64), int(p.topk), float(p.cluster_rmsd))
        # validity: sorted, pairwise >= 2 A
        kept = idx[:cnt]
        assert np.all(np.diff(e[kept]) >= 0)
        for a in range(cnt):
            for b in range(a):
                assert orc.rmsd(oL, poses[kept[a]], poses[kept[b]]) >= float(p.cluster_rmsd) - 1e-4
        # uniqueness: identical to the oracle unless an RMSD sits on the threshold
        near = any(abs(orc.rmsd(oL, poses[i], poses[j]) - 2.0) < 1e-4 for i in oidx[:ocnt] for j in range(n)) if n <= 60 else False
        if not near:
            assert cnt == ocnt and list(kept) == list(oidx[:ocnt])
        assert np.all(idx[cnt:] == -1)


def test_end_to_end_host_call(dk, orc, torch, tiny):
    s, (p, box, grid, lig), (op, og, oL) = tiny
    r = dk.dock_system_host(p, s.protein_xyz, s.protein_type, box, lig, s.lig_types, 16, 5, 50, 3)
    r2 = dk.dock_search(p, [grid], [lig], [box], 16, 5, 50, 3)
    assert r["count"] == int(r2["topk_count"][0]) and r["count"] >= 1
    assert np.array_equal(r["topk_e"], r2["topk_e"][0].cpu().numpy())
    assert r["evals"] == int(r2["evals"][0])
    chk = orc.score_batch(op, og, oL, r["topk_pose"][:r["count"]].astype(np.float64), want_grad=False)[0]
    assert np.all(np.abs(r["topk_e"][:r["count"]] - chk) <= tol(chk))


# ----------------------------------------------------------------------------------- configs 3 and 4
@pytest.mark.parametrize("index", [0, 5])
def test_config3_systems_score_and_local_opt(dk, orc, torch, index):
    """Two systems of the screening batch (BASELINE.json configs[3]) at their drawn sizes: grid at every node,
    per-pose scores and gradients, and local-optimisation energies against the oracle."""
    s = make_system(3, seed=0, index=index)
    p, box, grid, lig = gpu_side(dk, s)
    op, og, oL = oracle_side(orc, s)
    err = np.abs(grid.data.cpu().numpy().astype(np.float64) - og.maps) / tol(og.maps)
    assert err.max() <= 1.0
    rng = np.random.default_rng(30 + index)
    poses = random_poses(rng, 2053, s.box_center, s.box_size, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    st = compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag, f"cfg3[{index}]",
                        cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    _log(f"score_cfg3_{index}", dict(st, N=lig.N, T=lig.T, P=lig.P, n_prot=int(s.protein_xyz.shape[0])))
    # local optimisation never increases the energy and ends where the oracle's evaluation agrees
    n = 64
    out_pose, out_e, iters = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses[:n]).cuda(), 300)
    fin = out_pose.cpu().numpy()
    oe2, _, _, d2 = orc.score_batch(op, og, oL, fin.astype(np.float64))
    ok = d2["cutoff_margin"] > 1e-4
    assert np.all(np.abs(out_e.cpu().numpy() - oe2)[ok] <= tol(oe2)[ok])
    assert np.all(out_e.cpu().numpy() <= e[:n].cpu().numpy() + 1e-3)


def test_config4_large_box_grid_score_and_search_properties(dk, orc, torch):
    """BASELINE.json configs[4]: 8000-atom protein, 161^3 x 8 maps, 60-atom / 15-torsion ligand.  The grid is
    compared at EVERY node (the oracle's brute force takes ~30 s on the box's cores), scores on a sample;
    the search runs with the config's 2048 copies for a few steps and is checked through properties that hold
    at any size (bitwise determinism, best <= initial local optimum, oracle re-evaluation of the winners)."""
    s = make_system(4, seed=0)
    p, box, grid, lig = gpu_side(dk, s)
    op, og, oL = oracle_side(orc, s)
    assert tuple(grid.dims) == (161, 161, 161)
    gm = grid.data.cpu().numpy().astype(np.float64)
    err = np.abs(gm - og.maps) / tol(og.maps)
    assert err.max() <= 1.0
    del gm, err
    rng = np.random.default_rng(4)
    poses = random_poses(rng, 8192, s.box_center, s.box_size, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    st = compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag, "cfg4",
                        cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    _log("score_cfg4", dict(st, N=lig.N, T=lig.T, P=lig.P))
    steps = 3
    r1 = dk.dock_search(p, [grid], [lig], [box], s.copies, steps, s.bfgs_cap, 11)
    r2 = dk.dock_search(p, [grid], [lig], [box], s.copies, steps, s.bfgs_cap, 11)
    assert torch.equal(r1["best_e"], r2["best_e"]) and torch.equal(r1["best_pose"], r2["best_pose"])
    r0 = dk.dock_search(p, [grid], [lig], [box], s.copies, 0, s.bfgs_cap, 11)
    assert bool((r1["best_e"] <= r0["best_e"] + 1e-6).all())          # best only improves on the optimised start
    k = int(r1["topk_count"][0])
    assert 1 <= k <= 10
    tp = r1["topk_pose"][0, :k].cpu().numpy().astype(np.float64)
    te = r1["topk_e"][0, :k].cpu().numpy()
    oe3, _, _, d3 = orc.score_batch(op, og, oL, tp)
    ok = d3["cutoff_margin"] > 1e-4
    assert np.all(np.abs(te - oe3)[ok] <= tol(oe3)[ok])
    assert np.all(np.diff(te) >= 0)
    _log("search_cfg4", dict(copies=s.copies, steps=steps, evals=int(r1["evals"][0]), best=float(te[0])))


# ----------------------------------------------------------------------------------- NEXT-1: Barzilai-Borwein
@pytest.mark.parametrize("cfg,n", [(0, 256), (1, 256)])
def test_bb_local_opt(dk, orc, torch, tiny, micro, cfg, n):
    """The paper's own local optimizer (reading S13) on both sides: one evaluation per iteration,
    best point seen returned.  Deterministic prefix (1 and 2 iterations) against the oracle under S20; the
    free-running 150-iteration result as a distribution (BB is non-monotone, so round-off decides the path)."""
    s, (p0, box, grid, lig), (op0, og, oL) = tiny if cfg == 0 else micro
    p = dk.dock_default_params()
    p.optimizer = 1
    op = orc.params_as_fp32(orc.default_params())
    op.optimizer = 1
    rng = np.random.default_rng(17)
    poses = random_poses(rng, n, s.box_center, s.box_size * 0.6, lig.T)
    pd = torch.from_numpy(poses).cuda()
    e0 = orc.score_batch(op, og, oL, poses.astype(np.float64), want_grad=False)[0]
    for cap in (1, 2):
        o, e, it = dk.dock_local_opt_batch(p, grid, lig, pd, cap)
        ref = np.array([orc.local_opt(op, og, oL, poses[i].astype(np.float64), cap)[0] for i in range(n)])
        chk, _, _, dg = orc.score_batch(op, og, oL, o.cpu().numpy().astype(np.float64))
        ok = dg["cutoff_margin"] > KINK_MARGIN
        ge = e.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(ge - chk)[ok] <= tol(chk)[ok])                  # reported E = E of the reported pose
        assert np.all(it.cpu().numpy()[:, 1] == it.cpu().numpy()[:, 0] + 1)  # evaluations = iterations + 1
        agree = (np.abs(ge - ref) <= 10 * tol(ref))[ok]
        assert agree.mean() >= 0.97, (cap, float(agree.mean()))
    cap = 150
    o, e, it = dk.dock_local_opt_batch(p, grid, lig, pd, cap)
    ge = e.cpu().numpy().astype(np.float64)
    ref = [orc.local_opt(op, og, oL, poses[i].astype(np.float64), cap) for i in range(n)]
    re_ = np.array([r[0] for r in ref])
    chk, _, _, dg = orc.score_batch(op, og, oL, o.cpu().numpy().astype(np.float64))
    ok = dg["cutoff_margin"] > KINK_MARGIN
    assert np.all(np.abs(ge - chk)[ok] <= tol(chk)[ok])
    assert np.all(ge <= e0 + tol(e0))                                        # best-seen never exceeds the start
    qg, qr = np.quantile(ge, [0.25, 0.5, 0.75]), np.quantile(re_, [0.25, 0.5, 0.75])
    st = dict(cfg=cfg, n=n, cap=cap, agree_1e3=float((np.abs(ge - re_) <= 1e-3).mean()),
              gpu_quartiles=qg.tolist(), ref_quartiles=qr.tolist(), gpu_mean=float(ge.mean()), ref_mean=float(re_.mean()),
              gpu_iters=float(it.cpu().numpy()[:, 0].mean()), ref_iters=float(np.mean([r[2] for r in ref])))
    _log("bb_local_opt", st)
    assert np.all(np.abs(qg - qr) <= 0.75 + 0.15 * np.abs(qr)), st


def test_bb_search_properties(dk, orc, torch, tiny):
    """Search driven by BB: bitwise determinism, zero steps = local optimum of the start, winners re-scored by the oracle."""
    s, (p0, box, grid, lig), (op0, og, oL) = tiny
    p = dk.dock_default_params()
    p.optimizer = 1
    r1 = dk.dock_search(p, [grid], [lig], [box], s.copies, s.steps, 150, 5)
    r2 = dk.dock_search(p, [grid], [lig], [box], s.copies, s.steps, 150, 5)
    assert torch.equal(r1["best_e"], r2["best_e"]) and torch.equal(r1["best_pose"], r2["best_pose"])
    r0 = dk.dock_search(p, [grid], [lig], [box], s.copies, 0, 150, 5)
    assert bool((r1["best_e"] <= r0["best_e"] + 1e-6).all())
    k = int(r1["topk_count"][0])
    tp = r1["topk_pose"][0, :k].cpu().numpy().astype(np.float64)
    te = r1["topk_e"][0, :k].cpu().numpy()
    op = orc.params_as_fp32(orc.default_params())
    oe, _, _, d = orc.score_batch(op, og, oL, tp)
    ok = d["cutoff_margin"] > KINK_MARGIN
    assert np.all(np.abs(te - oe)[ok] <= tol(oe)[ok])
    ev = int(r1["evals"][0])
    _log("bb_search", dict(copies=s.copies, steps=s.steps, evals=ev, best=float(te[0])))


def test_maximum_ligand_size_local_opt_and_search(dk, orc, torch, micro):
    """DOCK_MAX_ATOMS x DOCK_MAX_TORSIONS through the optimizer and the search (4 atoms per lane, 38 x 38 inverse
    Hessian per warp): the optimizer never raises the energy, the reported energies are the oracle's energies of the
    reported poses, the search is deterministic."""
    s0, (p, box, grid, _), (op, og, _) = micro
    import dock_synth
    from dock_synth.generators import LIG_TYPES_FULL
    rng = np.random.default_rng(228)
    ligd = dock_synth.make_ligand(rng, 128, 32, LIG_TYPES_FULL)
    lig, oL = dk.LigandHandle(ligd), orc.Ligand(ligd)
    poses = random_poses(rng, 64, s0.box_center, s0.box_size * 0.5, 32)
    e0, _, _ = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    o, e, it = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses).cuda(), 30)
    assert bool((e <= e0 + 1e-3 + 1e-4 * e0.abs()).all())
    chk, _, _, dg = orc.score_batch(op, og, oL, o.cpu().numpy().astype(np.float64))
    ok = dg["cutoff_margin"] > KINK_MARGIN
    assert ok.any() and np.all(np.abs(e.cpu().numpy() - chk)[ok] <= tol(chk)[ok])
    r1 = dk.dock_search(p, [grid], [lig], [box], 32, 2, 20, 9)
    r2 = dk.dock_search(p, [grid], [lig], [box], 32, 2, 20, 9)
    assert torch.equal(r1["best_e"], r2["best_e"]) and int(r1["topk_count"][0]) >= 1
    assert bool(torch.isfinite(r1["best_e"]).all())


def test_search_from_site_restrained_initial_poses(dk, torch, tiny):
    """NEXT-3: copies start inside box ∩ union of balls around synthetic site points; with zero MC steps
    the search returns exactly the local optima of those poses."""
    from dock_synth import make_site_points
    s, (p, box, grid, lig), _ = tiny
    site = make_site_points(np.random.default_rng(2), s.box_center, s.box_size, n=20, step=1.0, margin=3.0)
    init = dk.dock_init_poses_site(box, lig.T, 99, 0, 32, site, 3.0)
    d = np.min(np.linalg.norm(init[:, None, :3] - site[None], axis=2), axis=1)
    assert np.all(d <= 3.0 + 1e-4)
    r = dk.dock_search(p, [grid], [lig], [box], 32, 0, 50, 99, init_poses=torch.from_numpy(init[None]).cuda())
    o, e, it = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(init).cuda(), 50)
    assert torch.equal(r["best_e"][0], e)
    r5 = dk.dock_search(p, [grid], [lig], [box], 32, 5, 50, 99, init_poses=torch.from_numpy(init[None]).cuda())
    assert bool((r5["best_e"] <= r["best_e"] + 1e-6).all())


# ----------------------------------------------------------------------------------- NEXT-2: eq. 4 gradient maps
def test_eq4_maps_scores_and_search(dk, orc, torch, tiny):
    """PAPER.md:51 / eq. 4 (221): four channels per map (score and its per-vertex gradient), gradient of a pose from the
    interpolated vertex gradients.  Maps at every node, per-pose energies and gradients on both evaluators (batch
    scoring: thread per pose; local optimisation with zero iterations: warp per pose), and a search on those maps."""
    s, (p3, box, grid3, lig), (op, og3, oL) = tiny
    p = dk.dock_default_params()
    p.grad_mode = 1
    grid = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types)
    og = orc.build_grid(op, s.protein_xyz, s.protein_type, s.box_center, s.box_size, s.spacing, s.lig_types, grad=True)
    gm = grid.data.cpu().numpy().astype(np.float64)                    # [n_maps, 4, nz, ny, nx]
    assert gm.shape[1] == 4 and int(grid.desc.n_channels) == 4
    g3m = grid3.data.cpu().numpy().astype(np.float64)                  # the score channel is the eq. 2 map (to round-off:
    assert np.all(np.abs(gm[:, 0] - g3m) <= 1e-5 + 1e-6 * np.abs(g3m))  # the two kernel variants contract their FMAs differently)
    assert np.all(np.abs(gm[:, 0] - og.maps) <= tol(og.maps))
    assert np.all(np.abs(gm[:, 1:] - og.gmaps) <= tol(og.gmaps))
    rng = np.random.default_rng(44)
    poses = random_poses(rng, 2051, s.box_center, s.box_size * 1.2, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    # eq. 4's gradient is continuous across cell faces (only the kinks of the intra pairs remain one-sided)
    diag4 = diag.copy()
    diag4["face_margin"] = 1.0
    st = compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag4, "eq4",
                        cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    _log("score_eq4", st)
    e3, g3, _ = dk.dock_score_batch(p3, grid3, lig, torch.from_numpy(poses).cuda())
    assert torch.allclose(e, e3, rtol=1e-6, atol=1e-5) and not torch.allclose(g, g3, atol=1e-3)   # same E, different gradient
    # warp evaluator: zero optimizer iterations = one evaluation; its energy matches, and one BFGS step agrees with the oracle
    o0, e0, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses[:128]).cuda(), 0)
    assert torch.allclose(e0, e[:128], rtol=1e-5, atol=1e-4)
    o1, e1, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses[:128]).cuda(), 1)
    r1 = np.array([orc.local_opt(op, og, oL, poses[i].astype(np.float64), 1)[0] for i in range(128)])
    c1, _, _, d1 = orc.score_batch(op, og, oL, o1.cpu().numpy().astype(np.float64))
    ok1 = d1["cutoff_margin"] > KINK_MARGIN
    assert (np.abs(e1.cpu().numpy() - r1) <= 10 * tol(r1))[ok1].mean() >= 0.97
    r = dk.dock_search(p, [grid], [lig], [box], s.copies, 5, 50, 3)
    r2 = dk.dock_search(p, [grid], [lig], [box], s.copies, 5, 50, 3)
    assert torch.equal(r["best_e"], r2["best_e"]) and int(r["topk_count"][0]) >= 1
    k = int(r["topk_count"][0])
    oe2, _, _, d2 = orc.score_batch(op, og, oL, r["topk_pose"][0, :k].cpu().numpy().astype(np.float64))
    ok = d2["cutoff_margin"] > KINK_MARGIN
    assert np.all(np.abs(r["topk_e"][0, :k].cpu().numpy() - oe2)[ok] <= tol(oe2)[ok])


@pytest.mark.parametrize("w", [(0.05, -0.004, 0.5, -0.03, -0.4), (0.03, 0.006, 0.0, 0.02, 0.3), (-0.02, 0.0, 1.2, 0.0, -0.9),
                               (0.0, -0.005, 0.84, -0.035, 0.0)])
def test_other_term_weights_and_signs(dk, orc, torch, tiny, w):
    """The evaluators fold the weights into exponent arguments and carry forces scaled by -sign(w1): every sign pattern
    (and zero weights) must reproduce the oracle, on both evaluators (batch scoring and the optimizer's evaluator)."""
    s, _, _ = tiny
    p = dk.dock_default_params()
    op = orc.default_params()
    for k in range(5):
        p.w[k] = w[k]
        op.w[k] = w[k]
    op = orc.params_as_fp32(op)
    box = dk.make_box(s.box_center, s.box_size, s.spacing)
    grid = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types)
    lig = dk.LigandHandle(s.ligand)
    og = orc.build_grid(op, s.protein_xyz, s.protein_type, s.box_center, s.box_size, s.spacing, s.lig_types)
    oL = orc.Ligand(s.ligand)
    assert np.all(np.abs(grid.data.cpu().numpy().astype(np.float64) - og.maps) <= tol(og.maps))
    rng = np.random.default_rng(91)
    poses = random_poses(rng, 1031, s.box_center, s.box_size * 1.1, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag, f"w={w}",
                   cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    # warp evaluator through the optimizer: zero iterations = one evaluation; one iteration = the oracle's first step
    o0, e0, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses[:128]).cuda(), 0)
    assert torch.allclose(e0, e[:128], rtol=1e-5, atol=1e-4)
    o1, e1, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses[:128]).cuda(), 1)
    r1 = np.array([orc.local_opt(op, og, oL, poses[i].astype(np.float64), 1)[0] for i in range(128)])
    c1, _, _, d1 = orc.score_batch(op, og, oL, o1.cpu().numpy().astype(np.float64))
    ok1 = d1["cutoff_margin"] > KINK_MARGIN
    assert (np.abs(e1.cpu().numpy() - r1) <= 10 * tol(r1))[ok1].mean() >= 0.95


def test_non_cubic_box_scores_and_search(dk, orc, torch, tiny):
    """Box with three different edge lengths (33 x 25 x 41 nodes): index arithmetic of the grid build, the packed
    cells and both evaluators; atoms outside on every axis exercise the per-axis wall."""
    s, _, _ = tiny
    center, size = [10.0, 9.5, 10.5], [12.0, 9.0, 15.0]
    p = dk.dock_default_params()
    op = orc.params_as_fp32(orc.default_params())
    box = dk.make_box(center, size, s.spacing)
    grid = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types)
    assert tuple(grid.dims) == (33, 25, 41)
    og = orc.build_grid(op, s.protein_xyz, s.protein_type, center, size, s.spacing, s.lig_types)
    assert np.all(np.abs(grid.data.cpu().numpy().astype(np.float64) - og.maps) <= tol(og.maps))
    lig, oL = dk.LigandHandle(s.ligand), orc.Ligand(s.ligand)
    rng = np.random.default_rng(77)
    poses = random_poses(rng, 1500, np.array(center, np.float32), np.array(size, np.float32) * 1.3, lig.T)
    e, g, t = dk.dock_score_batch(p, grid, lig, torch.from_numpy(poses).cuda())
    oe, ograd, oterms, diag = orc.score_batch(op, og, oL, poses.astype(np.float64))
    compare_scores(e.cpu().numpy(), g.cpu().numpy(), t.cpu().numpy(), oe, ograd, oterms, diag, "noncubic",
                   cond=orc.grad_cond(op, og, oL, poses.astype(np.float64)), n_atoms=lig.N, n_pairs=lig.P)
    o0, e0, _ = dk.dock_local_opt_batch(p, grid, lig, torch.from_numpy(poses[:96]).cuda(), 0)
    assert torch.allclose(e0, e[:96], rtol=1e-5, atol=1e-4)
    r = dk.dock_search(p, [grid], [lig], [box], 32, 4, 40, 21)
    k = int(r["topk_count"][0])
    oe2, _, _, d2 = orc.score_batch(op, og, oL, r["topk_pose"][0, :k].cpu().numpy().astype(np.float64))
    ok = d2["cutoff_margin"] > KINK_MARGIN
    assert np.all(np.abs(r["topk_e"][0, :k].cpu().numpy() - oe2)[ok] <= tol(oe2)[ok])
    # the host-generated initial poses lie inside this box
    init = dk.dock_init_poses(box, lig.T, 21, 0, 32)
    assert np.all(np.abs(init[:, :3] - np.array(center)) <= np.array(size) / 2 + 1e-5)


def test_batched_grid_build_equals_single_builds(dk, torch):
    """dock_build_grids_batch (SURVEY.md 8(b), configs[3]): heterogeneous proteins and boxes in one call give bitwise
    the maps of one call per system, in both images."""
    systems = [make_system(3, seed=0, index=i, n_prot=400 + 150 * i) for i in range(4)]
    p = dk.dock_default_params()
    boxes = [dk.make_box(s.box_center, s.box_size if i != 2 else s.box_size * np.array([0.5, 0.75, 1.0], np.float32), s.spacing)
             for i, s in enumerate(systems)]
    lt = systems[0].lig_types
    batch = dk.dock_build_grids_batch(p, [(s.protein_xyz, s.protein_type) for s in systems], boxes, lt)
    assert len(batch) == 4
    for s, b, g in zip(systems, boxes, batch):
        one = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, b, lt)
        assert tuple(g.dims) == tuple(one.dims)
        assert torch.equal(g.data, one.data)                                 # the maps ...
        off = (g.data.numel() * 4 + 255) // 256 * 256                        # ... and the packed gather image behind them
        assert torch.equal(g.buf[off:], one.buf[off:])
    assert dk.dock_build_grids_batch(p, [], [], lt) == []
