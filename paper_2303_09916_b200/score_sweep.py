"""When does the run-time specialised score kernel (dock_params.score_kernel = 2) pay?  (profiles/r2b.md)

    python -m paper_2303_09916_b200.score_sweep [--poses 524288] [--shapes "12,2 20,4 30,6"]

Scores one seeded batch of random poses per ligand shape (N atoms, T torsions; synthetic ligands of dock_synth on the
BASELINE configs[1] grid) with the generic and with the specialised kernel: CUDA-event medians with the L2 flushed
between calls, the compilation time of the specialised kernel, and the largest gradient difference between the two in
tolerance units (1e-3 + 1e-4 |g|).  Needs a GPU; marshalling and timing only -- no arithmetic of the method here.
"""
from __future__ import annotations

import argparse
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--poses", type=int, default=524288)
    ap.add_argument("--shapes", default="12,2 16,3 20,4 24,5 28,4 30,6 33,6")
    ap.add_argument("--reps", type=int, default=8)
    args = ap.parse_args()
    import torch
    import paper_2303_09916_b200 as dk
    from dock_synth import make_ligand, make_system, random_poses

    s = make_system(1, seed=0)
    p = dk.dock_default_params()
    box = dk.make_box(s.box_center, s.box_size, s.spacing)
    grid = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(params, lig, poses):
        t0 = time.perf_counter()
        out = dk.dock_score_batch(params, grid, lig, poses)
        torch.cuda.synchronize()
        first = time.perf_counter() - t0
        ts = []
        for _ in range(args.reps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            dk.dock_score_batch(params, grid, lig, poses, out=out)
            b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return out, float(np.median(ts)), first

    print(f"{args.poses} poses per batch; times in ms (median of {args.reps}, L2 flushed)")
    for shape in args.shapes.split():
        N, T = (int(v) for v in shape.split(","))
        rng = np.random.default_rng(100 + N)
        lig = dk.LigandHandle(make_ligand(rng, N, T, s.lig_types))
        poses = torch.from_numpy(random_poses(rng, args.poses, s.box_center, s.box_size, lig.T)).cuda()
        p.score_kernel = 1
        ref, t_gen, _ = timed(p, lig, poses)
        p.score_kernel = 2
        try:
            out, t_jit, first = timed(p, lig, poses)
        except dk.DockError as e:
            print(f"N={N:3d} T={T:2d} P={lig.P:4d}: generic {t_gen:.4f}  specialised unavailable ({e})")
            continue
        dg = float(((out[1] - ref[1]).abs() / (1e-3 + 1e-4 * ref[1].abs())).max())
        print(f"N={N:3d} T={T:2d} P={lig.P:4d}: generic {t_gen:.4f}  specialised {t_jit:.4f}  ratio {t_gen / t_jit:.2f}  "
              f"compile + first call {first:.1f} s  max |dgrad| {dg:.2f} tol", flush=True)


if __name__ == "__main__":
    main()
