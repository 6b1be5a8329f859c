"""Shared helpers for the GPU-vs-oracle parity tests (the two sides only share dock_synth inputs)."""
import numpy as np

FACE_MARGIN = 1e-4   # A: closer than this to a cell face the gradient of the interpolant is two-valued
KINK_MARGIN = 1e-4   # A: closer than this to the cutoff / a piecewise kink of an intra pair


def tol(ref):
    """S20: pass iff |gpu - ref| <= 1e-3 + 1e-4 |ref| (BASELINE.json:north_star)."""
    return 1e-3 + 1e-4 * np.abs(ref)


def oracle_side(O, s, build_grid=True):
    op = O.params_as_fp32(O.default_params())
    og = O.build_grid(op, s.protein_xyz, s.protein_type, s.box_center, s.box_size, s.spacing, s.lig_types) if build_grid else None
    return op, og, O.Ligand(s.ligand)


def gpu_side(dk, s, build_grid=True):
    p = dk.dock_default_params()
    box = dk.make_box(s.box_center, s.box_size, s.spacing)
    grid = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types) if build_grid else None
    return p, box, grid, dk.LigandHandle(s.ligand)


EPS32 = 2.0 ** -24   # unit round-off of the kernel's arithmetic
COND_C = 8.0         # S20': a component is resolvable in fp32 only to ~COND_C * EPS32 * A_k


def compare_scores(gpu_e, gpu_grad, gpu_terms, ref_e, ref_grad, ref_terms, diag, what="", cond=None,
                   n_atoms=30, n_pairs=300):
    """Element-by-element comparison with the discontinuity exemptions; returns a stats dict.

    `cond` (oracle.grad_cond) is the conditioning scale A_k of each gradient component.  Reading S20'
    (DESIGN.md): a component passes iff |gpu - ref| <= 1e-3 + 1e-4 |ref| + COND_C * EPS32 * A_k; the
    fraction that passes the plain S20 rule (without the last term) is reported and must be >= 99.99 %.
    """
    gpu_e = np.asarray(gpu_e, np.float64)
    n = len(ref_e)
    ok_e = diag["cutoff_margin"] > KINK_MARGIN          # E itself jumps only at the cutoff
    ok_g = (diag["kink_margin"] > KINK_MARGIN) & (diag["face_margin"] > FACE_MARGIN)
    # a pose is exempt if ANY of its pairs / atoms sits within the margin of a discontinuity, so the
    # expected exempt fraction grows with the ligand: ~ P * 2 kinks * 2e-4 / 8 A and N * 3 axes * 2e-4 / 0.375 A
    # (x2 safety, + 2 %)
    min_e = 1.0 - 2.0 * (n_pairs * 2 * KINK_MARGIN / 8.0) - 0.02
    min_g = min_e - 2.0 * (n_pairs * 2 * KINK_MARGIN / 8.0) - 2.0 * (n_atoms * 3 * 2 * FACE_MARGIN / 0.375) - 0.02
    assert ok_e.mean() > min_e and ok_g.mean() > min_g, (what, ok_e.mean(), ok_g.mean(), min_e, min_g)
    err_e = np.abs(gpu_e - ref_e) / tol(ref_e)
    assert np.all(np.isfinite(gpu_e)), what
    assert np.all(err_e[ok_e] <= 1.0), (what, "E", float(err_e[ok_e].max()), int(np.argmax(np.where(ok_e, err_e, 0))))
    stats = dict(n=n, compared_e=int(ok_e.sum()), compared_g=int(ok_g.sum()), max_err_e=float(err_e[ok_e].max()))
    if gpu_terms is not None:
        gt = np.asarray(gpu_terms, np.float64)
        err_t = np.abs(gt - ref_terms) / tol(ref_terms)
        assert np.all(err_t[ok_e] <= 1.0), (what, "terms", float(err_t[ok_e].max()))
        stats["max_err_terms"] = float(err_t[ok_e].max())
    if gpu_grad is not None:
        gg = np.asarray(gpu_grad, np.float64)
        err_g = np.abs(gg - ref_grad) / tol(ref_grad)
        assert np.all(np.isfinite(gg)), what
        stats["max_err_g_s20"] = float(err_g[ok_g].max())
        stats["frac_g_within_s20"] = float((err_g[ok_g] <= 1.0).mean())
        assert stats["frac_g_within_s20"] >= 0.9999, (what, stats)
        t_g = tol(ref_grad) + (COND_C * EPS32 * np.asarray(cond) if cond is not None else 0.0)
        err_c = np.abs(gg - ref_grad) / t_g
        assert np.all(err_c[ok_g] <= 1.0), (what, "grad", float(err_c[ok_g].max()),
                                            np.unravel_index(int(np.argmax(np.where(ok_g[:, None], err_c, 0))), err_c.shape))
        stats["max_err_g"] = float(err_c[ok_g].max())
    return stats


def oracle_self_agreement(O, op, og, oL, poses, cap, eps=6e-8, seeds=(1, 2, 3), tol_e=1e-3):
    """The chaos ceiling of a free-running local optimisation: fraction of poses whose
    final energy the ORACLE reproduces within tol_e when its start pose is perturbed by a relative eps (6e-8 = half an
    fp32 ulp: the smallest difference any single-precision implementation must introduce).  Mean over `seeds`."""
    poses = np.asarray(poses, np.float64)
    e0, _, info0 = O.local_opt_batch(op, og, oL, poses, cap)
    rates, med = [], []
    for sd in seeds:
        r = np.random.default_rng(sd)
        pp = poses * (1.0 + eps * (2.0 * r.random(poses.shape) - 1.0))
        e1, _, _ = O.local_opt_batch(op, og, oL, pp, cap)
        rates.append(float(np.mean(np.abs(e1 - e0) <= tol_e)))
        med.append(float(np.median(np.abs(e1 - e0))))
    return dict(agree=float(np.mean(rates)), median_abs=float(np.mean(med)), n=int(len(poses)), e0=e0, info0=info0)
