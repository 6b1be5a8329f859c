#!/usr/bin/env python
"""bench.py -- throughput of the docking hot path on B200 (driver contract).

Default arm: the CUDA library through its C-ABI binding.
    python bench.py [--gpus N] [--steps K] [--warmup W]
  N=1 workload = BASELINE.json:configs[1], the scoring microbench: 1,048,576 random poses of a
  30-atom / 6-torsion ligand scored (energy + gradient + terms) against 81^3 x 8 grid maps of a
  3000-atom synthetic protein.  One "step" = one dock_score_batch call over the whole batch
  (A2-A5).  The grid build (A1) and a config-2 site-docking search (A6-A8) are timed next to it
  and reported under "extra" so that one line covers every row of the hot path.
  N>1 (torchrun): every rank scores its own seeded batch of the same size (weak scaling, no
  data-path collective: poses are independent); value = all ranks' evals / max time.

Reference arm: `--impl reference` times the CPU oracle (oracle/), as it stands, on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "score+gradient pose evals/sec"
UNIT = "evals/s"
# FP32 ALU roof derived from the guide's unit counts and clocks:
# 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz (clocks.max.sm).  The MEASURED roof (dock_probe_peaks: an FFMA
# loop on the same GPU, same run) is printed beside it; MEASURED_PEAKS.json holds only HBM and tensor-core peaks,
# neither of which bounds this path.
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def algorithmic_flops(N: int, T: int, p_in: float, p_out: float) -> float:
    """Algorithmic fp operations of one score+gradient evaluation (counted on
    the oracle's statements, one per add/mul/div/sqrt/exp/compare/min/max, fused nothing)."""
    return 93.0 * N + 130.0 * T + 62.0 * p_in + 8.0 * p_out + 50.0


# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "10", "-f", self.path], stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        try:
            rows = [r.split(",") for r in open(self.path).read().strip().splitlines() if r.strip()]
            os.unlink(self.path)
        except OSError:
            return out
        sm, reasons, smax, pw = [], set(), None, []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                smax = float(r[1])
                pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].strip().lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            # "under load" = the upper half of the samples (the sampler also sees the idle edges)
            hi = sorted(sm)[len(sm) // 2:]
            out.update(sm_mhz=float(np.median(hi)), sm_max_mhz=smax, reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw) if pw else None)
        return out


def _dist_setup(n_gpus: int):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    import torch
    if world != n_gpus:
        # the driver launches N > 1 through torch.distributed.run (one rank per GPU); a plain `python bench.py --gpus N`
        # would silently measure one GPU, so it is refused
        sys.stderr.write(f"bench.py: --gpus {n_gpus} but WORLD_SIZE={world}: launch with\n  python -m torch.distributed.run "
                         f"--nnodes=1 --nproc-per-node {n_gpus} --master-addr 127.0.0.1 --master-port P bench.py --gpus {n_gpus} ...\n")
        sys.exit(2)
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        torch.cuda.set_device(0)
    return rank, world, local


def _max_over_ranks(x: float, world: int) -> float:
    from paper_2303_09916_b200.shard import max_over_ranks
    return max_over_ranks(x, device="cuda") if world > 1 else x


def _barrier(world: int):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------------
def _workload(rank: int):
    """Config 1 inputs (seeded): system, poses.  Rank r draws its own pose batch."""
    from dock_synth import CONFIGS, make_system, random_poses
    s = make_system(1, seed=0)
    n = CONFIGS[1]["n_poses"]
    rng = np.random.default_rng(np.random.PCG64([0, 1, 1000 + rank]))
    poses = random_poses(rng, n, s.box_center, s.box_size, s.ligand.T)
    return s, poses


def run_reference(args) -> dict:
    """The CPU oracle, as it stands, on the host cores; each step scores a bounded sample."""
    from oracle import oracle as O
    O.build()
    s, poses = _workload(0)
    op = O.params_as_fp32(O.default_params())
    og = O.build_grid(op, s.protein_xyz, s.protein_type, s.box_center, s.box_size, s.spacing, s.lig_types)
    oL = O.Ligand(s.ligand)
    n = min(args.ref_sample, poses.shape[0])
    p64 = poses[:n].astype(np.float64)
    for _ in range(args.warmup):
        O.score_batch(op, og, oL, p64)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.score_batch(op, og, oL, p64)
    dt = (time.perf_counter() - t0) / max(1, args.steps)
    v = n / dt
    cores = O.num_threads()
    sample = f"first {n} poses of the config-1 batch per step, fp64, OpenMP over poses"
    return {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[1] scoring microbench", "n_poses_per_step": n, "N": oL.N, "T": oL.T,
                   "P": oL.P, "grid": "81^3 x 8 fp64", "bounded_sample": n < poses.shape[0]},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def _time_events(torch, fn, reps: int, flush=None):
    """Per-call CUDA-event times (ms) on the current stream; `flush` runs untimed before each call."""
    out = []
    for _ in range(reps):
        if flush is not None:
            flush()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        b.synchronize()
        out.append(a.elapsed_time(b))
    return out


def run_ours(args) -> dict:
    import torch
    rank, world, local = _dist_setup(args.gpus)
    import paper_2303_09916_b200 as dk
    dk.load_library()
    from dock_synth import make_system

    s, poses_h = _workload(rank)
    p = dk.dock_default_params()
    box = dk.make_box(s.box_center, s.box_size, s.spacing)
    # which score kernel the headline times: 0 / 1 (default here) = the generic kernel, which is what dock_score_batch runs
    # unless the caller opts in; 2 = the kernel specialised for the ligand at run time (NVRTC; compiled during the
    # warm-up, i.e. its 0.4-6 s per ligand are NOT in the number); -1 = 2 if the compiler is there, else generic.
    # The other kernel is timed beside it (extra.*_score_kernel, with its first-call cost and break-even batch size).
    args.score_kernel_note = ""
    if args.score_kernel < 0:
        args.score_kernel = 2
        args.score_kernel_note = "auto"
    p.score_kernel = args.score_kernel
    lig = dk.LigandHandle(s.ligand)
    n = poses_h.shape[0]
    np_, ng = 7 + lig.T, 6 + lig.T

    # A1: grid maps (timed as an extra; the maps then stay resident for the scoring steps)
    grid = dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types)
    torch.cuda.synchronize()
    t_grid = _time_events(torch, lambda: dk.dock_build_grids(p, s.protein_xyz, s.protein_type, box, s.lig_types), 3)

    poses = torch.from_numpy(poses_h).cuda()
    out = (torch.empty(n, dtype=torch.float32, device="cuda"),
           torch.empty((n, ng), dtype=torch.float32, device="cuda"),
           torch.empty((n, 3), dtype=torch.float32, device="cuda"))
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def flush():
        flush_buf.fill_(1)

    def step():
        dk.dock_score_batch(p, grid, lig, poses, out=out)

    try:
        step()
    except dk.DockError as e:                      # NVRTC missing / ligand outside the generator: the generic kernel
        if args.score_kernel != 2 or args.score_kernel_note != "auto":
            raise
        args.score_kernel = p.score_kernel = 0
        args.score_kernel_note = f"auto: specialised kernel unavailable ({e}), generic kernel timed"
    for _ in range(max(3, args.warmup)):
        step()
    _barrier(world)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = dk.launch_count()
    wall0 = time.perf_counter()
    ts = _time_events(torch, step, args.steps, flush if not args.no_flush else None)
    _barrier(world)
    wall = time.perf_counter() - wall0
    launches = dk.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else {}
    t_step = _max_over_ranks(float(np.sum(ts)) / 1e3, world) / args.steps          # seconds per step, max over ranks
    value = world * n / t_step

    # e2e: the same call with HOST (pinned) buffers, copies inside the timed region
    ph = torch.from_numpy(poses_h).pin_memory()
    eh = (torch.empty(n, dtype=torch.float32).pin_memory(), torch.empty((n, ng), dtype=torch.float32).pin_memory(),
          torch.empty((n, 3), dtype=torch.float32).pin_memory())

    def step_host():
        dk.dock_score_batch_host(p, grid, lig, ph, want_grad=True, want_terms=True, out=eh)

    for _ in range(2):
        step_host()
    _barrier(world)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_host()
    torch.cuda.synchronize()
    t_e2e = _max_over_ranks((time.perf_counter() - t0) / args.steps, world)
    h2d = n * np_ * 4
    d2h = n * (1 + ng + 3) * 4
    assert np.array_equal(eh[0].numpy(), out[0].cpu().numpy()), "host and device entry points disagree"

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
        "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "configs[1] scoring microbench", "n_poses_per_gpu": n, "N": lig.N, "T": lig.T, "P": lig.P,
                   "grid": "81^3 x 8 fp32", "outputs": "energy+gradient+terms",
                   "score_kernel": ("specialised at run time (NVRTC, dock_params.score_kernel = 2; compiled during the warm-up)"
                                    if args.score_kernel == 2 else "generic (dock_params.score_kernel = 0, the library default)")
                                   + (f" [{args.score_kernel_note}]" if args.score_kernel_note else ""),
                   "l2": "flushed between timed steps (256 MiB write)" if not args.no_flush else "not flushed",
                   "parallelism": f"pose-sharded x{world}, no collective"},
        "e2e": {"value": world * n / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": t_e2e * 1e3},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "wall_s_timed_region": wall,
    }
    # measured roofs of the units this path is bound by (probe kernels in the library, same GPU, same run)
    peaks = dk.dock_probe_peaks()

    extra = {}
    # the other score kernel next to the headline (rank 0): same batch, same launch configuration, L2 flushed
    if rank == 0 and not args.no_search:
        po = dk.dock_default_params()
        po.score_kernel = 1 if args.score_kernel == 2 else 2
        name = "generic_score_kernel" if args.score_kernel == 2 else "specialised_score_kernel"
        try:
            t0 = time.perf_counter()
            oo = dk.dock_score_batch(po, grid, lig, poses)
            torch.cuda.synchronize()
            t_first = time.perf_counter() - t0
            to = _time_events(torch, lambda: dk.dock_score_batch(po, grid, lig, poses, out=oo), min(args.steps, 20), flush)
            de = float((oo[0] - out[0]).abs().max())
            dg = float(((oo[1] - out[1]).abs() / (1e-3 + 1e-4 * out[1].abs())).max())
            t_other, t_head = float(np.mean(to)) / 1e3, float(np.mean(ts)) / 1e3
            t_spec, t_gen = (t_other, t_head) if name.startswith("spec") else (t_head, t_other)
            extra[name] = {"ms_per_step": float(np.mean(to)), "evals_per_s": n / (float(np.mean(to)) / 1e3),
                           "specialised_over_generic": t_gen / t_spec,
                           "first_call_s": t_first, "max_abs_dE_vs_headline_kernel": de, "max_dgrad_tol_units_vs_headline_kernel": dg,
                           "note": "dock_params.score_kernel = 2 (jit_score.cu): first_call_s includes the NVRTC compilation for this ligand"
                                   if name.startswith("spec") else "dock_params.score_kernel = 1"}
            if name.startswith("spec"):
                gain = (t_gen - t_spec) / n                     # seconds saved per pose once the kernel is compiled
                extra[name]["break_even_poses"] = (t_first - t_spec) / gain if gain > 0 else None
                extra[name]["break_even_note"] = ("poses of ONE ligand after which first_call_s (compilation) is paid back by the faster "
                                                  "kernel; null = never (the generic kernel is at least as fast for this ligand)")
            del oo
        except dk.DockError as e:
            extra[name] = {"unavailable": str(e)}

    # ---- extras that shard over ranks (N > 1): the screening batch, systems [b, e) per rank, no exchange ----
    if not args.no_search:
        from paper_2303_09916_b200.shard import shard_range
        n3 = args.screen_systems
        b3, e3 = shard_range(n3, rank, world)
        sy = [make_system(3, seed=0, index=i) for i in range(b3, e3)]
        bx = [dk.make_box(q.box_center, q.box_size, q.spacing) for q in sy]
        lg = [dk.LigandHandle(q.ligand) for q in sy]
        pr = [(q.protein_xyz, q.protein_type) for q in sy]
        gr = dk.dock_build_grids_batch(p, pr, bx, sy[0].lig_types)            # warm-up (module load, allocator)
        torch.cuda.synchronize()
        del gr
        _barrier(world)
        t0 = time.perf_counter()
        gr = dk.dock_build_grids_batch(p, pr, bx, sy[0].lig_types)
        torch.cuda.synchronize()
        t_g3 = _max_over_ranks(time.perf_counter() - t0, world)
        run3 = lambda: dk.dock_search(p, gr, lg, bx, 128, 40, 300, 2023, system_base=b3)
        run3()
        _barrier(world)
        t0 = time.perf_counter()
        r3 = run3()
        torch.cuda.synchronize()
        t_3 = _max_over_ranks(time.perf_counter() - t0, world)
        ev3 = int(r3["evals"].sum())
        if world > 1:
            import torch.distributed as dist
            tot = torch.tensor([ev3], dtype=torch.int64, device="cuda")
            dist.all_reduce(tot)
            ev3 = int(tot.item())
        best3 = r3["topk_e"][:, 0].cpu().numpy()
        best3_pose = [r3["best_pose"][i].cpu().numpy() for i in range(min(2, len(sy)))]
        ev3_rank0, t_3_rank0 = int(r3["evals"].sum()), t_3
        extra["screening"] = {"workload": f"configs[3]: {n3} systems x 128 copies x 40 steps, BFGS<=300, ONE dock_build_grids_batch + ONE "
                                          f"dock_search launch per rank ({world} rank(s), systems sharded, no exchange)",
                              "systems": n3, "search_s": t_3, "grid_build_s": t_g3, "evals": ev3, "evals_per_s": ev3 / t_3,
                              "systems_per_s_search_only": n3 / t_3, "systems_per_s": n3 / (t_3 + t_g3),
                              "grid_bytes_resident": int(sum(g.buf.numel() for g in gr)) * world,
                              "best_e_median_rank0": float(np.median(best3)), "best_e_negative_frac_rank0": float((best3 < 0).mean())}
        sys3_keep = sy[:2]
        del gr, r3
    if rank != 0:
        return {}

    # roofline of the dominant kernel (score kernel = the whole step)
    from oracle import oracle as O          # cpu_baseline leg + in-range pair statistics / operation count for the flop figure
    O.build()
    op = O.params_as_fp32(O.default_params())
    og = O.build_grid(op, s.protein_xyz, s.protein_type, s.box_center, s.box_size, s.spacing, s.lig_types)
    oL = O.Ligand(s.ligand)
    ns = min(args.ref_sample, n)
    p64 = poses_h[:ns].astype(np.float64)
    O.score_batch(op, og, oL, p64[:4096])
    t0 = time.perf_counter()
    oe, ograd, oterms, diag = O.score_batch(op, og, oL, p64)
    t_cpu = time.perf_counter() - t0
    p_in = float(diag["pairs_in_range"].mean())
    flops = algorithmic_flops(lig.N, lig.T, p_in, lig.P - p_in)
    counted = O.count_eval_ops(op, og, oL, p64[:2048])                    # the oracle's own statements, operation by operation
    t_kernel = float(np.mean(ts)) / 1e3
    achieved = flops * n / t_kernel / 1e12
    counters = kernel_counters()
    head_kernel = "dock_score_jit" if args.score_kernel == 2 else "score_thread_kernel"
    kc_head = counters.get(head_kernel, {})
    for name in ("generic_score_kernel", "specialised_score_kernel"):
        if name in extra and "ms_per_step" in extra[name]:
            extra[name]["roofline_frac"] = flops * n / (extra[name]["ms_per_step"] / 1e3) / 1e12 / ALU_PEAK_TFLOPS
    peak_meas = max(peaks["ffma_tflops"], peaks["ffma2_tflops"])
    line["roofline"] = {"bound": "alu", "achieved": achieved, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                        "frac": achieved / ALU_PEAK_TFLOPS,
                        "traffic": kc_head.get("dram_bytes_per_launch"),
                        "traffic_source": (f"{kc_head['source']} at commit {kc_head['commit']} (profiles/kernel_counters.json; ncu, not "
                                           "measured by this run)") if kc_head else None,
                        "achieved_occupancy_pct_ncu": kc_head.get("achieved_occupancy_pct"),
                        "kernel": head_kernel, "flops_per_eval": flops, "pairs_in_range_mean": p_in,
                        "peak_source": "derived: 148 SM x 128 lanes x 2 x 1.965 GHz (DESIGN.md)",
                        "peak_measured": peak_meas, "frac_of_measured": achieved / peak_meas,
                        "peak_measured_source": "dock_probe_peaks: FFMA / FFMA2 loops, 8 independent chains per thread, this run",
                        "probes": peaks,
                        "flops_per_eval_opcounted": counted["total"], "opcount": counted,
                        "achieved_opcounted": counted["total"] * n / t_kernel / 1e12,
                        "frac_opcounted": counted["total"] * n / t_kernel / 1e12 / ALU_PEAK_TFLOPS,
                        "flops_note": "frac uses SURVEY.md 8(d)'s formula (93 N + 130 T + 62 P_in + 8 P_out + 50); the *_opcounted "
                                      "figures count every add/mul/div/compare/sqrt/exp of the unoptimised oracle (oracle/opcount.hpp) "
                                      "and are reported for reference",
                        "mufu_frac": (3.0 * p_in + 2.0 * lig.T + 2.0) * n / t_kernel / 1e12 / peaks["mufu_tops"],
                        "gather_frac": lig.N * n / t_kernel / 1e12 / peaks["gather32_tlanes"]}
    line["cpu_baseline"] = {"value": ns / t_cpu, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                            "sample": f"first {ns} poses of the same batch, fp64, OpenMP over poses"}
    # spot parity inside the bench run: what is timed is what is correct
    ge = out[0][:ns].cpu().numpy().astype(np.float64)
    safe = diag["cutoff_margin"] > 1e-4
    err = np.abs(ge - oe) / (1e-3 + 1e-4 * np.abs(oe))
    line["parity_in_bench"] = {"poses": int(safe.sum()), "max_err_tol_units": float(err[safe].max())}

    pairs_in_range = {}

    def oracle_search_rate(q, n_copies, steps, cap, system=0, gpu_best=None, tag=None):
        """The oracle's own search on the first n_copies copies (copies are independent): evaluations/s on the host cores.
        gpu_best: poses the GPU search ended at; their mean number of in-range intra pairs (an oracle diagnostic) is kept
        under `tag` for the flop figure of search_roofline()."""
        qp = O.params_as_fp32(O.default_params())
        qg = O.build_grid(qp, q.protein_xyz, q.protein_type, q.box_center, q.box_size, q.spacing, q.lig_types)
        qL = O.Ligand(q.ligand)
        if gpu_best is not None:
            dg = O.score_batch(qp, qg, qL, np.asarray(gpu_best, np.float64)[:, :7 + qL.T], want_grad=False)[3]
            pairs_in_range[tag] = float(dg["pairs_in_range"].mean())
        init = O.init_poses(q.box_center, q.box_size, qL.T, 2023, system, n_copies)
        t0 = time.perf_counter()
        r = O.search(qp, qg, qL, init, steps, cap, 2023, system)
        dt = time.perf_counter() - t0
        return r["evals"], dt

    def search_roofline(parts, seconds, kernel):
        """SURVEY.md 8(d) "Search configs": the roofline fraction of a search, for information.  parts = [(evaluations,
        ligand, mean in-range pairs)]; flops = evaluations x 8(d)'s per-evaluation formula, so the optimizer's own
        vector algebra (BFGS update, line-search bookkeeping, Philox) counts as overhead, not as work."""
        fl = sum(ev * algorithmic_flops(L.N, L.T, pin, L.P - pin) for ev, L, pin in parts)
        kc = counters.get(kernel, {})
        return {"roofline_frac": fl / seconds / 1e12 / ALU_PEAK_TFLOPS, "achieved_tflops": fl / seconds / 1e12, "kernel": kernel,
                "pairs_in_range_mean": float(np.mean([pin for _, _, pin in parts])),
                "pairs_in_range_source": "oracle diagnostic on the poses the GPU search ended at",
                "achieved_occupancy_pct_ncu": kc.get("achieved_occupancy_pct"),
                "occupancy_source": f"{kc['source']} at commit {kc['commit']}" if kc else None}

    # extras: A1 and A6-A8 next to the headline
    extra.update({"grid_build_ms": float(np.median(t_grid)), "grid_nodes": int(np.prod(grid.dims)) * len(s.lig_types)})
    if not args.no_search:
        s2 = make_system(2, seed=0)
        box2 = dk.make_box(s2.box_center, s2.box_size, s2.spacing)
        lig2 = dk.LigandHandle(s2.ligand)
        grid2 = dk.dock_build_grids(p, s2.protein_xyz, s2.protein_type, box2, s2.lig_types)
        run = lambda: dk.dock_search(p, [grid2], [lig2], [box2], s2.copies, s2.steps, s2.bfgs_cap, 2023)
        run()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        res = run()
        torch.cuda.synchronize()
        t_s = time.perf_counter() - t0
        t0 = time.perf_counter()
        r_h = dk.dock_system_host(p, s2.protein_xyz, s2.protein_type, box2, lig2, s2.lig_types, s2.copies, s2.steps,
                                  s2.bfgs_cap, 2023)
        t_h = time.perf_counter() - t0
        oev, odt = oracle_search_rate(s2, s2.copies, s2.steps, s2.bfgs_cap, gpu_best=res["best_pose"][0].cpu().numpy(), tag="cfg2")
        extra["site_docking"] = {"workload": "configs[2]: 384 copies x 40 steps, BFGS<=300", "search_s": t_s,
                                 "evals": int(res["evals"][0]), "evals_per_s": int(res["evals"][0]) / t_s,
                                 "systems_per_s_search_only": 1.0 / t_s, "end_to_end_host_s": t_h,
                                 "systems_per_s_end_to_end": 1.0 / t_h, "best_e": float(res["topk_e"][0, 0]),
                                 "cpu_baseline": {"kind": "oracle", "cores": O.num_threads(), "sample": "all 384 copies x 40 steps (grid build not included)",
                                                  "search_s": odt, "evals": oev, "evals_per_s": oev / odt, "systems_per_s": 1.0 / odt},
                                 "paper_context": "DSDP 384x40 redocking 0.55 s/system on RTX 2080 SUPER (PAPER.md:108)"}
        extra["site_docking"].update(search_roofline([(int(res["evals"][0]), lig2, pairs_in_range["cfg2"])], t_s, "search_cta_kernel"))
        # the same site docking driven by the paper's Barzilai-Borwein optimizer (NEXT-1), 150 iterations
        pb = dk.dock_default_params()
        pb.optimizer = 1
        runb = lambda: dk.dock_search(pb, [grid2], [lig2], [box2], s2.copies, s2.steps, 150, 2023)
        runb()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rb = runb()
        torch.cuda.synchronize()
        t_b = time.perf_counter() - t0
        extra["site_docking_bb"] = {"workload": "configs[2] with the Barzilai-Borwein optimizer, <=150 iterations", "search_s": t_b,
                                    "evals": int(rb["evals"][0]), "evals_per_s": int(rb["evals"][0]) / t_b,
                                    "systems_per_s_search_only": 1.0 / t_b, "best_e": float(rb["topk_e"][0, 0])}
        extra["site_docking_bb"].update(search_roofline([(int(rb["evals"][0]), lig2, pairs_in_range["cfg2"])], t_b, "search_cta_kernel"))
        # configs[3] oracle baseline: the first two systems of the batch, 32 copies x 40 steps each
        oev = odt = 0.0
        for i, q in enumerate(sys3_keep):
            a, b_ = oracle_search_rate(q, 32, 40, 300, system=i, gpu_best=best3_pose[i], tag=f"cfg3_{i}")
            oev += a
            odt += b_
        # flop figure of the batch: the launch has ONE evaluation counter, so the evaluations are spread evenly over the
        # systems' ligands; the in-range pair FRACTION of the systems the oracle looked at stands in for the others
        frac3 = float(np.mean([pairs_in_range[f"cfg3_{i}"] / max(1, lg[i].P) for i in range(len(sys3_keep))]))
        extra["screening"].update(search_roofline([(ev3_rank0 / len(lg), L_, frac3 * L_.P) for L_ in lg], t_3_rank0, "search_kernel"))
        extra["screening"]["roofline_note"] = (f"rank 0's {len(lg)} systems, evaluations spread evenly over them; in-range pair "
                                               f"fraction {frac3:.3f} from the first {len(sys3_keep)}")
        extra["screening"]["cpu_baseline"] = {"kind": "oracle", "cores": O.num_threads(),
                                              "sample": f"first {len(sys3_keep)} systems, 32 of 128 copies x 40 steps each (grid build not included)",
                                              "search_s": odt, "evals": int(oev), "evals_per_s": oev / odt,
                                              "systems_per_s_scaled": len(sys3_keep) / (odt * 128 / 32)}
        # configs[4]: large blind box, 161^3 x 8 maps (1.07 GB gather image), 2048 copies x 80 steps, N = 60, T = 15
        s4 = make_system(4, seed=0)
        box4 = dk.make_box(s4.box_center, s4.box_size, s4.spacing)
        lig4 = dk.LigandHandle(s4.ligand)
        grid4 = dk.dock_build_grids(p, s4.protein_xyz, s4.protein_type, box4, s4.lig_types)   # warm-up
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        grid4 = dk.dock_build_grids(p, s4.protein_xyz, s4.protein_type, box4, s4.lig_types)
        torch.cuda.synchronize()
        t_g4 = time.perf_counter() - t0
        run4 = lambda: dk.dock_search(p, [grid4], [lig4], [box4], s4.copies, s4.steps, s4.bfgs_cap, 2023)
        dk.dock_search(p, [grid4], [lig4], [box4], 64, 1, 10, 2023)                             # warm-up: module load, smem attribute
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r4 = run4()
        torch.cuda.synchronize()
        t_4 = time.perf_counter() - t0
        oev, odt = oracle_search_rate(s4, 32, s4.steps, s4.bfgs_cap, gpu_best=r4["best_pose"][0].cpu().numpy(), tag="cfg4")
        extra["large_blind_box"] = {"workload": "configs[4]: 8000 atoms, 161^3 x 8 maps, 2048 copies x 80 steps, BFGS<=300",
                                    "search_s": t_4, "grid_build_s": t_g4, "evals": int(r4["evals"][0]),
                                    "evals_per_s": int(r4["evals"][0]) / t_4, "systems_per_s_with_grid": 1.0 / (t_4 + t_g4),
                                    "best_e": float(r4["topk_e"][0, 0]),
                                    "cpu_baseline": {"kind": "oracle", "cores": O.num_threads(),
                                                     "sample": "first 32 of 2048 copies x 80 steps (grid build not included)",
                                                     "search_s": odt, "evals": oev, "evals_per_s": oev / odt,
                                                     "systems_per_s_scaled": 1.0 / (odt * 2048 / 32)}}
        extra["large_blind_box"].update(search_roofline([(int(r4["evals"][0]), lig4, pairs_in_range["cfg4"])], t_4, "search_kernel"))
        del grid4
    line["extra"] = extra
    return line


def kernel_counters() -> dict:
    """ncu-only counters (DRAM bytes per launch, achieved occupancy) of the committed captures: profiles/kernel_counters.json,
    each entry with the capture file and the commit it was taken at.  {} if the file is missing (the fields print as null)."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "kernel_counters.json")
    try:
        with open(path) as f:
            return {k: v for k, v in json.load(f).items() if isinstance(v, dict)}
    except (OSError, ValueError):
        return {}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-sample", type=int, default=1048576, help="poses the CPU oracle scores per step")
    ap.add_argument("--no-flush", action="store_true")
    ap.add_argument("--no-search", action="store_true")
    ap.add_argument("--score-kernel", type=int, default=0, choices=[-1, 0, 1, 2],
                    help="dock_params.score_kernel for the headline step: 0/1 generic (the library default, and the default here), "
                         "2 specialised at run time (compilation outside the timed region), -1 = 2 if NVRTC is available, else generic")
    ap.add_argument("--screen-systems", type=int, default=256, help="systems of the configs[3] screening batch (256 = the config)")
    args = ap.parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)))
        return
    line = run_ours(args)
    if line:
        print(json.dumps(line))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
