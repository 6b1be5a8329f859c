"""ctypes binding of the CPU oracle (oracle/dock_oracle.c).

TEST INFRASTRUCTURE ONLY.  May be imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py -- never by paper_2303_09916_b200/.
It imports nothing from the CUDA package.  All numerics are float64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "dock_oracle.c")
_HDR = os.path.join(_HERE, "dock_oracle.h")
ORC_MAX_TYPES = 32


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math, no contraction)."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _SO
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-o", _SO, _SRC, "-lm"]
    subprocess.check_call(cmd)
    return _SO


_SO_COUNT = os.path.join(_HERE, "liboracle_count.so")
_lib_count = None
OP_KINDS = ("add_sub", "mul", "div", "compare", "sqrt", "exp", "sin_cos", "floor_abs_min")


def build_counted(force: bool = False) -> str:
    """Compile dock_oracle.c, unchanged, with the operation-counting scalar of opcount.hpp in place of double."""
    srcs = [_SRC, _HDR, os.path.join(_HERE, "opcount.hpp"), os.path.join(_HERE, "dock_oracle_count.cpp")]
    if not force and os.path.exists(_SO_COUNT) and os.path.getmtime(_SO_COUNT) >= max(os.path.getmtime(f) for f in srcs):
        return _SO_COUNT
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-w",
                           "-o", _SO_COUNT, srcs[3], "-lm"], cwd=_HERE)
    return _SO_COUNT


def count_eval_ops(p, g, L, poses, want_grad: bool = True) -> dict:
    """Mean floating-point operations of ONE score(+gradient) evaluation over `poses`, counted on the oracle's own
    statements (one per add/sub, mul, div, compare, sqrt, exp, sin/cos, floor/fabs/fmin; nothing fused).  Single-threaded."""
    global _lib_count
    if _lib_count is None:
        _lib_count = C.CDLL(build_counted())
        _lib_count.orc_eval.restype = C.c_double
    poses = _f64(poses).reshape(-1, 7 + L.T)
    terms = np.zeros(3)
    grad = np.zeros(6 + L.T)
    _lib_count.orc_count_reset()
    for k in range(poses.shape[0]):
        row = np.ascontiguousarray(poses[k])
        _lib_count.orc_eval(C.byref(p), C.byref(g.c), C.byref(L.c), _p(row), _p(terms), _p(grad) if want_grad else None, None)
    out = (C.c_uint64 * len(OP_KINDS))()
    _lib_count.orc_count_get(out)
    n = max(1, poses.shape[0])
    per = {k: out[i] / n for i, k in enumerate(OP_KINDS)}
    per["total"] = float(sum(per.values()))
    return per


class Params(C.Structure):
    _fields_ = [
        ("n_types", C.c_int),
        ("radius", C.c_double * ORC_MAX_TYPES),
        ("hydrophobic", C.c_int * ORC_MAX_TYPES),
        ("donor", C.c_int * ORC_MAX_TYPES),
        ("acceptor", C.c_int * ORC_MAX_TYPES),
        ("w", C.c_double * 5),
        ("cutoff", C.c_double),
        ("k_wall", C.c_double),
        ("t_mc", C.c_double),
        ("amp_trans", C.c_double),
        ("amp_rot", C.c_double),
        ("bfgs_c1", C.c_double),
        ("bfgs_shrink", C.c_double),
        ("bfgs_max_trials", C.c_int),
        ("bfgs_gtol", C.c_double),
        ("bfgs_curv_eps", C.c_double),
        ("cluster_rmsd", C.c_double),
        ("topk", C.c_int),
        ("optimizer", C.c_int),
        ("bb_step", C.c_double),
        ("bb_fallback", C.c_double),
    ]


class _Ligand(C.Structure):
    _fields_ = [
        ("N", C.c_int), ("T", C.c_int), ("P", C.c_int),
        ("ref", C.c_void_p), ("type", C.c_void_p), ("frag", C.c_void_p),
        ("tors_parent", C.c_void_p), ("tors_a", C.c_void_p), ("tors_b", C.c_void_p),
        ("pairs", C.c_void_p),
    ]


class _Grid(C.Structure):
    _fields_ = [
        ("dims", C.c_int * 3),
        ("origin", C.c_double * 3),
        ("h", C.c_double),
        ("n_maps", C.c_int),
        ("type_to_map", C.c_int * ORC_MAX_TYPES),
        ("data", C.c_void_p),
        ("gdata", C.c_void_p),
    ]


class Diag(C.Structure):
    _fields_ = [("face_margin", C.c_double), ("kink_margin", C.c_double), ("cutoff_margin", C.c_double),
                ("pairs_in_range", C.c_int), ("atoms_outside", C.c_int)]


class StepRec(C.Structure):
    _fields_ = [("e_cur", C.c_double), ("e_cand", C.c_double), ("u", C.c_double),
                ("accept", C.c_int), ("iters", C.c_int), ("evals", C.c_int)]


ORC_MAX_TRIALS = 64
EXIT_GTOL, EXIT_CAP, EXIT_LINESEARCH = 1, 2, 3
ITER_DTYPE = np.dtype([("status", "i4"), ("reset", "i4"), ("fresh_in", "i4"), ("fresh_out", "i4"), ("trials", "i4"),
                       ("updated", "i4"), ("f", "f8"), ("gnorm", "f8"), ("gp", "f8"), ("alpha0", "f8"), ("alpha", "f8"),
                       ("f_new", "f8"), ("armijo_margin", "f8", (ORC_MAX_TRIALS,)), ("curv_margin", "f8"),
                       ("min_cutoff_margin", "f8")])
assert ITER_DTYPE.itemsize == 6 * 4 + 8 * (6 + ORC_MAX_TRIALS + 2)

BB_DTYPE = np.dtype([("status", "i4"), ("branch", "i4"), ("capped", "i4"), ("_pad", "i4"), ("f", "f8"), ("gnorm", "f8"),
                     ("alpha", "f8"), ("f_new", "f8"), ("sy_margin", "f8"), ("cap_margin", "f8"), ("min_cutoff_margin", "f8")])

STEP_DTYPE = np.dtype([("e_cur", "f8"), ("e_cand", "f8"), ("u", "f8"),
                       ("accept", "i4"), ("iters", "i4"), ("evals", "i4"), ("_pad", "i4")])
DIAG_DTYPE = np.dtype([("face_margin", "f8"), ("kink_margin", "f8"), ("cutoff_margin", "f8"),
                       ("pairs_in_range", "i4"), ("atoms_outside", "i4")])
assert STEP_DTYPE.itemsize == C.sizeof(StepRec)
assert DIAG_DTYPE.itemsize == C.sizeof(Diag)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_pair.restype = C.c_double
        _lib.orc_eval.restype = C.c_double
        _lib.orc_local_opt.restype = C.c_double
        _lib.orc_mc_uniform.restype = C.c_double
        _lib.orc_search_copy.restype = C.c_double
        _lib.orc_search.restype = C.c_int64
        _lib.orc_rmsd.restype = C.c_double
        _lib.orc_topk.restype = C.c_int
        _lib.orc_mc_perturb.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_local_opt_ex.restype = C.c_double
        _lib.orc_bfgs_step.restype = C.c_int
        _lib.orc_grid_cutoff_flags.restype = C.c_int64
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def default_params() -> Params:
    p = Params()
    lib().orc_default_params(C.byref(p))
    return p


def params_as_fp32(p: Params) -> Params:
    """The CUDA library's dock_params are fp32; widen those fp32 values back to double so
    both sides start from the same numbers (S14: 'the oracle widens to double')."""
    q = Params()
    C.memmove(C.byref(q), C.byref(p), C.sizeof(Params))
    for i in range(ORC_MAX_TYPES):
        q.radius[i] = float(np.float32(p.radius[i]))
    for i in range(5):
        q.w[i] = float(np.float32(p.w[i]))
    for name in ("cutoff", "k_wall", "t_mc", "amp_trans", "amp_rot", "bfgs_c1", "bfgs_shrink",
                 "bfgs_gtol", "bfgs_curv_eps", "cluster_rmsd", "bb_step", "bb_fallback"):
        setattr(q, name, float(np.float32(getattr(p, name))))
    return q


class round_eval_fp32:
    """Context manager for the chaos-ceiling diagnostic: inside, the optimizers see the oracle's energy and gradient
    rounded to a (24 - drop_bits)-bit significand (dock_oracle.c: orc_diag_round_eval_fp32): 0 = fp32 correctly
    rounded, 3 = an fp32 result off by up to 4 ulp.  Off outside; nothing else may switch it on."""

    def __init__(self, drop_bits: int = 3):
        self.drop_bits = int(drop_bits)

    def __enter__(self):
        lib().orc_diag_round_eval_fp32(self.drop_bits)

    def __exit__(self, *exc):
        lib().orc_diag_round_eval_fp32(-1)
        return False


def num_threads() -> int:
    return int(lib().orc_num_threads())


def pair(p: Params, t1: int, t2: int, r: float):
    d = C.c_double()
    e = lib().orc_pair(C.byref(p), int(t1), int(t2), C.c_double(r), C.byref(d))
    return float(e), float(d.value)


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


class Ligand:
    """Keeps the numpy arrays alive for the C struct."""

    def __init__(self, lig):
        self.ref = _f64(lig.ref_xyz)
        self.type = _i32(lig.type)
        self.frag = _i32(lig.frag)
        self.tors_parent = _i32(lig.tors_parent)
        self.tors_a = _i32(lig.tors_a)
        self.tors_b = _i32(lig.tors_b)
        self.pairs = _i32(lig.pairs).reshape(-1, 2)
        self.N, self.T, self.P = self.ref.shape[0], self.tors_a.shape[0], self.pairs.shape[0]
        self.c = _Ligand(self.N, self.T, self.P, _p(self.ref), _p(self.type), _p(self.frag),
                         _p(self.tors_parent), _p(self.tors_a), _p(self.tors_b), _p(self.pairs))


class Grid:
    def __init__(self, dims, origin, h, lig_types, data, gdata=None):
        self.dims = tuple(int(d) for d in dims)
        self.origin = np.array(origin, dtype=np.float64)
        self.h = float(h)
        self.lig_types = list(lig_types)
        self.data = _f64(data)
        g = _Grid()
        for c in range(3):
            g.dims[c] = self.dims[c]
            g.origin[c] = self.origin[c]
        g.h = self.h
        g.n_maps = len(self.lig_types)
        for t in range(ORC_MAX_TYPES):
            g.type_to_map[t] = -1
        for m, t in enumerate(self.lig_types):
            g.type_to_map[t] = m
        g.data = _p(self.data)
        self.gdata = None if gdata is None else _f64(gdata)
        g.gdata = None if gdata is None else _p(self.gdata)
        self.c = g

    @property
    def gmaps(self):
        """NEXT-2 (eq. 4): per-vertex gradients [n_maps][3][nz][ny][nx], or None."""
        if self.gdata is None:
            return None
        nx, ny, nz = self.dims
        return self.gdata.reshape(len(self.lig_types), 3, nz, ny, nx)

    @property
    def maps(self):
        nx, ny, nz = self.dims
        return self.data.reshape(len(self.lig_types), nz, ny, nx)


def grid_geometry(center, size, h):
    c = (C.c_double * 3)(*[float(x) for x in center])
    s = (C.c_double * 3)(*[float(x) for x in size])
    dims = (C.c_int * 3)()
    org = (C.c_double * 3)()
    lib().orc_grid_geometry(c, s, C.c_double(h), dims, org)
    return [int(d) for d in dims], [float(o) for o in org]


def build_grid(p: Params, pxyz, ptype, center, size, h, lig_types, grad=False) -> Grid:
    dims, org = grid_geometry(center, size, h)
    pxyz = _f64(pxyz)
    ptype = _i32(ptype)
    lt = _i32(lig_types)
    G = np.zeros(len(lig_types) * dims[0] * dims[1] * dims[2], dtype=np.float64)
    lib().orc_build_grid(C.byref(p), int(pxyz.shape[0]), _p(pxyz), _p(ptype),
                         (C.c_int * 3)(*dims), (C.c_double * 3)(*org), C.c_double(h),
                         len(lig_types), _p(lt), _p(G))
    GD = None
    if grad:                                               # NEXT-2: eq. 4's per-vertex gradients
        GD = np.zeros(3 * len(lig_types) * dims[0] * dims[1] * dims[2], dtype=np.float64)
        lib().orc_build_grid_grad(C.byref(p), int(pxyz.shape[0]), _p(pxyz), _p(ptype),
                                  (C.c_int * 3)(*dims), (C.c_double * 3)(*org), C.c_double(h),
                                  len(lig_types), _p(lt), _p(GD))
    return Grid(dims, org, h, lig_types, G, GD)


def grid_cutoff_flags(p: Params, pxyz, g: Grid, margin: float = 1e-5) -> np.ndarray:
    """Diagnostic: bool [nz, ny, nx], True where some atom lies within `margin` of the node's cutoff sphere."""
    pxyz = _f64(pxyz)
    nx, ny, nz = g.dims
    flags = np.zeros(nx * ny * nz, dtype=np.uint8)
    lib().orc_grid_cutoff_flags(int(pxyz.shape[0]), _p(pxyz), (C.c_int * 3)(*g.dims), (C.c_double * 3)(*g.origin),
                                C.c_double(g.h), C.c_double(p.cutoff), C.c_double(margin), _p(flags))
    return flags.reshape(nz, ny, nx).astype(bool)


def coords(L: Ligand, pose) -> np.ndarray:
    pose = _f64(pose)
    x = np.zeros((L.N, 3), dtype=np.float64)
    lib().orc_coords(C.byref(L.c), _p(pose), _p(x))
    return x


def evaluate(p: Params, g: Grid, L: Ligand, pose, want_grad=True):
    pose = _f64(pose)
    terms = np.zeros(3)
    grad = np.zeros(6 + L.T) if want_grad else None
    d = Diag()
    e = lib().orc_eval(C.byref(p), C.byref(g.c), C.byref(L.c), _p(pose), _p(terms), _p(grad), C.byref(d))
    return float(e), terms, grad, d


def score_batch(p: Params, g: Grid, L: Ligand, poses, want_grad=True):
    poses = _f64(poses).reshape(-1, 7 + L.T)
    n = poses.shape[0]
    E = np.zeros(n)
    grad = np.zeros((n, 6 + L.T)) if want_grad else None
    terms = np.zeros((n, 3))
    diag = np.zeros(n, dtype=DIAG_DTYPE)
    lib().orc_score_batch(C.byref(p), C.byref(g.c), C.byref(L.c), C.c_int64(n), _p(poses),
                          _p(E), _p(grad), _p(terms), _p(diag))
    return E, grad, terms, diag


def grad_cond(p: Params, g: Grid, L: Ligand, poses) -> np.ndarray:
    """Diagnostic: conditioning scale A[n, 6+T] of each gradient component (sum of |terms|)."""
    poses = _f64(poses).reshape(-1, 7 + L.T)
    n = poses.shape[0]
    A = np.zeros((n, 6 + L.T))
    lib().orc_grad_cond_batch(C.byref(p), C.byref(g.c), C.byref(L.c), C.c_int64(n), _p(poses), _p(A))
    return A


def pose_add(T: int, pose, s) -> np.ndarray:
    pose, s = _f64(pose), _f64(s)
    out = np.zeros(7 + T)
    lib().orc_pose_add(int(T), _p(pose), _p(s), _p(out))
    return out


def local_opt(p: Params, g: Grid, L: Ligand, pose, cap: int):
    pose = _f64(pose)
    out = np.zeros(7 + L.T)
    it, ne = C.c_int(), C.c_int()
    e = lib().orc_local_opt(C.byref(p), C.byref(g.c), C.byref(L.c), int(cap), _p(pose), _p(out),
                            C.byref(it), C.byref(ne))
    return float(e), out, it.value, ne.value


def local_opt_ex(p: Params, g: Grid, L: Ligand, pose, cap: int, max_recs: int = 0):
    """local_opt plus the exit reason and (BFGS) the per-iteration decision records."""
    pose = _f64(pose)
    out = np.zeros(7 + L.T)
    it, ne, why = C.c_int(), C.c_int(), C.c_int()
    recs = np.zeros(max(1, max_recs), dtype=ITER_DTYPE)
    e = lib().orc_local_opt_ex(C.byref(p), C.byref(g.c), C.byref(L.c), int(cap), _p(pose), _p(out),
                               C.byref(it), C.byref(ne), C.byref(why), _p(recs) if max_recs else None, int(max_recs))
    started = it.value + (0 if why.value == EXIT_CAP else 1)          # iterations started = records written
    return float(e), out, it.value, ne.value, why.value, recs[:min(max_recs, started)]


def local_opt_batch(p: Params, g: Grid, L: Ligand, poses, cap: int):
    """OpenMP over poses.  Returns (e [n], pose [n,7+T], info [n,3] = iters, evals, exit reason)."""
    poses = _f64(poses).reshape(-1, 7 + L.T)
    n = poses.shape[0]
    out = np.zeros_like(poses)
    e = np.zeros(n)
    info = np.zeros((n, 3), dtype=np.int32)
    lib().orc_local_opt_batch(C.byref(p), C.byref(g.c), C.byref(L.c), int(cap), C.c_int64(n), _p(poses), _p(out), _p(e), _p(info))
    return e, out, info


def bfgs_step_batch(p: Params, g: Grid, L: Ligand, x, H, fresh, grad=None):
    """One O8 iteration from each given state (x [m,7+T], H [m,n,n], fresh [m], optional gradient [m,n] at x).
    Returns (recs, x_new, H_new)."""
    n = 6 + L.T
    x = _f64(x).reshape(-1, 7 + L.T)
    m = x.shape[0]
    H = _f64(H).reshape(m, n, n)
    fresh = _i32(fresh).reshape(m)
    grad = None if grad is None else _f64(grad).reshape(m, n)
    recs = np.zeros(m, dtype=ITER_DTYPE)
    x_new, H_new = np.zeros_like(x), np.zeros_like(H)
    lib().orc_bfgs_step_batch(C.byref(p), C.byref(g.c), C.byref(L.c), C.c_int64(m), _p(x), _p(grad), _p(H), _p(fresh),
                              _p(recs), _p(x_new), _p(H_new))
    return recs, x_new, H_new


def bb_step_batch(p: Params, g: Grid, L: Ligand, x, grad, s_prev, y_prev, first):
    """One O8' iteration from each given state.  Returns (recs, x_new)."""
    n = 6 + L.T
    x = _f64(x).reshape(-1, 7 + L.T)
    m = x.shape[0]
    grad = None if grad is None else _f64(grad).reshape(m, n)
    s_prev, y_prev = _f64(s_prev).reshape(m, n), _f64(y_prev).reshape(m, n)
    first = _i32(first).reshape(m)
    recs = np.zeros(m, dtype=BB_DTYPE)
    x_new = np.zeros_like(x)
    lib().orc_bb_step_batch(C.byref(p), C.byref(g.c), C.byref(L.c), C.c_int64(m), _p(x), _p(grad), _p(s_prev), _p(y_prev),
                            _p(first), _p(recs), _p(x_new))
    return recs, x_new


def replay_steps(p: Params, g: Grid, L: Ligand, cap: int, seed: int, system: int, pre_pose, copy, step):
    """Teacher-forced replay of recorded MC steps (level 3'), OpenMP over records."""
    pre = _f64(pre_pose).reshape(-1, 7 + L.T)
    n = pre.shape[0]
    copy, step = _i32(copy).reshape(n), _i32(step).reshape(n)
    out = dict(e_cur=np.zeros(n), cur_cutoff_margin=np.zeros(n), kind=np.zeros(n, np.int32), e_cand=np.zeros(n),
               u=np.zeros(n), accept=np.zeros(n, np.int32), iters=np.zeros(n, np.int32), evals=np.zeros(n, np.int32))
    lib().orc_replay_steps(C.byref(p), C.byref(g.c), C.byref(L.c), int(cap), C.c_uint64(seed), C.c_uint32(system),
                           C.c_int64(n), _p(pre), _p(copy), _p(step), _p(out["e_cur"]), _p(out["cur_cutoff_margin"]),
                           _p(out["kind"]), _p(out["e_cand"]), _p(out["u"]), _p(out["accept"]), _p(out["iters"]),
                           _p(out["evals"]))
    return out


def init_pose(center, size, T, seed, system, copy) -> np.ndarray:
    out = np.zeros(7 + T)
    lib().orc_init_pose((C.c_double * 3)(*[float(x) for x in center]),
                        (C.c_double * 3)(*[float(x) for x in size]), int(T),
                        C.c_uint64(seed), C.c_uint32(system), C.c_uint32(copy), _p(out))
    return out


def init_poses_site(center, size, T, seed, system, copies, site_xyz, radius) -> np.ndarray:
    """NEXT-3: initial poses with the translation restrained to box ∩ union of balls (reading S22)."""
    site = _f64(site_xyz).reshape(-1, 3)
    out = np.zeros((copies, 7 + T))
    for c in range(copies):
        row = np.zeros(7 + T)
        lib().orc_init_pose_site((C.c_double * 3)(*[float(x) for x in center]),
                                 (C.c_double * 3)(*[float(x) for x in size]), int(T),
                                 C.c_uint64(seed), C.c_uint32(system), C.c_uint32(c),
                                 int(site.shape[0]), _p(site), C.c_double(radius), _p(row))
        out[c] = row
    return out


def init_poses(center, size, T, seed, system, copies) -> np.ndarray:
    return np.stack([init_pose(center, size, T, seed, system, c) for c in range(copies)])


def mc_perturb(p: Params, T, seed, system, copy, step, pose):
    pose = _f64(pose)
    out = np.zeros(7 + T)
    kind = lib().orc_mc_perturb(C.byref(p), int(T), C.c_uint64(seed), C.c_uint32(system),
                                C.c_uint32(copy), C.c_uint32(step), _p(pose), _p(out))
    return int(kind), out


def mc_uniform(seed, system, copy, step) -> float:
    return float(lib().orc_mc_uniform(C.c_uint64(seed), C.c_uint32(system), C.c_uint32(copy), C.c_uint32(step)))


def search(p: Params, g: Grid, L: Ligand, init, steps, cap, seed, system=0, want_trace=True):
    init = _f64(init).reshape(-1, 7 + L.T)
    copies = init.shape[0]
    best_pose = np.zeros((copies, 7 + L.T))
    best_e = np.zeros(copies)
    tp = np.zeros((copies, steps, 7 + L.T)) if want_trace else None
    tr = np.zeros((copies, steps), dtype=STEP_DTYPE) if want_trace else None
    ir = np.zeros(copies, dtype=STEP_DTYPE)
    evals = lib().orc_search(C.byref(p), C.byref(g.c), C.byref(L.c), int(copies), int(steps), int(cap),
                             C.c_uint64(seed), C.c_uint32(system), _p(init), _p(best_pose), _p(best_e),
                             _p(tp), _p(tr), _p(ir))
    return dict(best_pose=best_pose, best_e=best_e, trace_pose=tp, trace=tr, init_rec=ir, evals=int(evals))


def rmsd(L: Ligand, a, b) -> float:
    a, b = _f64(a), _f64(b)
    return float(lib().orc_rmsd(C.byref(L.c), _p(a), _p(b)))


def topk(p: Params, L: Ligand, poses, e, k: int, rmsd_min: float):
    poses = _f64(poses).reshape(-1, 7 + L.T)
    e = _f64(e)
    out = np.full(k, -1, dtype=np.int32)
    n = lib().orc_topk(C.byref(p), C.byref(L.c), int(poses.shape[0]), _p(poses), _p(e), int(k),
                       C.c_double(rmsd_min), _p(out))
    return int(n), out


_OBJ_FN = C.CFUNCTYPE(C.c_double, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double))
_ADD_FN = C.CFUNCTYPE(None, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double))
_OBS_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_double),
                      C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int)


def bfgs_generic(p: Params, x0, fn, cap: int, observer=None):
    """Run the oracle's O8 optimizer on a Python objective fn(x)->(f, grad) with the
    Euclidean retraction x+s.  observer(it, f, H, s, y, updated) is optional.  Pin tests only."""
    x0 = _f64(x0)
    n = x0.shape[0]

    def _fn(_ctx, xp, gp):
        x = np.ctypeslib.as_array(xp, shape=(n,))
        f, g = fn(x.copy())
        for k in range(n):
            gp[k] = float(g[k])
        return float(f)

    def _add(_ctx, xp, sp, op):
        for k in range(n):
            op[k] = xp[k] + sp[k]

    def _obs(_ctx, it, f, Hp, sp, yp, updated):
        if observer is not None:
            observer(int(it), float(f), np.ctypeslib.as_array(Hp, shape=(n, n)).copy(),
                     np.ctypeslib.as_array(sp, shape=(n,)).copy(),
                     np.ctypeslib.as_array(yp, shape=(n,)).copy(), bool(updated))

    out = np.zeros(n)
    it, ne = C.c_int(), C.c_int()
    l = lib()
    l.orc_bfgs.restype = C.c_double
    f = l.orc_bfgs(C.byref(p), n, n, int(cap), _p(x0), _OBJ_FN(_fn), _ADD_FN(_add), None, _p(out),
                   C.byref(it), C.byref(ne), _OBS_FN(_obs), None, None, None, 0)
    return float(f), out, it.value, ne.value


def bb_generic(p: Params, x0, fn, cap: int, observer=None):
    """Run the oracle's O8' Barzilai-Borwein optimizer on a Python objective fn(x)->(f, grad) with the
    Euclidean retraction x+s.  observer(it, f, s, y) is optional.  Pin tests only."""
    x0 = _f64(x0)
    n = x0.shape[0]

    def _fn(_ctx, xp, gp):
        x = np.ctypeslib.as_array(xp, shape=(n,))
        f, g = fn(x.copy())
        for k in range(n):
            gp[k] = float(g[k])
        return float(f)

    def _add(_ctx, xp, sp, op):
        for k in range(n):
            op[k] = xp[k] + sp[k]

    def _obs(_ctx, it, f, Hp, sp, yp, updated):
        if observer is not None:
            observer(int(it), float(f), np.ctypeslib.as_array(sp, shape=(n,)).copy(),
                     np.ctypeslib.as_array(yp, shape=(n,)).copy())

    out = np.zeros(n)
    it, ne = C.c_int(), C.c_int()
    l = lib()
    l.orc_bb.restype = C.c_double
    f = l.orc_bb(C.byref(p), n, n, int(cap), _p(x0), _OBJ_FN(_fn), _ADD_FN(_add), None, _p(out),
                 C.byref(it), C.byref(ne), _OBS_FN(_obs), None, None)
    return float(f), out, it.value, ne.value
