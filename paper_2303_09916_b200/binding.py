"""Thin ctypes binding of include/dock.h (argument marshalling only).

Every step of the hot path runs inside libdock_b200.so's CUDA kernels; PyTorch is used here only
to own device memory and to supply the CUDA stream.  There is no CPU fallback: if the shared
library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libdock_b200.so")

DOCK_MAX_XS_TYPES = 32
DOCK_MAX_TORSIONS = 32
DOCK_MAX_ATOMS = 128
DOCK_TRACE_HEADER = 8
DOCK_ITER_HEADER = 12
DOCK_EXIT_GTOL, DOCK_EXIT_CAP, DOCK_EXIT_LINESEARCH = 1, 2, 3
DOCK_OK, DOCK_EINVAL, DOCK_EWORKSPACE, DOCK_ECUDA, DOCK_ECAPACITY = 0, -1, -2, -3, -4
DOCK_TOPK_FIXED_BYTES = 65536

EXPORTS = [
    "dock_default_params", "dock_grid_dims", "dock_grid_bytes", "dock_build_grids", "dock_build_grids_batch", "dock_score_batch",
    "dock_score_batch_host", "dock_local_opt_batch", "dock_local_opt_trace", "dock_init_poses", "dock_init_poses_site",
    "dock_search", "dock_topk", "dock_topk_fixed", "dock_system_host", "dock_probe_peaks", "dock_last_cuda_error", "dock_version",
    "dock_launch_count", "dock_score_jit_source", "dock_score_jit_compile", "dock_score_jit_log", "dock_score_jit_cache",
]


class DockError(RuntimeError):
    pass


class dock_params(C.Structure):
    _fields_ = [
        ("n_types", C.c_int32),
        ("radius", C.c_float * DOCK_MAX_XS_TYPES),
        ("hydrophobic", C.c_int32 * DOCK_MAX_XS_TYPES),
        ("donor", C.c_int32 * DOCK_MAX_XS_TYPES),
        ("acceptor", C.c_int32 * DOCK_MAX_XS_TYPES),
        ("w", C.c_float * 5),
        ("cutoff", C.c_float), ("k_wall", C.c_float), ("t_mc", C.c_float),
        ("amp_trans", C.c_float), ("amp_rot", C.c_float),
        ("bfgs_c1", C.c_float), ("bfgs_shrink", C.c_float), ("bfgs_max_trials", C.c_int32),
        ("bfgs_gtol", C.c_float), ("bfgs_curv_eps", C.c_float),
        ("cluster_rmsd", C.c_float), ("topk", C.c_int32),
        ("optimizer", C.c_int32), ("bb_step", C.c_float), ("bb_fallback", C.c_float), ("grad_mode", C.c_int32),
        ("search_kernel", C.c_int32), ("score_kernel", C.c_int32),
    ]


class dock_box(C.Structure):
    _fields_ = [("center", C.c_float * 3), ("size", C.c_float * 3), ("spacing", C.c_float)]


class dock_protein(C.Structure):
    _fields_ = [("n", C.c_int32), ("xyz", C.c_void_p), ("type", C.c_void_p)]


class dock_ligand(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("T", C.c_int32), ("P", C.c_int32),
        ("ref_xyz", C.c_void_p), ("type", C.c_void_p), ("atom_fragment", C.c_void_p),
        ("tors_parent", C.c_void_p), ("tors_a", C.c_void_p), ("tors_b", C.c_void_p), ("pairs", C.c_void_p),
    ]


class dock_grid(C.Structure):
    _fields_ = [
        ("dims", C.c_int32 * 3), ("origin", C.c_float * 3), ("spacing", C.c_float),
        ("n_maps", C.c_int32), ("type_to_map", C.c_int32 * DOCK_MAX_XS_TYPES), ("data_dev", C.c_void_p),
        ("packed_dev", C.c_void_p), ("n_channels", C.c_int32), ("quad_dev", C.c_void_p),
    ]


_lib = None


def load_library(path: Optional[str] = None):
    """dlopen libdock_b200.so (built in-tree by build.py).  Raises if it is missing."""
    global _lib
    if _lib is None:
        path = path or _LIB_PATH
        if not os.path.exists(path):
            raise DockError(f"{path} not found: run `python -m paper_2303_09916_b200.build` "
                            "(there is no CPU fallback)")
        _lib = C.CDLL(path)
        _lib.dock_version.restype = C.c_char_p
        _lib.dock_score_jit_log.restype = C.c_char_p
        _lib.dock_launch_count.restype = C.c_uint64
        _lib.dock_grid_bytes.restype = C.c_size_t
    return _lib


def _check(rc: int, what: str):
    if rc == DOCK_OK:
        return
    names = {DOCK_EINVAL: "DOCK_EINVAL", DOCK_EWORKSPACE: "DOCK_EWORKSPACE", DOCK_ECUDA: "DOCK_ECUDA",
             DOCK_ECAPACITY: "DOCK_ECAPACITY"}
    extra = ""
    if rc == DOCK_ECUDA:
        extra = f" (cudaError {load_library().dock_last_cuda_error()})"
    raise DockError(f"{what} failed: {names.get(rc, rc)}{extra}")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise DockError("no CUDA device: the docking hot path has no CPU fallback")
    return torch


def _stream_obj(stream=None):
    return stream if stream is not None else _torch().cuda.current_stream()


def _stream(stream=None) -> C.c_void_p:
    return C.c_void_p(_stream_obj(stream).cuda_stream)


def _ptr(t) -> C.c_void_p:
    return C.c_void_p(0 if t is None else t.data_ptr())


def _np_ptr(a: Optional[np.ndarray]) -> C.c_void_p:
    return C.c_void_p(0) if a is None else a.ctypes.data_as(C.c_void_p)


class _Workspace:
    """Grow-only device scratch buffers (torch uint8 tensors) reused across calls, ONE PER (device, stream).

    The library stages ligand tables, system descriptors and cell lists in the workspace and returns without
    synchronising, so a kernel still in flight on stream A must never see a later call on stream B overwrite them:
    calls on different streams get different buffers; calls on one stream are ordered by the stream.  When a buffer
    is replaced by a larger one the old tensor is handed to the caching allocator with record_stream, so its memory
    is not reused before the work queued on that stream has finished."""

    def __init__(self):
        self.bufs = {}

    def get(self, nbytes: int, stream=None):
        torch = _torch()
        st = _stream_obj(stream)
        key = (torch.cuda.current_device(), int(st.cuda_stream))
        buf = self.bufs.get(key)
        if buf is None or buf.numel() < nbytes:
            if buf is not None:
                buf.record_stream(st)
            buf = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device="cuda")
            self.bufs[key] = buf
        return buf


_ws = _Workspace()


def score_jit_cache(new_limit: int = -1):
    """(limit before the call, cached specialised kernels); new_limit >= 1 sets the per-device limit (dock.h)."""
    old, n = C.c_int32(0), C.c_int32(0)
    _check(load_library().dock_score_jit_cache(int(new_limit), C.byref(old), C.byref(n)), "dock_score_jit_cache")
    return int(old.value), int(n.value)


def launch_count() -> int:
    return int(load_library().dock_launch_count())


def dock_default_params() -> dock_params:
    p = dock_params()
    _check(load_library().dock_default_params(C.byref(p)), "dock_default_params")
    return p


def make_box(center, size, spacing) -> dock_box:
    b = dock_box()
    for c in range(3):
        b.center[c] = float(center[c])
        b.size[c] = float(size[c])
    b.spacing = float(spacing)
    return b


class LigandHandle:
    """Host arrays (fp32 / int32) + the dock_ligand struct pointing at them."""

    def __init__(self, lig):
        self.ref = np.ascontiguousarray(lig.ref_xyz, dtype=np.float32)
        self.type = np.ascontiguousarray(lig.type, dtype=np.int32)
        self.frag = np.ascontiguousarray(lig.frag, dtype=np.int32)
        self.tors_parent = np.ascontiguousarray(lig.tors_parent, dtype=np.int32)
        self.tors_a = np.ascontiguousarray(lig.tors_a, dtype=np.int32)
        self.tors_b = np.ascontiguousarray(lig.tors_b, dtype=np.int32)
        self.pairs = np.ascontiguousarray(lig.pairs, dtype=np.int32).reshape(-1, 2)
        self.N, self.T, self.P = int(self.ref.shape[0]), int(self.tors_a.shape[0]), int(self.pairs.shape[0])
        self.c = dock_ligand(self.N, self.T, self.P, _np_ptr(self.ref), _np_ptr(self.type), _np_ptr(self.frag),
                             _np_ptr(self.tors_parent), _np_ptr(self.tors_a), _np_ptr(self.tors_b), _np_ptr(self.pairs))


class GridMaps:
    """Device grid maps + descriptor.  `buf` owns the memory (both images, see dock.h);
    `data` is the [n_maps, nz, ny, nx] view of the maps themselves ([n_maps, 4, nz, ny, nx] in eq. 4 mode)."""

    def __init__(self, buf, data, desc: dock_grid):
        self.buf = buf
        self.data = data
        self.desc = desc

    @property
    def dims(self):
        return tuple(self.desc.dims)


def dock_grid_dims(box: dock_box):
    d = (C.c_int32 * 3)()
    _check(load_library().dock_grid_dims(C.byref(box), d), "dock_grid_dims")
    return tuple(int(x) for x in d)


def dock_grid_bytes(params: dock_params, box: dock_box, n_lig_types: int) -> int:
    n = int(load_library().dock_grid_bytes(C.byref(params), C.byref(box), int(n_lig_types)))
    if n == 0:
        raise DockError("dock_grid_bytes: bad box or type count")
    return n


def dock_build_grids(params: dock_params, protein_xyz, protein_type, box: dock_box,
                     lig_types: Sequence[int], stream=None) -> GridMaps:
    torch = _torch()
    lib = load_library()
    xyz = np.ascontiguousarray(protein_xyz, dtype=np.float32).reshape(-1, 3)
    typ = np.ascontiguousarray(protein_type, dtype=np.int32)
    prot = dock_protein(int(xyz.shape[0]), _np_ptr(xyz), _np_ptr(typ))
    lt = np.ascontiguousarray(lig_types, dtype=np.int32)
    nx, ny, nz = dock_grid_dims(box)
    ch = 4 if int(params.grad_mode) == 1 else 1                      # eq. 4: (score, d/dx, d/dy, d/dz) per map
    buf = torch.empty(dock_grid_bytes(params, box, len(lt)), dtype=torch.uint8, device="cuda")
    data = buf[: len(lt) * ch * nz * ny * nx * 4].view(torch.float32)
    data = data.view(len(lt), nz, ny, nx) if ch == 1 else data.view(len(lt), ch, nz, ny, nx)
    desc = dock_grid()
    need = C.c_size_t(0)
    rc = lib.dock_build_grids(C.byref(params), C.byref(prot), C.byref(box), len(lt), _np_ptr(lt),
                              None, C.c_size_t(0), None, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_build_grids(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_build_grids(C.byref(params), C.byref(prot), C.byref(box), len(lt), _np_ptr(lt),
                                _ptr(buf), C.c_size_t(buf.numel()), C.byref(desc), _ptr(ws), C.c_size_t(ws.numel()),
                                C.byref(need), _stream(stream)), "dock_build_grids")
    return GridMaps(buf, data, desc)


def dock_build_grids_batch(params: dock_params, proteins, boxes: Sequence[dock_box], lig_types: Sequence[int],
                           stream=None):
    """proteins: sequence of (xyz [n,3], type [n]).  One C call for all systems (BASELINE.json configs[3]); returns a
    list of GridMaps."""
    torch = _torch()
    lib = load_library()
    ns = len(proteins)
    assert len(boxes) == ns
    lt = np.ascontiguousarray(lig_types, dtype=np.int32)
    ch = 4 if int(params.grad_mode) == 1 else 1
    keep, prots, bxs = [], (dock_protein * ns)(), (dock_box * ns)()
    bufs, datas = [], []
    ptrs = (C.c_void_p * ns)()
    sizes = (C.c_size_t * ns)()
    for s, (xyz, typ) in enumerate(proteins):
        xyz = np.ascontiguousarray(xyz, dtype=np.float32).reshape(-1, 3)
        typ = np.ascontiguousarray(typ, dtype=np.int32)
        keep.append((xyz, typ))
        prots[s] = dock_protein(int(xyz.shape[0]), _np_ptr(xyz), _np_ptr(typ))
        bxs[s] = boxes[s]
        nx, ny, nz = dock_grid_dims(boxes[s])
        buf = torch.empty(dock_grid_bytes(params, boxes[s], len(lt)), dtype=torch.uint8, device="cuda")
        data = buf[: len(lt) * ch * nz * ny * nx * 4].view(torch.float32)
        datas.append(data.view(len(lt), nz, ny, nx) if ch == 1 else data.view(len(lt), ch, nz, ny, nx))
        bufs.append(buf)
        ptrs[s] = buf.data_ptr()
        sizes[s] = buf.numel()
    descs = (dock_grid * ns)()
    need = C.c_size_t(0)
    rc = lib.dock_build_grids_batch(C.byref(params), ns, prots, bxs, len(lt), _np_ptr(lt), None, None, None, None,
                                    C.c_size_t(0), C.byref(need), None)
    if rc not in (DOCK_EWORKSPACE, DOCK_OK):
        _check(rc, "dock_build_grids_batch(size query)")
    ws = _ws.get(max(need.value, 256), stream)
    _check(lib.dock_build_grids_batch(C.byref(params), ns, prots, bxs, len(lt), _np_ptr(lt), ptrs, sizes, descs, _ptr(ws),
                                      C.c_size_t(ws.numel()), C.byref(need), _stream(stream)), "dock_build_grids_batch")
    out = []
    for s in range(ns):
        d = dock_grid()
        C.memmove(C.byref(d), C.byref(descs[s]), C.sizeof(dock_grid))
        out.append(GridMaps(bufs[s], datas[s], d))
    return out


def dock_score_batch(params: dock_params, grid: GridMaps, ligand: LigandHandle, poses,
                     want_grad: bool = True, want_terms: bool = True, out=None, stream=None):
    """poses: torch.cuda float32 [n, 7+T].  Returns (energy [n], grad [n,6+T] | None, terms [n,3] | None)."""
    torch = _torch()
    lib = load_library()
    assert poses.is_cuda and poses.dtype == torch.float32 and poses.is_contiguous()
    n = int(poses.shape[0])
    assert poses.shape[1] == 7 + ligand.T
    if out is None:
        energy = torch.empty(n, dtype=torch.float32, device="cuda")
        grad = torch.empty((n, 6 + ligand.T), dtype=torch.float32, device="cuda") if want_grad else None
        terms = torch.empty((n, 3), dtype=torch.float32, device="cuda") if want_terms else None
    else:
        energy, grad, terms = out
    need = C.c_size_t(0)
    rc = lib.dock_score_batch(C.byref(params), C.byref(grid.desc), C.byref(ligand.c), C.c_int64(n), None, None,
                              None, None, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_score_batch(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_score_batch(C.byref(params), C.byref(grid.desc), C.byref(ligand.c), C.c_int64(n), _ptr(poses),
                                _ptr(energy), _ptr(grad), _ptr(terms), _ptr(ws), C.c_size_t(ws.numel()),
                                C.byref(need), _stream(stream)), "dock_score_batch")
    return energy, grad, terms


def dock_score_batch_host(params: dock_params, grid: GridMaps, ligand: LigandHandle, poses_host: np.ndarray,
                          want_grad: bool = True, want_terms: bool = False, out=None, stream=None):
    """HOST numpy (or pinned torch CPU) poses [n,7+T] in, host energy / grad / terms out; copies inside the call."""
    lib = load_library()
    _torch()
    n = int(poses_host.shape[0])
    hp = lambda a: C.c_void_p(0) if a is None else (C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else _np_ptr(a))
    if out is None:
        energy = np.empty(n, dtype=np.float32)
        grad = np.empty((n, 6 + ligand.T), dtype=np.float32) if want_grad else None
        terms = np.empty((n, 3), dtype=np.float32) if want_terms else None
    else:
        energy, grad, terms = out
    need = C.c_size_t(0)
    args = (C.byref(params), C.byref(grid.desc), C.byref(ligand.c), C.c_int64(n), hp(poses_host), hp(energy), hp(grad), hp(terms))
    rc = lib.dock_score_batch_host(*args, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_score_batch_host(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_score_batch_host(*args, _ptr(ws), C.c_size_t(ws.numel()), C.byref(need), _stream(stream)),
           "dock_score_batch_host")
    return energy, grad, terms


def dock_local_opt_batch(params: dock_params, grid: GridMaps, ligand: LigandHandle, poses, max_iters: int, stream=None,
                         trace_cap: int = 0):
    """Returns (out_pose [n,7+T], out_e [n], out_it [n,3] = iterations, evaluations, DOCK_EXIT_* reason) and, with
    trace_cap > 0, a 4th item: the per-iteration trace [n, trace_cap, DOCK_ITER_HEADER + (7+T) + (6+T) + (6+T)^2] (dock.h)."""
    torch = _torch()
    lib = load_library()
    assert poses.is_cuda and poses.dtype == torch.float32 and poses.is_contiguous()
    n = int(poses.shape[0])
    out_pose = torch.empty_like(poses)
    out_e = torch.empty(n, dtype=torch.float32, device="cuda")
    out_it = torch.empty((n, 3), dtype=torch.int32, device="cuda")
    need = C.c_size_t(0)
    rc = lib.dock_local_opt_batch(C.byref(params), C.byref(grid.desc), C.byref(ligand.c), C.c_int64(n), int(max_iters),
                                  None, None, None, None, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_local_opt_batch(size query)")
    ws = _ws.get(need.value, stream)
    if trace_cap > 0:
        nn = 6 + ligand.T
        trace = torch.zeros((n, int(trace_cap), DOCK_ITER_HEADER + 7 + ligand.T + nn + nn * nn), dtype=torch.float32, device="cuda")
        _check(lib.dock_local_opt_trace(C.byref(params), C.byref(grid.desc), C.byref(ligand.c), C.c_int64(n), int(max_iters),
                                        _ptr(poses), _ptr(out_pose), _ptr(out_e), _ptr(out_it), _ptr(trace), int(trace_cap),
                                        _ptr(ws), C.c_size_t(ws.numel()), C.byref(need), _stream(stream)), "dock_local_opt_trace")
        return out_pose, out_e, out_it, trace
    _check(lib.dock_local_opt_batch(C.byref(params), C.byref(grid.desc), C.byref(ligand.c), C.c_int64(n), int(max_iters),
                                    _ptr(poses), _ptr(out_pose), _ptr(out_e), _ptr(out_it), _ptr(ws),
                                    C.c_size_t(ws.numel()), C.byref(need), _stream(stream)), "dock_local_opt_batch")
    return out_pose, out_e, out_it


def dock_init_poses(box: dock_box, T: int, seed: int, system: int, copies: int, copy_base: int = 0) -> np.ndarray:
    out = np.zeros((copies, 7 + T), dtype=np.float32)
    _check(load_library().dock_init_poses(C.byref(box), int(T), C.c_uint64(seed), C.c_uint32(system), C.c_uint32(copy_base),
                                          int(copies), _np_ptr(out)), "dock_init_poses")
    return out


def dock_init_poses_site(box: dock_box, T: int, seed: int, system: int, copies: int, site_xyz, radius: float = 7.0,
                         copy_base: int = 0) -> np.ndarray:
    """NEXT-3: initial poses with the translation restrained to box ∩ union of balls around the site points."""
    site = np.ascontiguousarray(site_xyz, dtype=np.float32).reshape(-1, 3)
    out = np.zeros((copies, 7 + T), dtype=np.float32)
    _check(load_library().dock_init_poses_site(C.byref(box), int(T), C.c_uint64(seed), C.c_uint32(system), C.c_uint32(copy_base),
                                               int(copies), int(site.shape[0]), _np_ptr(site), C.c_float(radius), _np_ptr(out)),
           "dock_init_poses_site")
    return out


def dock_search(params: dock_params, grids: Sequence[GridMaps], ligands: Sequence[LigandHandle],
                boxes: Optional[Sequence[dock_box]], copies: int, steps: int, bfgs_max_iters: int, seed: int,
                init_poses=None, want_trace: bool = False, want_topk: bool = True, stream=None,
                system_base: int = 0, copy_base: int = 0):
    """Many-copy MC search for n_systems systems in one launch.  Returns a dict of torch tensors.
    system_base / copy_base: Philox indices of the first system / copy of this call (sharded runs, dock.h)."""
    torch = _torch()
    lib = load_library()
    ns = len(grids)
    assert len(ligands) == ns
    t_max = max(l.T for l in ligands)
    row = 7 + t_max
    k = int(params.topk)
    g_arr = (dock_grid * ns)(*[g.desc for g in grids])
    l_arr = (dock_ligand * ns)(*[l.c for l in ligands])
    b_arr = (dock_box * ns)(*boxes) if boxes is not None else None
    dev = "cuda"
    best_pose = torch.empty((ns, copies, row), dtype=torch.float32, device=dev)
    best_e = torch.empty((ns, copies), dtype=torch.float32, device=dev)
    topk_pose = torch.zeros((ns, k, row), dtype=torch.float32, device=dev) if want_topk else None
    topk_e = torch.zeros((ns, k), dtype=torch.float32, device=dev) if want_topk else None
    topk_idx = torch.full((ns, k), -1, dtype=torch.int32, device=dev) if want_topk else None
    topk_cnt = torch.zeros(ns, dtype=torch.int32, device=dev) if want_topk else None
    trace = torch.zeros((ns, copies, steps, DOCK_TRACE_HEADER + row), dtype=torch.float32, device=dev) if want_trace else None
    evals = torch.zeros(1, dtype=torch.int64, device=dev)
    if init_poses is not None:
        assert init_poses.is_cuda and init_poses.dtype == torch.float32 and init_poses.is_contiguous()
        assert tuple(init_poses.shape) == (ns, copies, row)
    need = C.c_size_t(0)
    head = (C.byref(params), ns, g_arr, l_arr, b_arr, int(copies), int(steps), int(bfgs_max_iters), C.c_uint64(seed),
            C.c_uint32(system_base), C.c_uint32(copy_base), _ptr(init_poses))
    rc = lib.dock_search(*head, _ptr(best_pose), _ptr(best_e), None, None, None, None, None, None,
                         None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_search(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_search(*head, _ptr(best_pose), _ptr(best_e), _ptr(topk_pose), _ptr(topk_e), _ptr(topk_idx),
                           _ptr(topk_cnt), _ptr(trace), _ptr(evals), _ptr(ws), C.c_size_t(ws.numel()), C.byref(need),
                           _stream(stream)), "dock_search")
    return dict(best_pose=best_pose, best_e=best_e, topk_pose=topk_pose, topk_e=topk_e, topk_idx=topk_idx,
                topk_count=topk_cnt, trace=trace, evals=evals)


def dock_topk(params: dock_params, ligand: LigandHandle, poses, e, stream=None):
    torch = _torch()
    lib = load_library()
    n = int(poses.shape[0])
    k = int(params.topk)
    out_idx = torch.full((k,), -1, dtype=torch.int32, device="cuda")
    out_cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    need = C.c_size_t(0)
    rc = lib.dock_topk(C.byref(params), C.byref(ligand.c), n, None, None, None, None, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_topk(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_topk(C.byref(params), C.byref(ligand.c), n, _ptr(poses), _ptr(e), _ptr(out_idx), _ptr(out_cnt),
                         _ptr(ws), C.c_size_t(ws.numel()), C.byref(need), _stream(stream)), "dock_topk")
    return out_idx, out_cnt


def dock_topk_fixed(params: dock_params, ligand: LigandHandle, poses, e, out_idx, out_cnt, stream=None):
    """dock_topk for callers that cannot allocate on the device (dock.h: dock_topk_fixed).

    Nothing is allocated here either: `out_idx` (int32 [params.topk]) and `out_cnt` (int32 [1]) are the caller's
    device tensors, and the kernel's tables live in the library's built-in scratch array, DOCK_TOPK_FIXED_BYTES per
    GPU, shared by all calls on that GPU (so overlapping calls race).  Raises DockError("... DOCK_ECAPACITY ...") when
    the ligand's tables do not fit.  Make the first call on a device outside stream capture."""
    _torch()
    lib = load_library()
    need = C.c_size_t(0)
    rc = lib.dock_topk_fixed(C.byref(params), C.byref(ligand.c), int(poses.shape[0]), _ptr(poses), _ptr(e), _ptr(out_idx),
                             _ptr(out_cnt), C.byref(need), _stream(stream))
    if rc == DOCK_ECAPACITY:
        raise DockError(f"dock_topk_fixed failed: DOCK_ECAPACITY (ligand tables need {need.value} bytes, the built-in "
                        f"scratch holds {DOCK_TOPK_FIXED_BYTES}; use dock_topk with a workspace)")
    _check(rc, "dock_topk_fixed")
    return out_idx, out_cnt


def dock_probe_peaks(stream=None) -> dict:
    """Measured roofs of the units this path is bound by (dock.h): FP32 FMA, packed FMA, MUFU, divergent 32-byte gathers."""
    lib = load_library()
    need = C.c_size_t(0)
    out = (C.c_float * 4)()
    rc = lib.dock_probe_peaks(out, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_probe_peaks(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_probe_peaks(out, _ptr(ws), C.c_size_t(ws.numel()), C.byref(need), _stream(stream)), "dock_probe_peaks")
    return dict(ffma_tflops=float(out[0]), ffma2_tflops=float(out[1]), mufu_tops=float(out[2]), gather32_tlanes=float(out[3]))


def dock_system_host(params: dock_params, protein_xyz, protein_type, box: dock_box, ligand: LigandHandle,
                     lig_types: Sequence[int], copies: int, steps: int, bfgs_max_iters: int, seed: int,
                     grid_buf=None, stream=None):
    """End to end for one system with HOST inputs/outputs: build grids + search + top-k."""
    torch = _torch()
    lib = load_library()
    xyz = np.ascontiguousarray(protein_xyz, dtype=np.float32).reshape(-1, 3)
    typ = np.ascontiguousarray(protein_type, dtype=np.int32)
    prot = dock_protein(int(xyz.shape[0]), _np_ptr(xyz), _np_ptr(typ))
    lt = np.ascontiguousarray(lig_types, dtype=np.int32)
    if grid_buf is None:
        grid_buf = torch.empty(dock_grid_bytes(params, box, len(lt)), dtype=torch.uint8, device="cuda")
    k = int(params.topk)
    out_pose = np.zeros((k, 7 + ligand.T), dtype=np.float32)
    out_e = np.zeros(k, dtype=np.float32)
    out_cnt = np.zeros(1, dtype=np.int32)
    out_ev = np.zeros(1, dtype=np.uint64)
    need = C.c_size_t(0)
    head = (C.byref(params), C.byref(prot), C.byref(box), C.byref(ligand.c), len(lt), _np_ptr(lt), int(copies),
            int(steps), int(bfgs_max_iters), C.c_uint64(seed), _np_ptr(out_pose), _np_ptr(out_e), _np_ptr(out_cnt),
            _np_ptr(out_ev), _ptr(grid_buf), C.c_size_t(grid_buf.numel()))
    rc = lib.dock_system_host(*head, None, C.c_size_t(0), C.byref(need), None)
    if rc != DOCK_EWORKSPACE:
        _check(rc, "dock_system_host(size query)")
    ws = _ws.get(need.value, stream)
    _check(lib.dock_system_host(*head, _ptr(ws), C.c_size_t(ws.numel()), C.byref(need), _stream(stream)),
           "dock_system_host")
    return dict(topk_pose=out_pose, topk_e=out_e, count=int(out_cnt[0]), evals=int(out_ev[0]))
