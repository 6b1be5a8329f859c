"""CPU-only checks of the C-ABI boundary: the library builds, loads and exports every symbol that
include/dock.h declares; host-side validation and size queries behave as documented (no kernel
is launched here -- none of these calls touches the device)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2303_09916_b200 as dk
from paper_2303_09916_b200 import binding as B
from paper_2303_09916_b200 import build as dkbuild
from dock_synth import make_system

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    dkbuild.build()
    return dk.load_library()


def test_header_symbols_are_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "dock.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(dock_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(dk.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_product_does_not_import_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2303_09916_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                for pat in (r"import\s+oracle", r"from\s+oracle", r"from\s+\.+oracle", "dock_oracle", "liboracle", r"orc_\w+\("):
                    assert not re.search(pat, text), (f, pat)


def test_default_params_match_the_readings(lib):
    p = dk.dock_default_params()
    assert p.n_types == 17
    assert np.allclose(list(p.w), [-0.0356, -0.00516, 0.840, -0.0351, -0.587])
    assert np.allclose(list(p.radius)[:17], [1.9, 1.9, 1.8, 1.8, 1.8, 1.8, 1.7, 1.7, 1.7, 1.7, 2.0, 2.1, 1.5, 1.8, 2.0, 2.2, 1.2])
    assert list(p.hydrophobic)[:17] == [1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 1, 1, 1, 0]
    assert list(p.donor)[:17] == [0, 0, 0, 1, 0, 1, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0, 1]
    assert list(p.acceptor)[:17] == [0, 0, 0, 0, 1, 1, 0, 0, 1, 1, 0, 0, 0, 0, 0, 0, 0]
    assert (p.cutoff, p.k_wall, p.bfgs_max_trials, p.topk) == (8.0, 10.0, 12, 10)
    assert lib.dock_default_params(None) == B.DOCK_EINVAL


def test_grid_dims_rule(lib):
    for size, n in ((15.0, 41), (30.0, 81), (60.0, 161)):
        assert dk.dock_grid_dims(dk.make_box([0, 0, 0], [size] * 3, 0.375)) == (n, n, n)
    d = (C.c_int32 * 3)()
    assert lib.dock_grid_dims(C.byref(dk.make_box([0, 0, 0], [10, 10, 10], 0.0)), d) == B.DOCK_EINVAL
    assert lib.dock_grid_dims(None, d) == B.DOCK_EINVAL


def test_build_grids_size_query_and_validation(lib):
    s = make_system(0, seed=0)
    p = dk.dock_default_params()
    xyz = np.ascontiguousarray(s.protein_xyz, np.float32)
    typ = np.ascontiguousarray(s.protein_type, np.int32)
    prot = B.dock_protein(len(typ), xyz.ctypes.data_as(C.c_void_p), typ.ctypes.data_as(C.c_void_p))
    box = dk.make_box(s.box_center, s.box_size, s.spacing)
    lt = np.array(s.lig_types, np.int32)
    need = C.c_size_t(0)
    rc = lib.dock_build_grids(C.byref(p), C.byref(prot), C.byref(box), len(lt), lt.ctypes.data_as(C.c_void_p),
                              None, C.c_size_t(0), None, None, C.c_size_t(0), C.byref(need), None)
    assert rc == B.DOCK_EWORKSPACE and need.value > 0
    bad = np.array([0, 99], np.int32)
    rc = lib.dock_build_grids(C.byref(p), C.byref(prot), C.byref(box), 2, bad.ctypes.data_as(C.c_void_p),
                              None, C.c_size_t(0), None, None, C.c_size_t(0), C.byref(need), None)
    assert rc == B.DOCK_EINVAL
    typ_bad = typ.copy()
    typ_bad[3] = -1
    prot_bad = B.dock_protein(len(typ), xyz.ctypes.data_as(C.c_void_p), typ_bad.ctypes.data_as(C.c_void_p))
    rc = lib.dock_build_grids(C.byref(p), C.byref(prot_bad), C.byref(box), len(lt), lt.ctypes.data_as(C.c_void_p),
                              None, C.c_size_t(0), None, None, C.c_size_t(0), C.byref(need), None)
    assert rc == B.DOCK_EINVAL
    # the grid buffer size is part of the contract: a buffer sized for one channel is rejected in eq. 4 mode (4 channels)
    # before anything touches the device (fake non-null pointers: the check comes first)
    one = dk.dock_grid_bytes(p, box, len(lt))
    p4 = dk.dock_default_params()
    p4.grad_mode = 1
    nodes = int(np.prod(dk.dock_grid_dims(box))) * len(lt)
    up = lambda b: (b + 255) // 256 * 256
    assert one == up(4 * nodes) + up(32 * nodes) + 16 * nodes              # maps + 8-corner image + 4-corner image (dock.h)
    four = dk.dock_grid_bytes(p4, box, len(lt))
    assert four == up(16 * nodes) + up(128 * nodes) and four > one         # eq. 4: four channels, no 4-corner image
    desc = B.dock_grid()
    rc = lib.dock_build_grids(C.byref(p4), C.byref(prot), C.byref(box), len(lt), lt.ctypes.data_as(C.c_void_p),
                              C.c_void_p(1 << 20), C.c_size_t(one), C.byref(desc), C.c_void_p(1 << 21), C.c_size_t(need.value),
                              C.byref(need), None)
    assert rc == B.DOCK_EINVAL
    rc = lib.dock_build_grids(C.byref(p), C.byref(prot), C.byref(box), len(lt), lt.ctypes.data_as(C.c_void_p),
                              C.c_void_p(1 << 20), C.c_size_t(one - 1), C.byref(desc), C.c_void_p(1 << 21), C.c_size_t(need.value),
                              C.byref(need), None)
    assert rc == B.DOCK_EINVAL
    # batched form: the workspace holds every system's cell lists
    prots = (B.dock_protein * 3)(prot, prot, prot)
    boxes = (B.dock_box * 3)(box, box, box)
    need3 = C.c_size_t(0)
    rc = lib.dock_build_grids_batch(C.byref(p), 3, prots, boxes, len(lt), lt.ctypes.data_as(C.c_void_p), None, None, None,
                                    None, C.c_size_t(0), C.byref(need3), None)
    assert rc == B.DOCK_EWORKSPACE and need.value < need3.value <= 3 * need.value
    assert lib.dock_build_grids_batch(C.byref(p), 0, None, None, len(lt), lt.ctypes.data_as(C.c_void_p), None, None, None,
                                      None, C.c_size_t(0), C.byref(need3), None) == B.DOCK_OK


def _fake_grid(s, lig_types):
    g = B.dock_grid()
    for c in range(3):
        g.dims[c] = 41
        g.origin[c] = 0.0
    g.spacing = 0.375
    g.n_maps = len(lig_types)
    for t in range(32):
        g.type_to_map[t] = -1
    for m, t in enumerate(lig_types):
        g.type_to_map[t] = m
    g.data_dev = 256  # never dereferenced by the size query
    g.packed_dev = 512
    return g


def test_score_batch_validates_the_ligand_on_the_host(lib):
    s = make_system(0, seed=0)
    p = dk.dock_default_params()
    g = _fake_grid(s, s.lig_types)
    need = C.c_size_t(0)

    def query(lig):
        h = dk.LigandHandle(lig)
        return lib.dock_score_batch(C.byref(p), C.byref(g), C.byref(h.c), C.c_int64(4), None, None, None, None,
                                    None, C.c_size_t(0), C.byref(need), None)

    assert query(s.ligand) == B.DOCK_EWORKSPACE and need.value > 0
    import copy
    bad = copy.deepcopy(s.ligand)
    bad.tors_parent = bad.tors_parent.copy()
    bad.tors_parent[0] = 1                      # parent > k
    assert query(bad) == B.DOCK_EINVAL
    bad = copy.deepcopy(s.ligand)
    bad.tors_a, bad.tors_b = bad.tors_b.copy(), bad.tors_a.copy()   # axis atoms in the wrong fragments
    assert query(bad) == B.DOCK_EINVAL
    bad = copy.deepcopy(s.ligand)
    bad.pairs = bad.pairs.copy()
    bad.pairs[0, 1] = 99                        # pair index out of range
    assert query(bad) == B.DOCK_EINVAL
    bad = copy.deepcopy(s.ligand)
    bad.type = bad.type.copy()
    bad.type[0] = 12                            # F_H: valid XS id but no map in this grid
    assert query(bad) == B.DOCK_EINVAL
    bad.type[0] = 40                            # outside the table
    assert query(bad) == B.DOCK_EINVAL


def test_init_poses_follow_the_philox_rule(orc, lib):
    """Host logic of dock_init_poses against the oracle's independent implementation (S16, R-rules)."""
    box = dk.make_box([1.5, -2.25, 3.0], [30, 30, 30], 0.375)
    for T in (0, 3, 7, 15):
        a = dk.dock_init_poses(box, T, 0xDEADBEEF12345678, 3, 64)
        b = orc.init_poses([1.5, -2.25, 3.0], [30, 30, 30], T, 0xDEADBEEF12345678, 3, 64)
        assert a.shape == b.shape == (64, 7 + T)
        assert np.max(np.abs(a.astype(np.float64) - b)) <= 1e-6
        assert np.mean(a.astype(np.float64) == b) > 0.99   # same formulas in double, rounded once
        # copy_base: a shard of copies starts exactly where those copies of the unsharded run start
        assert np.array_equal(dk.dock_init_poses(box, T, 0xDEADBEEF12345678, 3, 24, copy_base=40), a[40:])


def test_site_restrained_initial_poses(orc, lib):
    """NEXT-3 (Fig. 3; reading S22): host logic of dock_init_poses_site against the oracle, and the
    properties that define it: every translation lies in box ∩ union of 7 A balls, the accepted points are uniform
    in that set, one ball that covers the box reduces to the plain rule, orientation / torsions are untouched."""
    from dock_synth import make_site_points
    center, size = [1.5, -2.25, 3.0], [30.0, 30.0, 30.0]
    box = dk.make_box(center, size, 0.375)
    site = make_site_points(np.random.default_rng(1), center, size, n=120)
    assert site.shape == (120, 3) and np.all(np.abs(site - np.array(center)) <= 8.0 + 1e-6)
    seed = 0x1234ABCD5678
    for T in (0, 7):
        a = dk.dock_init_poses_site(box, T, seed, 2, 512, site, 7.0)
        b = orc.init_poses_site(center, size, T, seed, 2, 512, site, 7.0)
        assert np.array_equal(a[:, :3].astype(np.float64), b[:, :3])             # same integers, same affine map, one rounding
        assert np.max(np.abs(a.astype(np.float64) - b)) <= 1e-6
        d = np.min(np.linalg.norm(b[:, None, :3] - site[None].astype(np.float64), axis=2), axis=1)
        assert np.all(d <= 7.0 + 1e-5)
        assert np.all(np.abs(b[:, :3] - np.array(center)) <= 15.0)
        plain = orc.init_poses(center, size, T, seed, 2, 512)
        assert np.array_equal(plain[:, 3:], b[:, 3:])                             # q, theta as S16
    # uniform in the set: with two far-apart site points, each ball receives about half of the copies
    two = np.array([[center[0] - 7.5, center[1], center[2]], [center[0] + 7.5, center[1], center[2]]], np.float32)
    c = orc.init_poses_site(center, size, 0, seed, 0, 2000, two, 7.0)
    left = (c[:, 0] < center[0]).mean()
    assert abs(left - 0.5) < 0.04
    # a ball that contains the whole box accepts attempt 0 -> equals slot 0x100's draw, inside the box
    big = orc.init_poses_site(center, size, 0, seed, 0, 64, np.array([center], np.float32), 100.0)
    assert np.all(np.abs(big[:, :3] - np.array(center)) <= 15.0)
    # no point of the box is within reach -> the fallback site point
    far = np.array([[500.0, 0.0, 0.0], [600.0, 0.0, 0.0]], np.float32)
    f = dk.dock_init_poses_site(box, 0, seed, 0, 4, far, 7.0)
    assert np.array_equal(f[:, :3], far[[0, 1, 0, 1]])
    full = dk.dock_init_poses_site(box, 7, seed, 2, 64, site, 7.0)
    assert np.array_equal(dk.dock_init_poses_site(box, 7, seed, 2, 20, site, 7.0, copy_base=44), full[44:])


def test_search_rejects_before_it_enqueues(lib):
    """dock_search validates everything on the host first: a copy count whose top-k sort does not fit shared memory and
    mixed gradient modes are DOCK_EINVAL at the size query already (no device pointer is ever touched)."""
    s = make_system(0, seed=0)
    p = dk.dock_default_params()
    g = _fake_grid(s, s.lig_types)
    h = dk.LigandHandle(s.ligand)
    box = dk.make_box(s.box_center, s.box_size, s.spacing)
    need = C.c_size_t(0)
    fake = C.c_void_p(1 << 20)

    def query(copies, grids, want_topk=True):
        ns = len(grids)
        g_arr = (B.dock_grid * ns)(*grids)
        l_arr = (B.dock_ligand * ns)(*[h.c] * ns)
        b_arr = (B.dock_box * ns)(*[box] * ns)
        tk = fake if want_topk else None
        return lib.dock_search(C.byref(p), ns, g_arr, l_arr, b_arr, copies, 2, 10, C.c_uint64(1), C.c_uint32(0), C.c_uint32(0),
                               None, fake, fake, tk, tk, tk, tk, None, None, None, C.c_size_t(0), C.byref(need), None)

    assert query(64, [g]) == B.DOCK_EWORKSPACE
    assert query(1 << 16, [g]) == B.DOCK_EINVAL             # 2 x 65536 sort keys + poses > 200 KB of shared memory
    assert query(1 << 16, [g], want_topk=False) == B.DOCK_EWORKSPACE
    g4 = _fake_grid(s, s.lig_types)
    g4.n_channels = 4
    assert query(64, [g, g4]) == B.DOCK_EINVAL               # one gradient mode per launch


def test_specialised_score_kernel_source_and_compilation(lib):
    """score_kernel = 2: the generated CUDA text for configs[0] and a 21-atom ligand compiles for sm_100a with NVRTC on
    this (GPU-less) box; every listed pair appears in exactly one chain; out-of-range ligands are refused."""
    import re
    from dock_synth import make_system, make_ligand
    from dock_synth.generators import LIG_TYPES_FULL
    lib.dock_score_jit_log.restype = C.c_char_p
    p = B.dock_default_params()
    s = make_system(0, seed=0)
    g = B.dock_grid()
    g.dims[0] = g.dims[1] = g.dims[2] = 41
    g.spacing = 0.375
    for t in range(32):
        g.type_to_map[t] = -1
    for m, t in enumerate(LIG_TYPES_FULL):
        g.type_to_map[int(t)] = m
    g.n_maps = len(LIG_TYPES_FULL)
    g.n_channels = 1
    g.data_dev, g.packed_dev = 256, 512            # never dereferenced: no device work in these calls
    for ligd in (s.ligand, make_ligand(np.random.default_rng(3), 21, 4, LIG_TYPES_FULL)):
        lig = B.LigandHandle(ligd)
        need = C.c_size_t(0)
        assert lib.dock_score_jit_source(C.byref(p), C.byref(g), C.byref(lig.c), 1, None, C.c_size_t(0), C.byref(need)) == B.DOCK_EWORKSPACE
        buf = C.create_string_buffer(need.value)
        assert lib.dock_score_jit_source(C.byref(p), C.byref(g), C.byref(lig.c), 1, buf, C.c_size_t(need.value), C.byref(need)) == B.DOCK_OK
        src = buf.value.decode()
        assert "dock_score_jit" in src and "fma.rn.f32x2" in src
        m = re.search(r"A4, (\d+) chains for (\d+) pairs", src)
        assert m and int(m.group(2)) == lig.P and (lig.P + 1) // 2 <= int(m.group(1)) <= lig.P
        assert src.count("rsq(") - 1 == lig.P          # one reciprocal square root per listed pair (+ the helper's definition)
        nb = C.c_size_t(0)
        rc = lib.dock_score_jit_compile(C.byref(p), C.byref(g), C.byref(lig.c), 1, C.byref(nb))
        assert rc == B.DOCK_OK and nb.value > 10000, (rc, lib.dock_score_jit_log())
    big = B.LigandHandle(make_ligand(np.random.default_rng(4), 44, 6, LIG_TYPES_FULL))
    assert lib.dock_score_jit_source(C.byref(p), C.byref(g), C.byref(big.c), 1, None, C.c_size_t(0), C.byref(need)) == B.DOCK_EINVAL
    g.n_channels = 4
    assert lib.dock_score_jit_source(C.byref(p), C.byref(g), C.byref(lig.c), 1, None, C.c_size_t(0), C.byref(need)) == B.DOCK_EINVAL


def test_specialised_kernel_cache_limit_arguments():
    """dock_score_jit_cache: query, set, and the rejected limits (host only)."""
    import paper_2303_09916_b200 as dk
    from paper_2303_09916_b200 import binding as B
    old, n = dk.score_jit_cache()
    assert old >= 1 and n >= 0
    assert dk.score_jit_cache(5) == (old, n) and dk.score_jit_cache()[0] == 5
    lib = dk.load_library()
    assert lib.dock_score_jit_cache(0, None, None) == B.DOCK_EINVAL and lib.dock_score_jit_cache(1 << 20, None, None) == B.DOCK_EINVAL
    assert dk.score_jit_cache(old)[0] == 5 and dk.score_jit_cache()[0] == old
