"""Seeded generators: proteins, ligand torsion trees, boxes, pose batches.

Recipe = SURVEY.md §8(d) / BASELINE.json:configs.  No scoring, kinematics, optimizer
or Philox code lives here (those are implemented twice, independently, in `oracle/`
and in the CUDA library).  Everything is drawn from `numpy.random.Generator(PCG64(seed))`.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

# XS atom-type ids, in the order fixed by SURVEY.md §8(c) S2.
XS_NAMES = [
    "C_H", "C_P", "N_P", "N_D", "N_A", "N_DA", "O_P", "O_D", "O_A", "O_DA",
    "S_P", "P_P", "F_H", "Cl_H", "Br_H", "I_H", "Met_D",
]
XS: Dict[str, int] = {n: i for i, n in enumerate(XS_NAMES)}

LIG_TYPES_TINY = [XS["C_H"], XS["C_P"], XS["N_D"], XS["O_A"]]
LIG_TYPES_FULL = [XS["C_H"], XS["C_P"], XS["N_P"], XS["N_D"], XS["N_A"], XS["O_A"], XS["O_D"], XS["O_DA"]]


@dataclass
class Ligand:
    """Flexible ligand as a torsion tree (layout = include/dock.h `dock_ligand`)."""
    ref_xyz: np.ndarray       # [N,3] float64 reference conformation
    type: np.ndarray          # [N] int32 XS type ids
    frag: np.ndarray          # [N] int32 rigid fragment of each atom (0 = root)
    tors_parent: np.ndarray   # [T] int32 fragment index of the parent of fragment k+1 (<= k)
    tors_a: np.ndarray        # [T] int32 axis atom in the parent fragment
    tors_b: np.ndarray        # [T] int32 axis atom in fragment k+1
    pairs: np.ndarray         # [P,2] int32 intra-ligand scoring pairs (i<j)
    bonds: np.ndarray         # [N-1,2] int32 bond list (generator bookkeeping only)

    @property
    def N(self) -> int:
        return int(self.ref_xyz.shape[0])

    @property
    def T(self) -> int:
        return int(self.tors_a.shape[0])

    @property
    def P(self) -> int:
        return int(self.pairs.shape[0])


@dataclass
class System:
    name: str
    protein_xyz: np.ndarray   # [Np,3] float32
    protein_type: np.ndarray  # [Np] int32
    ligand: Ligand
    box_center: np.ndarray    # [3] float32
    box_size: np.ndarray      # [3] float32
    spacing: float
    lig_types: List[int]      # ligand XS types for which maps are built
    copies: int = 0
    steps: int = 0
    bfgs_cap: int = 0
    extra: dict = field(default_factory=dict)


def _unit(v):
    return v / np.linalg.norm(v)


def _protein_types(rng: np.random.Generator, n: int) -> np.ndarray:
    """70 % C_H/C_P, 15 % N_P/N_D/N_A, 15 % O_A/O_DA, uniform within each group."""
    grp = rng.random(n)
    t = np.empty(n, dtype=np.int32)
    c = np.array([XS["C_H"], XS["C_P"]])
    nn = np.array([XS["N_P"], XS["N_D"], XS["N_A"]])
    oo = np.array([XS["O_A"], XS["O_DA"]])
    for i in range(n):
        if grp[i] < 0.70:
            t[i] = c[rng.integers(2)]
        elif grp[i] < 0.85:
            t[i] = nn[rng.integers(3)]
        else:
            t[i] = oo[rng.integers(2)]
    return t


def make_protein_tiny(rng, n=200, cube=20.0, dmin=2.8) -> Tuple[np.ndarray, np.ndarray]:
    """Tiny config: n points uniform in a cube by rejection at dmin; cube spans [0,cube]^3."""
    pts = np.zeros((0, 3))
    tries = 0
    while pts.shape[0] < n:
        p = rng.random(3) * cube
        tries += 1
        if tries > 2_000_000:
            raise RuntimeError("rejection sampling did not terminate")
        if pts.shape[0] and np.min(np.sum((pts - p) ** 2, axis=1)) < dmin * dmin:
            continue
        pts = np.vstack([pts, p])
    return pts.astype(np.float32), _protein_types(rng, n)


def make_protein_globule(rng, n, a=2.46, jitter=0.3, return_lattice=False):
    """Compact globule: jittered cubic lattice, keep the n sites nearest the origin.
    With return_lattice the whole lattice sorted by distance and the permutation are returned too (carve_pocket)."""
    r_need = (3.0 * n / (4.0 * np.pi)) ** (1.0 / 3.0) * a * 1.25 + 2 * a
    m = int(np.ceil(r_need / a))
    ax = np.arange(-m, m + 1) * a
    gx, gy, gz = np.meshgrid(ax, ax, ax, indexing="ij")
    pts = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1)
    pts = pts + (rng.random(pts.shape) * 2.0 - 1.0) * jitter
    d = np.linalg.norm(pts, axis=1)
    full = pts[np.argsort(d, kind="stable")]
    pts = full[:n]
    radius = float(np.max(np.linalg.norm(pts, axis=1)))
    perm = rng.permutation(n)  # no spatial ordering in the input
    types = _protein_types(rng, n)
    if return_lattice:
        return pts[perm].astype(np.float32), types, radius, full, perm
    return pts[perm].astype(np.float32), types, radius


POCKET_RADIUS = 7.0   # A: radius of the carved cavity
POCKET_DEPTH = 4.0    # A: its centre lies this far below the surface point the box is centred on


def carve_pocket(full_sorted: np.ndarray, n: int, perm: np.ndarray, surface_point: np.ndarray) -> np.ndarray:
    """A binding pocket at the box centre (configs 1-3): the globule is re-selected as the n lattice sites nearest the
    origin that lie OUTSIDE a sphere of POCKET_RADIUS centred POCKET_DEPTH below `surface_point` -- a half-open cavity
    of about the ligand's volume, so that the search landscape has a real minimum (a convex lattice surface has none:
    best energies stayed positive).  Atom count, density, types and input order are unchanged; no random draw is used,
    so ligand and box are the ones of the uncarved system."""
    sp = np.asarray(surface_point, dtype=np.float64)
    r = float(np.linalg.norm(sp))
    centre = sp * (1.0 - POCKET_DEPTH / r) if r > 0 else sp
    keep = np.linalg.norm(full_sorted - centre, axis=1) >= POCKET_RADIUS
    pts = full_sorted[keep][:n]
    assert pts.shape[0] == n
    return pts[perm].astype(np.float32)


def _grow_tree(rng, N: int):
    bond, ang = 1.5, np.deg2rad(109.5)
    xyz = np.zeros((N, 3))
    nbrs: List[List[int]] = [[] for _ in range(N)]
    bonds = []
    xyz[1] = [bond, 0.0, 0.0]
    nbrs[0].append(1)
    nbrs[1].append(0)
    bonds.append((0, 1))
    n, fails = 2, 0
    while n < N:
        if fails > 5000:
            return None
        p = int(rng.integers(n))
        if len(nbrs[p]) >= 4:
            fails += 1
            continue
        r = nbrs[p][int(rng.integers(len(nbrs[p])))]
        b = _unit(xyz[r] - xyz[p])
        v = rng.normal(size=3)
        v = v - v.dot(b) * b
        if np.linalg.norm(v) < 1e-6:
            fails += 1
            continue
        v = _unit(v)
        cand = xyz[p] + bond * (np.cos(ang) * b + np.sin(ang) * v)
        dist = np.linalg.norm(xyz[:n] - cand, axis=1)
        dist[p] = np.inf
        if dist.min() < 2.0:
            fails += 1
            continue
        xyz[n] = cand
        nbrs[p].append(n)
        nbrs[n].append(p)
        bonds.append((p, n))
        n += 1
    return xyz, nbrs, bonds


def make_ligand(rng, N: int, T: int, lig_types: Sequence[int], carbon_frac=0.65) -> Ligand:
    """Random tree ligand: 1.5 A bonds, 109.5 deg angles, random dihedrals, <=4 neighbours,
    no non-bonded contact under 2.0 A; T torsions among non-terminal bonds; fragments
    numbered parents-first; pairs = different fragment AND bond-graph distance >= 4 (S9)."""
    for _ in range(500):
        g = _grow_tree(rng, N)
        if g is None:
            continue
        xyz, nbrs, bonds = g
        cand = [(u, v) for (u, v) in bonds if len(nbrs[u]) >= 2 and len(nbrs[v]) >= 2]
        if len(cand) < T:
            continue
        sel = rng.choice(len(cand), size=T, replace=False) if T > 0 else []
        tors = {tuple(sorted(cand[int(k)])) for k in sel}
        # rigid fragments = components of the bond graph without the torsion bonds
        comp = -np.ones(N, dtype=np.int64)
        nc = 0
        for s in range(N):
            if comp[s] >= 0:
                continue
            stack = [s]
            comp[s] = nc
            while stack:
                u = stack.pop()
                for w in nbrs[u]:
                    if comp[w] < 0 and tuple(sorted((u, w))) not in tors:
                        comp[w] = nc
                        stack.append(w)
            nc += 1
        assert nc == T + 1
        # fragment tree, BFS from the fragment of atom 0; new fragment index k+1 <-> torsion k
        new_id = {int(comp[0]): 0}
        order = [int(comp[0])]
        tors_parent, tors_a, tors_b = [], [], []
        qi = 0
        while qi < len(order):
            c = order[qi]
            qi += 1
            for (u, v) in sorted(tors):
                for (a, b) in ((u, v), (v, u)):
                    if comp[a] == c and int(comp[b]) not in new_id:
                        new_id[int(comp[b])] = len(order)
                        order.append(int(comp[b]))
                        tors_parent.append(new_id[c])
                        tors_a.append(a)
                        tors_b.append(b)
        frag = np.array([new_id[int(c)] for c in comp], dtype=np.int32)
        # element/type assignment: ~65 % carbon, carbons next to a heteroatom are C_P
        hetero = [t for t in lig_types if t not in (XS["C_H"], XS["C_P"])]
        is_c = rng.random(N) < carbon_frac
        typ = np.empty(N, dtype=np.int32)
        for i in range(N):
            if not is_c[i]:
                typ[i] = hetero[int(rng.integers(len(hetero)))]
        for i in range(N):
            if is_c[i]:
                typ[i] = XS["C_P"] if any(not is_c[w] for w in nbrs[i]) else XS["C_H"]
        # bond-graph distances (BFS from every atom)
        dist = np.full((N, N), 10 ** 6, dtype=np.int64)
        for s in range(N):
            dist[s, s] = 0
            q = [s]
            while q:
                u = q.pop(0)
                for w in nbrs[u]:
                    if dist[s, w] > dist[s, u] + 1:
                        dist[s, w] = dist[s, u] + 1
                        q.append(w)
        pairs = [(i, j) for i in range(N) for j in range(i + 1, N)
                 if frag[i] != frag[j] and dist[i, j] >= 4]
        return Ligand(
            # fp32-representable values (stored as float64): the CUDA library takes fp32, the oracle widens them
            ref_xyz=np.ascontiguousarray(xyz.astype(np.float32), dtype=np.float64),
            type=typ,
            frag=frag,
            tors_parent=np.array(tors_parent, dtype=np.int32).reshape(T),
            tors_a=np.array(tors_a, dtype=np.int32).reshape(T),
            tors_b=np.array(tors_b, dtype=np.int32).reshape(T),
            pairs=np.array(pairs, dtype=np.int32).reshape(-1, 2),
            bonds=np.array(bonds, dtype=np.int32).reshape(-1, 2),
        )
    raise RuntimeError("could not build a ligand with the requested N, T")


def make_box(rng, kind: str, radius: float = 0.0, size: float = 30.0, center=None):
    if kind == "surface":  # box centred at a random surface point R*u (configs 1-3)
        u = _unit(rng.normal(size=3))
        c = radius * u
    elif kind == "center":
        c = np.zeros(3) if center is None else np.asarray(center, dtype=np.float64)
    else:
        raise ValueError(kind)
    return c.astype(np.float32), np.full(3, size, dtype=np.float32)


def random_poses(rng, n: int, box_center, box_size, T: int) -> np.ndarray:
    """n poses [t(3), q(w,x,y,z), theta(T)]: t uniform in the box, uniform random unit
    quaternions, torsions uniform in [-pi, pi).  Drawn in double, stored fp32 (config 1)."""
    c = np.asarray(box_center, dtype=np.float64)
    s = np.asarray(box_size, dtype=np.float64)
    out = np.empty((n, 7 + T), dtype=np.float64)
    out[:, 0:3] = c - 0.5 * s + rng.random((n, 3)) * s
    u1, u2, u3 = rng.random(n), rng.random(n), rng.random(n)
    out[:, 3] = np.sqrt(u1) * np.cos(2 * np.pi * u3)
    out[:, 4] = np.sqrt(1 - u1) * np.sin(2 * np.pi * u2)
    out[:, 5] = np.sqrt(1 - u1) * np.cos(2 * np.pi * u2)
    out[:, 6] = np.sqrt(u1) * np.sin(2 * np.pi * u3)
    if T:
        out[:, 7:] = -np.pi + 2 * np.pi * rng.random((n, T))
    return out.astype(np.float32)


# BASELINE.json:configs, by index.
def make_site_points(rng: np.random.Generator, box_center, box_size, n: int = 120, step: float = 1.5,
                     margin: float = 7.0) -> np.ndarray:
    """Synthetic 'predicted binding site' points (Fig. 3): a connected random-walk cluster of n points on a
    `step` lattice that starts at the box centre and stays at least `margin` inside the box -- a cavity-shaped blob that
    stands in for the output of the paper's site-prediction network (out of scope here)."""
    c = np.asarray(box_center, dtype=np.float64)
    half = 0.5 * np.asarray(box_size, dtype=np.float64) - margin
    if int(np.prod(2 * np.floor(np.maximum(half, 0.0) / step) + 1)) < n:
        raise ValueError("box too small for n site points at this step and margin")
    pts = {(0, 0, 0)}
    frontier = [(0, 0, 0)]
    moves = [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    while len(pts) < n:
        base = frontier[int(rng.integers(len(frontier)))]
        m = moves[int(rng.integers(6))]
        q = (base[0] + m[0], base[1] + m[1], base[2] + m[2])
        if q in pts or np.any(np.abs(np.array(q) * step) > half):
            continue
        pts.add(q)
        frontier.append(q)
    return (c + step * np.array(sorted(pts), dtype=np.float64)).astype(np.float32)


CONFIGS = {
    0: dict(name="tiny", n_prot=200, box=15.0, N=12, T=2, copies=16, steps=20, cap=50),
    1: dict(name="scoring_microbench", n_prot=3000, box=30.0, N=30, T=6, n_poses=1_048_576),
    2: dict(name="site_docking", n_prot=3000, box=30.0, N=32, T=7, copies=384, steps=40, cap=300),
    3: dict(name="batched_screening", n_systems=256, box=30.0, copies=128, steps=40, cap=300),
    4: dict(name="large_blind_box", n_prot=8000, box=60.0, N=60, T=15, copies=2048, steps=80, cap=300),
}


def make_system(config: int, seed: int = 0, index: int = 0,
                n_prot: Optional[int] = None, N: Optional[int] = None, T: Optional[int] = None) -> System:
    """One synthetic system of BASELINE.json:configs[config].  For config 3, `index`
    selects the system inside the batch (sizes drawn per system)."""
    cfg = CONFIGS[config]
    rng = np.random.default_rng(np.random.PCG64([seed, config, index]))
    if config == 0:
        pxyz, ptyp = make_protein_tiny(rng, n_prot or cfg["n_prot"])
        lig = make_ligand(rng, N or cfg["N"], cfg["T"] if T is None else T, LIG_TYPES_TINY)
        c, s = make_box(rng, "center", size=cfg["box"], center=[10.0, 10.0, 10.0])
        return System(cfg["name"], pxyz, ptyp, lig, c, s, 0.375, list(LIG_TYPES_TINY),
                      cfg["copies"], cfg["steps"], cfg["cap"])
    if config == 3:
        npr = int(rng.integers(1500, 6001)) if n_prot is None else n_prot
        nl = int(rng.integers(15, 51)) if N is None else N
        tl = int(np.clip(nl // 4 + int(rng.integers(-1, 2)), 2, 12)) if T is None else T
    else:
        npr = n_prot or cfg["n_prot"]
        nl = N or cfg["N"]
        tl = cfg["T"] if T is None else T
    pxyz, ptyp, radius, lattice, perm = make_protein_globule(rng, npr, return_lattice=True)
    lig = make_ligand(rng, nl, tl, LIG_TYPES_FULL)
    if config == 4:
        c, s = make_box(rng, "center", size=cfg["box"])
    else:
        c, s = make_box(rng, "surface", radius=radius, size=cfg["box"])
        pxyz = carve_pocket(lattice, npr, perm, c)
    return System(cfg["name"], pxyz, ptyp, lig, c, s, 0.375, list(LIG_TYPES_FULL),
                  cfg.get("copies", 0), cfg.get("steps", 0), cfg.get("cap", 0),
                  extra=dict(radius=radius))
