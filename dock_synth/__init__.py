"""Seeded synthetic inputs for the docking hot path (BASELINE.json:configs).

This module is the ONLY code shared between the CPU oracle (`oracle/`) and the CUDA
library (`paper_2303_09916_b200/`).  It holds no arithmetic of the method itself (no
scoring, no kinematics, no optimizer, no Philox): it only draws proteins, ligand
topologies, boxes and pose batches with NumPy's seeded generators.  The paper measures
on scPDB / PDBBind / DUD-E complexes which are not available
here; these synthetic systems take their shapes from BASELINE.json:configs and stand
in for them (recipe restated in DESIGN.md).
"""
from .generators import (  # noqa: F401
    XS_NAMES,
    XS,
    Ligand,
    System,
    make_protein_tiny,
    make_protein_globule,
    make_ligand,
    make_box,
    make_site_points,
    random_poses,
    make_system,
    CONFIGS,
)
