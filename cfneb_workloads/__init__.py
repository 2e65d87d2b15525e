"""Seeded synthetic inputs for the CFNEB hot path (BASELINE.json `configs`).

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2510_16721_b200/`).  It holds no arithmetic of the method itself:
no potential, no cell filter, no tangent, no FIRE.  It only builds lattices,
draws seeded noise and interpolates paths linearly, and hands plain numpy
arrays to both sides.

The recipe is documented in DESIGN.md §"Input recipe"; it stands in for the
paper's Ti3O5 / graphite NEP workloads (up to 1e5
atoms x 100 images, periodic solids, variable cell), which need trained weights
and structures that are not available.
"""
from .lattices import fcc_supercell, bcc_supercell, bain_final_cell, diamond_supercell
from .noise import splitmix64_normals
from .configs import (
    CONFIGS,
    WorkloadSpec,
    lj_params,
    fs_params,
    sw_params,
    dn_params,
    nep_params,
    two_sublattice_types,
    diamond_strain_band,
    vacancy_endpoints_unrelaxed,
    bain_endpoints,
    linear_path,
    load_lattice_constants,
    load_vacancy_endpoints,
    build_workload,
)

__all__ = [
    "fcc_supercell",
    "bcc_supercell",
    "bain_final_cell",
    "diamond_supercell",
    "sw_params",
    "dn_params",
    "nep_params",
    "two_sublattice_types",
    "diamond_strain_band",
    "splitmix64_normals",
    "CONFIGS",
    "WorkloadSpec",
    "lj_params",
    "fs_params",
    "vacancy_endpoints_unrelaxed",
    "bain_endpoints",
    "linear_path",
    "load_lattice_constants",
    "load_vacancy_endpoints",
    "build_workload",
]
