"""Seeded synthetic inputs for the BEM Poisson-Boltzmann hot path.

This module holds NONE of the method's arithmetic (no kernels, quadrature,
operators or energies): it only draws geometry and site parameters, so the CPU
oracle (oracle/) and the CUDA path can both be fed from it without sharing
method code.  It imports neither of them.

The inputs stand in for the paper's workloads (PDB structures, msms meshes and
amoebapro parameters, Table 3), which are not available; the
recipes are those of BASELINE.json `configs` as read in DESIGN.md section 4.
"""
from .meshes import icosphere, check_closed_oriented, mesh_stats
from .solutes import draw_sites, random_chain_globule, vdw_surface
from .configs import CONFIGS, make_config, Workload, seed_for

__all__ = [
    "icosphere", "check_closed_oriented", "mesh_stats", "draw_sites",
    "random_chain_globule", "vdw_surface", "CONFIGS", "make_config", "Workload", "seed_for",
]
