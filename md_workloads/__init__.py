"""Seeded synthetic MD workloads (inputs only).

This module is the ONE piece shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2003_14061_b200/`): it generates initial states.  It holds none of
the method's arithmetic (no cells, no neighbor matrix, no forces, no
integrator) -- only lattices, seeded random numbers and chain topology.

The recipes follow the paper's statement of its test systems
(section 3.1: "The initial state consists of a cubic grid of atoms
of size N_a = N_e^3 that are assigned random velocities") and the five
BASELINE.json configs; see DESIGN.md "Input recipe".
"""
from .configs import CONFIGS, MDConfig, get_config, scaled_config
from .generators import (
    body_inertia,
    box_edge,
    chain_melt,
    chain_walks,
    cross_body,
    fcc_lattice,
    gaussian_velocities,
    jitter,
    make_state,
    random_rotations,
    rigid_state,
    sc_lattice,
    splitmix64,
    tetrahedron_body,
    uniform01,
)

__all__ = [
    "CONFIGS",
    "MDConfig",
    "get_config",
    "scaled_config",
    "body_inertia",
    "box_edge",
    "chain_melt",
    "chain_walks",
    "cross_body",
    "fcc_lattice",
    "gaussian_velocities",
    "jitter",
    "make_state",
    "random_rotations",
    "rigid_state",
    "sc_lattice",
    "splitmix64",
    "tetrahedron_body",
    "uniform01",
]
