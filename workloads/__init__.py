"""Seeded synthetic input generators for the five BASELINE.json configs.

This package produces INPUTS only (voxel ``site_type`` arrays, iolet densities, the
relaxation time, an initial rho/u field). It contains none of the lattice-Boltzmann
arithmetic, imports neither ``oracle/`` nor ``paper_1906_11925_b200/``, and is the one
piece of code both sides of the parity tests share.
"""
from .geometries import (  # noqa: F401
    Workload,
    pipe,
    periodic_cube,
    aneurysm,
    tree,
    random_mask,
    by_name,
    with_velocity_inlet,
    pulsatile_waveform,
    with_inlet_profile,
    with_bfl_walls,
    wall_distance_by_bisection,
    CONFIG_NAMES,
)
