"""Seeded synthetic workloads (BASELINE.json `configs`; recipe in DESIGN.md §4).

This module produces *inputs only*: geometries, Gaussian shell tables, quadrature
points/weights and density matrices.  It holds none of the method's arithmetic
(no AO evaluation, no density, no functional, no contraction), so both the CPU
oracle's tests and the CUDA path may draw their inputs from it.
"""
from .generate import (  # noqa: F401
    ANG2BOHR,
    Workload,
    alkane_geometry,
    atomic_grid,
    becke_weights,
    density_matrix,
    make_workload,
    named_config,
    shells_for,
    water_cluster_geometry,
    water_monomer,
)
