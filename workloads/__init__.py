"""Seeded synthetic workloads (BASELINE.json configs 0-4) for the direct-cut pass.

This package is the single source of input arrays for BOTH the CPU oracle
(`oracle/`) and the CUDA path (`paper_1711_07663_b200/`).  It holds none of the
method's arithmetic (no distances, boxes, Bezier nets, labels): only geometry
construction from closed-form recipes and `numpy.random.default_rng(seed)`.
"""
from .synth import (  # noqa: F401
    BASE_SEED,
    Workload,
    background_grid,
    cubed_sphere_dirs,
    cubed_sphere_faces,
    dimple_centres,
    dimpled_radius,
    ellipsoid_bodies,
    make_config,
    random_rotation,
    rotation_about_axis,
    spin_axis,
    check_watertight,
    check_conforming,
)
