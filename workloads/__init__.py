"""Seeded synthetic inputs (numpy only).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path's tests / bench.  It holds none of the rasteriser's arithmetic: it draws
surfel parameters, poses, and simulates the *scan* (the LiDAR range image the
paper treats as an input) by analytic ray casting of the
synthetic scene.  Recipes: DESIGN.md "Input recipe".
"""
from .generators import (  # noqa: F401
    Sensor,
    Workload,
    make_tiny,
    make_newer_college,
    make_kitti,
    make_large_map,
    make_mapping_batch,
    make_random_shell,
    simulate_scan,
    CONFIGS,
)
