"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the method (no voxel keys, no hashing, no
nearest-neighbour search, no GICP): only point clouds, poses and LiDAR-shaped
scans produced by analytic ray casting.  Both `oracle/` and
`paper_2606_26010_b200/` are fed the fp32 arrays produced here; neither of them
imports the other.  Recipes are described in DESIGN.md ("Input recipe") and
follow SURVEY.md section 8(d) / BASELINE.json configs C1..C5.
"""
from .generators import (  # noqa: F401
    pose_from_rpy_t,
    pose_identity,
    pose_inverse,
    pose_compose,
    pose_apply,
    perturb_pose,
    c1_tiny,
    UrbanScene,
    RaceTrack,
    c2_single_frame,
    c3_racing_frame,
    c4_insert_stress,
    c5_nn_sweep,
    motion_distorted_scan,
)
