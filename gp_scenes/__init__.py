"""Seeded synthetic driving worlds (input generator only).

This module is shared test infrastructure: it serves BOTH the CPU oracle
(`oracle/`) and the CUDA path (`paper_2606_19641_b200/`) with identical fp32
input arrays, and it holds NONE of the renderer's arithmetic (no camera,
no ray, no slab test, no shading).  It imports neither of them.

Recipe (BASELINE.json
configs[0..4]).  The scenes stand in for the paper's nuPlan-derived
scenarios (PAPER.md:127, :343 — not available here): tens to ~100 oriented
vehicle boxes, hundreds of thin lane-marking strips, a ground plane.
"""
from .generator import (  # noqa: F401
    PRIM_DTYPE, SceneConfig, CONFIGS, config, gen_world_prims, gen_dynamics,
    gen_pitch, poses_at_frames, splitmix64_stream, CLASS_SKY, CLASS_GROUND,
    CLASS_MARKING, CLASS_VEHICLE, DEFAULT_PALETTE, DEFAULT_LIGHT,
    DEFAULT_AMBIENT, CLASS_PEDESTRIAN, CLASS_CYCLIST, CLASS_OBSTACLE, CLASS_LIGHT,
    RIG_FRONT, RIG_PAPER4, rig_array, SHAPE_BOX, SHAPE_SPHERE, gen_lane_polylines,
)
