"""Seeded synthetic input generators shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no back-projection, TSDF update, trilinear
sampling, fitness or swarm update).  It only manufactures inputs: analytic scenes, ray-cast depth
frames, camera trajectories, analytic TSDF fills and pre-sampled particle swarm templates (PST).
Both the CPU oracle (``oracle/``) and the CUDA path (``paper_2105_05600_b200``) receive the arrays
produced here; neither imports the other.  Recipes follow SURVEY.md section 8(d) and are restated in
DESIGN.md ("Input recipe").
"""
from .scene import Scene, make_scene, scene_sdf, analytic_volume
from .camera import (look_at, raycast_depth, add_noise, random_free_position, compose_delta,
                     rot_axis_angle, rotation_angle_deg)
from .pst import sample_pst, sample_pst_poisson
from .configs import (BASE_SEED, config_seed, make_config1, make_config2_inputs, make_config3_scene,
                      make_config3_trajectory, make_config5_poses, render_frame, INTRINSICS)

__all__ = [
    "Scene", "make_scene", "scene_sdf", "analytic_volume", "look_at", "raycast_depth", "add_noise",
    "random_free_position", "compose_delta", "rot_axis_angle", "rotation_angle_deg", "sample_pst", "sample_pst_poisson",
    "BASE_SEED", "config_seed", "make_config1", "make_config2_inputs", "make_config3_scene",
    "make_config3_trajectory", "make_config5_poses", "render_frame", "INTRINSICS",
]
