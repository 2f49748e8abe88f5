"""Seeded synthetic inputs (scenes, cameras, upstream gradients) for the 2DGS renderer.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2506_00970_b200/`).  It holds none of the method's arithmetic: no
projection, no binning, no blending.  It only draws numbers from a
counter-based SplitMix64 stream and arranges them into the arrays that
SURVEY.md §8(d) / DESIGN.md "input recipe" describe.

The paper's RGB-D datasets (Replica, TUM-RGBD, ScanNet) are not
available; these scenes take only their shapes (image sizes, intrinsics,
room-scale geometry, centimetre-scale surface-aligned splats).
"""
from .rng import SplitMix
from .scenes import (Scene, Camera, make_config, tiny_scene, room_scene, stress_scene, stress_camera,
                     upstream_normal, look_at, se3_exp, perturb_pose, CONFIG_NAMES)

__all__ = ["SplitMix", "Scene", "Camera", "make_config", "tiny_scene", "room_scene", "stress_scene", "stress_camera",
           "upstream_normal", "look_at", "se3_exp", "perturb_pose", "CONFIG_NAMES"]
