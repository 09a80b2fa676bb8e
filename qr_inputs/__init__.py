"""Seeded synthetic inputs for the Q-Render hot path.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2512_20927_b200/``).  It holds none of the method's arithmetic: it only
draws Gaussian parameters, features, cameras and upstream gradients with the
shapes and distributions of ``BASELINE.json``'s five configs (recipe in
DESIGN.md, "Input recipe").
"""
from .scenes import Camera, Scene, CONFIGS, make_scene, make_camera, look_at, pose_on_circle

__all__ = ["Camera", "Scene", "CONFIGS", "make_scene", "make_camera", "look_at", "pose_on_circle"]
