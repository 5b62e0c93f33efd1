"""Seeded synthetic inputs for the DrivingVoxels hot path (shared by oracle tests and CUDA tests).

This package depends on NumPy only and contains no arithmetic of the rendering method.
"""
from .configs import Camera, Scene, make_config, tiny_random_scene, look_yaw, pose_yaw  # noqa: F401
from .octree import Octree, encode, decode, make_octree  # noqa: F401
