"""Seeded synthetic inputs for the sparse-voxel rasterizer (scenes, cameras, targets).

This package is shared by the tests of the CPU oracle and of the CUDA path and by bench.py.
It holds NONE of the method's arithmetic (no projection, no compositing, no SH basis, no loss):
only NumPy `Generator(PCG64(seed))` draws and the octree/camera *layout* of BASELINE.json's five
configs. The scenes stand in for Mip-NeRF 360 / Tanks & Temples, which are
not in the container: only voxel counts, resolutions and camera layouts follow the paper.

See DESIGN.md "Input recipe" for every parameter.
"""
from .scenes import (Scene, Camera, Config, look_at_camera, make_config, perturbed_copy,
                     tiny_scene, uniform_grid_scene, CONFIG_NAMES)

__all__ = ["Scene", "Camera", "Config", "look_at_camera", "make_config", "perturbed_copy",
           "tiny_scene", "uniform_grid_scene", "CONFIG_NAMES"]
