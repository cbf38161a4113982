"""r360 -- B200-native equirectangular renderer for radiance fields made of thousands of
tiny MLPs (render hot path of 360Roam, arxiv 2208.02705).

Thin ctypes binding over the C ABI in include/r360.h (libr360.so, hand-written CUDA for
sm_100a).  Argument marshalling only: every step of the path runs in the CUDA kernels.
There is no CPU fallback; loading fails loudly if the library is missing.
"""
from .binding import (Fusion, fusion_fuse_static, STATIC_MAX_VOXELS, STATIC_MAX_W, STATIC_MAX_H, R360Error, Scene, Stats, assign_subfields, floorplan, occupancy_fuse, lib,
                      lib_path, measure_fp32_fma, params_per_subfield, scene_from,
                      version, STATUS)

__all__ = ["Fusion", "fusion_fuse_static", "STATIC_MAX_VOXELS", "STATIC_MAX_W", "STATIC_MAX_H", "R360Error", "Scene", "Stats", "assign_subfields", "floorplan", "occupancy_fuse", "lib", "lib_path", "measure_fp32_fma", "params_per_subfield", "scene_from", "version",
           "STATUS"]
