"""Deterministic synthetic scenes for the five configurations of BASELINE.json.

This package is *data only*: it builds the occupancy grid, the voxel->subfield
labels, the per-subfield MLP weight blobs and the camera poses that both the CPU
oracle (``oracle/``) and the CUDA library (``paper_2208_02705_b200``) consume.  It
contains none of the renderer's arithmetic (no ray casting, no positional
encoding, no MLP evaluation, no compositing) and imports neither side.

The scenes stand in for the 360Roam dataset and trained weights (PAPER.md:190,
:240), which are not available; their shapes follow the paper (2:1 panoramas,
multi-room indoor floors, camera about 1 m above the floor, n from 16 to ~4000
tiny 32/64-wide MLPs).  Recipe: DESIGN.md "Input recipe".
"""
from .rng import SplitMix64
from .scenes import CONFIGS, Scene, make_nondyadic_scene, make_scene, mlp_param_count, weight_layout

__all__ = ["SplitMix64", "CONFIGS", "Scene", "make_scene", "make_nondyadic_scene", "mlp_param_count", "weight_layout"]
