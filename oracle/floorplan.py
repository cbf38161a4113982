"""r360 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Floorplan estimation from the occupancy map (section 5.0.2; Fig. 6), step by step:

  "We project a range of occupied voxels in the upper slicing regions (60% to 65% of the height ...) to a
   floor-parallel plane to form an initial boundary layout ... we apply simple morphological operations and segment
   out the inner boundary ... we project occupied voxels in the lower slicing region (20% to 30% of the height ...)
   to the floor-parallel plane and intersect the projected voxels with the inner boundary."

Readings (the paper names the steps but not their parameters):
  F1  the height axis is the grid's z axis (the scenes are gravity-aligned, :178); a voxel layer k belongs to the
      slice [a, b] of the height iff its centre fraction (k + 0.5)/Nz lies in [a, b];
  F2  projection = logical OR over the layers of the slice;
  F3  "simple morphological operations" = one closing with the 3x3 square: dilation (outside the image = empty),
      then erosion (outside the image = set, so that walls on the image border survive);
  F4  the interior segment (Fig. 6b, gray) = the 4-connected component of the non-wall cells that contains a seed
      cell (the viewer's position);
  F5  inner boundary (Fig. 6b, black line) = interior cells with a 4-neighbour that is not interior (cells outside
      the image are not interior);
  F6  "intersect the projected voxels with the inner boundary" (Fig. 6c) = lower-slice cells inside the interior;
  F7  floorplan = inner boundary OR those obstacle cells.
Output: uint8 image [Ny][Nx], bit 0 interior, bit 1 inner boundary, bit 2 obstacle; floorplan = bits 1|2.
"""
import numpy as np
from scipy import ndimage

INTERIOR, BOUNDARY, OBSTACLE = 1, 2, 4


def slice_layers(nz, lo, hi):
    """F1: layers whose centre fraction lies in [lo, hi] (binary64)."""
    return [k for k in range(nz) if lo <= (k + 0.5) / nz <= hi]


def floorplan(occupancy, dims, occ_threshold, seed_xy, upper=(0.60, 0.65), lower=(0.20, 0.30)):
    nx, ny, nz = (int(v) for v in dims)
    occ = (np.asarray(occupancy).reshape(nz, ny, nx) >= occ_threshold)
    up = occ[slice_layers(nz, *upper)].any(0) if slice_layers(nz, *upper) else np.zeros((ny, nx), bool)     # F2
    lowp = occ[slice_layers(nz, *lower)].any(0) if slice_layers(nz, *lower) else np.zeros((ny, nx), bool)
    sq = np.ones((3, 3), bool)
    wall = ndimage.binary_erosion(ndimage.binary_dilation(up, sq, border_value=0), sq, border_value=1)      # F3
    sx, sy = seed_xy
    if not (0 <= sx < nx and 0 <= sy < ny) or wall[sy, sx]:
        raise ValueError("seed outside the image or on a wall")
    lab, _ = ndimage.label(~wall, structure=[[0, 1, 0], [1, 1, 1], [0, 1, 0]])                              # F4
    interior = lab == lab[sy, sx]
    pad = np.pad(interior, 1, constant_values=False)
    all_nb = pad[:-2, 1:-1] & pad[2:, 1:-1] & pad[1:-1, :-2] & pad[1:-1, 2:]
    boundary = interior & ~all_nb                                                                           # F5
    obstacle = lowp & interior                                                                              # F6
    return (interior * INTERIOR + boundary * BOUNDARY + obstacle * OBSTACLE).astype(np.uint8)               # F7
