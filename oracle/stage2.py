"""r360 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Algorithm 1, stage II (text :157): geometry-aware assignment of the occupied voxels to n
tiny networks, followed step by step in the paper's order:

    s <- S / n
    for k <- 1..n:  pop an unassigned voxel with the minimum coordinate as the anchor;
                    search s-1 nearest unassigned neighbours; assign these s voxels to network k

Readings (the paper is silent on each):
  S1  sizes: S = n*q + r  ->  the first r networks get q+1 voxels, the others q ("similar amount of occupied
      voxels", :157), so that every occupied voxel is assigned;
  S2  "minimum coordinate" = smallest linear index (iz*Ny + iy)*Nx + ix, i.e. lexicographic in (z, y, x);
  S3  "nearest" = squared Euclidean distance between voxel centres in metres, binary32, every operation
      rounded: d2 = ((dx*sx)^2 + (dy*sy)^2) + (dz*sz)^2 with dx = ix - ax (exact integer difference as a
      float), s = voxel size (box_max - box_min)/dims as the renderer computes it (one subtract, one divide);
  S4  ties in d2 go to the smaller linear index: candidates are ordered by the pair (d2, index).
"""
import numpy as np


def voxel_size(dims, box_min, box_max):
    bmin = np.asarray(box_min, np.float32)
    bmax = np.asarray(box_max, np.float32)
    return ((bmax - bmin).astype(np.float32) / np.asarray(dims, np.float32)).astype(np.float32)


def dist2(ix, iy, iz, anchor, vs):
    """S3, binary32, one rounding per operation (numpy float32 arithmetic never contracts)."""
    dx = (ix - anchor[0]).astype(np.float32) * vs[0]
    dy = (iy - anchor[1]).astype(np.float32) * vs[1]
    dz = (iz - anchor[2]).astype(np.float32) * vs[2]
    return ((dx * dx).astype(np.float32) + (dy * dy).astype(np.float32)).astype(np.float32) + (dz * dz).astype(np.float32)


def assign_subfields(occupancy, dims, box_min, box_max, occ_threshold, n):
    """Returns int32 labels[N]: network of every occupied voxel, -1 for empty voxels."""
    nx, ny, nz = (int(v) for v in dims)
    occ = np.asarray(occupancy).reshape(-1) >= occ_threshold
    lin = np.flatnonzero(occ).astype(np.int64)            # ascending linear index = ascending "coordinate" (S2)
    S = lin.size
    if n < 1 or n > max(S, 1):
        raise ValueError("n must be in [1, S]")
    vs = voxel_size(dims, box_min, box_max)
    ix = (lin % nx).astype(np.int32)
    iy = ((lin // nx) % ny).astype(np.int32)
    iz = (lin // (nx * ny)).astype(np.int32)
    labels = np.full(occ.size, -1, np.int32)
    free = np.ones(S, bool)
    q, r = divmod(S, n)
    first = 0                                             # position of the first unassigned voxel
    for k in range(n):
        size = q + (1 if k < r else 0)                    # S1
        while not free[first]:
            first += 1
        a = first                                         # the anchor (S2)
        free[a] = False
        labels[lin[a]] = k
        if size > 1:
            cand = np.flatnonzero(free)
            d2 = dist2(ix[cand], iy[cand], iz[cand], (ix[a], iy[a], iz[a]), vs)
            key = (d2.view(np.uint32).astype(np.uint64) << np.uint64(32)) | lin[cand].astype(np.uint64)   # S3, S4
            take = cand[np.argpartition(key, size - 2)[:size - 1]]
            free[take] = False
            labels[lin[take]] = k
    return labels
