"""r360 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Progressive probabilistic occupancy (PAPER.md:117-128, Eq. 6; Algorithm 1 stage I, :139-146): one observation =
a depth panorama (Eq. 4) and, optionally, an uncertainty panorama from one pose, fused into the log-odds grid

    logit(p | z_1:t) = logit(p | z_1:t-1) + logit(p | z_t),   logit in [-2, 3.5],   occupied iff p > 0.97.

The paper adopts Octomap [43] for the rest (:128) and gives no measurement model.  Readings:
  O1  natural-log odds, clamped after every observation: L <- min(3.5, max(-2, L + l));
  O2  Octomap's scan insertion: per observation every voxel is updated at most once -- "occupied" if the end point
      of at least one ray lies in it, else "free" if at least one ray crosses it before its end point;
  O3  l_free = ln(0.4/0.6), l_occ = ln(p/(1-p)) with p = 0.7: Octomap's defaults, whose default clamping
      probabilities 0.1192 / 0.971 ARE the paper's -2 / 3.5.  With an uncertainty map u in [0,1] ("the measurement
      probability will be changed according to the current 360NeRF estimation", :128) p = 0.5 + 0.2 (1 - u), u the
      smallest uncertainty among the rays that end in the voxel (u = 0 without a map);
  O4  rays = the panorama's rays (Eq. 2-3, readings B); a ray ends at distance D = depth[pixel] (Eq. 4's radial
      distance); pixels with D <= 0 or non-finite D are skipped; voxels come from the walk of reading C: a crossed
      voxel [t_in, t_out) with t_in < D is free, unless t_in <= D < t_out, which makes it the end-point voxel;
  O5  occupied iff L > ln(0.97/0.03) (:122).
Arithmetic of the update: binary32, one add, then the clamp.
"""
import math

import numpy as np

L_MIN, L_MAX = np.float32(-2.0), np.float32(3.5)
L_FREE = np.float32(math.log(0.4 / 0.6))
L_OCC_THRESHOLD = np.float32(math.log(0.97 / 0.03))


def l_occ(u):
    """O3, binary32: p = 0.5 + 0.2 (1 - u); l = ln(p / (1 - p)) evaluated in binary64 and rounded once."""
    p = np.float32(0.5) + np.float32(0.2) * (np.float32(1.0) - np.float32(u))
    return np.float32(math.log(float(p) / (1.0 - float(p))))


def fuse(oracle, logodds, dims, box_min, box_max, pose, W, H, depth, uncertainty=None):
    """One observation.  oracle: oracle.Oracle (its ray / walk follow readings B and C).  Returns the new grid."""
    nx, ny, nz = (int(v) for v in dims)
    N = nx * ny * nz
    scene = oracle.scene(dims=dims, box_min=box_min, box_max=box_max, n_subfields=1, occupancy=np.zeros(N, np.uint8),
                         voxel_subfield=np.zeros(N, np.int32),
                         weights=np.zeros(int(oracle.params_per_subfield(hidden_width=32, n_hidden=2)), np.float32),
                         occ_threshold=1)
    depth = np.asarray(depth, np.float32).reshape(H, W)
    unc = None if uncertainty is None else np.asarray(uncertainty, np.float32).reshape(H, W)
    free = np.zeros(N, bool)
    occ = np.zeros(N, bool)
    umin = np.full(N, np.float32(1.0))
    with np.errstate(invalid="ignore"):
        valid = np.isfinite(depth) & (depth > 0)                       # O4: the other pixels are skipped
    for j, i in zip(*np.nonzero(valid)):
        if True:
            D = depth[j, i]
            o, d = oracle.ray(pose, W, H, int(i), int(j))
            vox, t_in, t_out = scene.walk(o, d, only_occupied=False, cap=nx + ny + nz + 8)
            for v, a, b in zip(vox, t_in, t_out):
                if not a < D:
                    break
                if D < b:                                             # the end point lies in this voxel
                    occ[v] = True
                    u = np.float32(0.0) if unc is None else min(max(unc[j, i], np.float32(0.0)), np.float32(1.0))
                    umin[v] = min(umin[v], u)
                    break
                free[v] = True
    scene.close()
    L = np.asarray(logodds, np.float32).reshape(-1).copy()
    for v in np.flatnonzero(occ | free):                              # O2: occupied wins
        inc = l_occ(umin[v]) if occ[v] else L_FREE
        L[v] = min(L_MAX, max(L_MIN, np.float32(L[v] + inc)))         # O1
    return L
