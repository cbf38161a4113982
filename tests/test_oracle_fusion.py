"""Pins for the occupancy-fusion oracle (Eq. 6): the constants the paper prints, a corridor whose
update can be written down by hand, saturation at the clamps, occupied-wins, the uncertainty reading, a sphere."""
import math

import numpy as np

from oracle.fusion import L_FREE, L_MAX, L_MIN, L_OCC_THRESHOLD, fuse, l_occ

# camera z (forward) -> world +x, camera y (down) -> world -z, camera x (right) -> world -y
POSE = np.array([0, 0, 1, 0.5, -1, 0, 0, 0.0, 0, -1, 0, 0.0], np.float32)
DIMS, BMIN, BMAX = (8, 1, 1), (0.0, -0.5, -0.5), (8.0, 0.5, 0.5)
W, H = 2048, 1024


def test_constants_printed_by_the_paper():
    # "The range of logit(p) is from -2 and 3.5 which indicates the occupied probability of 0.12 and 0.97" (:122)
    assert abs(1 / (1 + math.exp(2.0)) - 0.12) < 0.005 and abs(1 / (1 + math.exp(-3.5)) - 0.97) < 0.005
    assert L_MIN == -2 and L_MAX == 3.5
    assert abs(float(L_OCC_THRESHOLD) - math.log(0.97 / 0.03)) < 1e-6 and L_OCC_THRESHOLD < L_MAX
    # Octomap's defaults (reading O3): hit 0.7, miss 0.4; its clamping probabilities 0.1192 / 0.971 are -2 / 3.5
    assert abs(float(l_occ(0.0)) - math.log(0.7 / 0.3)) < 1e-6 and abs(float(L_FREE) - math.log(0.4 / 0.6)) < 1e-6
    assert abs(math.log(0.1192 / 0.8808) + 2.0) < 2e-3 and abs(math.log(0.971 / 0.029) - 3.5) < 2e-2
    assert l_occ(1.0) == 0 and abs(float(l_occ(0.5)) - math.log(0.6 / 0.4)) < 1e-6


def test_corridor_by_hand(oracle):
    # one ray along +x from x = 0.5, end point at x = 0.5 + 4.2 = 4.7: voxels 0..3 free, voxel 4 occupied
    L0 = np.zeros(8, np.float32)
    centre = (W // 2, H // 2)                       # looks along camera +z up to half a pixel
    L = fuse(oracle, L0, DIMS, BMIN, BMAX, POSE, W, H, _depth_one(centre, 4.2))
    exp = np.array([L_FREE] * 4 + [l_occ(0.0)] + [0, 0, 0], np.float32)
    assert np.array_equal(L, exp)
    # five more identical observations: both ends saturate at the clamps (Eq. 6 with the range of :122)
    for _ in range(5):
        L = fuse(oracle, L, DIMS, BMIN, BMAX, POSE, W, H, _depth_one(centre, 4.2))
    assert np.all(L[:4] == L_MIN) and L[4] == L_MAX and np.all(L[5:] == 0)
    assert L[4] > L_OCC_THRESHOLD                    # occupied after five hits, not after four
    L4 = L0
    for _ in range(4):
        L4 = fuse(oracle, L4, DIMS, BMIN, BMAX, POSE, W, H, _depth_one(centre, 4.2))
    assert L4[4] < L_OCC_THRESHOLD


def _depth_one(pix, v):
    d = np.zeros((H, W), np.float32)
    d[pix[1], pix[0]] = v
    return d


def test_occupied_wins_beyond_the_box_and_bad_depths(oracle):
    c = (W // 2, H // 2)
    d = _depth_one(c, 4.2)
    d[H // 2, W // 2 - 1] = 6.3                      # the neighbouring pixel passes through voxel 4 and ends in 6
    d[0, 0] = np.nan
    d[1, 1] = -3.0
    L = fuse(oracle, np.zeros(8, np.float32), DIMS, BMIN, BMAX, POSE, W, H, d)
    exp = np.array([L_FREE] * 4 + [l_occ(0.0), L_FREE, l_occ(0.0), 0], np.float32)
    assert np.array_equal(L, exp)
    # a depth beyond the box: every crossed voxel is free, nothing is occupied
    L = fuse(oracle, np.zeros(8, np.float32), DIMS, BMIN, BMAX, POSE, W, H, _depth_one(c, 50.0))
    assert np.all(L == L_FREE)


def test_uncertainty_scales_the_hit(oracle):
    c = (W // 2, H // 2)
    u = np.zeros((H, W), np.float32)
    u[c[1], c[0]] = 0.5
    L = fuse(oracle, np.zeros(8, np.float32), DIMS, BMIN, BMAX, POSE, W, H, _depth_one(c, 4.2), u)
    assert L[4] == l_occ(0.5) and abs(float(L[4]) - math.log(1.5)) < 1e-6
    u[c[1], c[0]] = 1.0
    L = fuse(oracle, np.zeros(8, np.float32), DIMS, BMIN, BMAX, POSE, W, H, _depth_one(c, 4.2), u)
    assert L[4] == 0 and np.all(L[:4] == L_FREE)


def test_sphere_of_constant_depth(oracle):
    # every pixel sees depth 1.5 from the centre of a 16^3 grid of 0.25 m voxels: the occupied voxels form the
    # shell of radius 1.5 (centre within half a voxel diagonal), everything strictly inside is free
    dims, bmin, bmax = (16, 16, 16), (-2.0, -2.0, -2.0), (2.0, 2.0, 2.0)
    pose = np.array([1, 0, 0, 0.01, 0, 1, 0, 0.02, 0, 0, 1, 0.03], np.float32)
    w, h = 96, 48
    L = fuse(oracle, np.zeros(16 ** 3, np.float32), dims, bmin, bmax, pose, w, h, np.full((h, w), 1.5, np.float32))
    idx = np.arange(16 ** 3)
    c = np.stack([idx % 16, (idx // 16) % 16, idx // 256], 1) * 0.25 - 2.0 + 0.125
    r = np.linalg.norm(c - pose.reshape(3, 4)[:, 3], axis=1)
    half_diag = 0.125 * math.sqrt(3)
    occ, free = L > 0, L < 0
    assert occ.any() and np.all(np.abs(r[occ] - 1.5) <= half_diag + 1e-6)
    assert np.all(r[free] < 1.5 + half_diag) and free[r < 1.5 - half_diag - 0.3].all()
    assert not (L != 0)[r > 1.5 + half_diag].any()
