"""Pins for the oracle's ray generation (Eq. 2-3; readings B1-B4)."""
import math

import numpy as np
import pytest


@pytest.mark.parametrize("W,H", [(64, 32), (512, 256), (2048, 1024), (30, 17)])
def test_eq2_round_trip(oracle, W, H):
    # pixel centre -> (phi,theta) -> Eq.2 forward must return (i+1/2, j+1/2)
    for i in [0, 1, W // 3, W // 2, W - 1]:
        for j in [0, 1, H // 2, H - 1]:
            phi, theta = oracle.pixel_to_sphere(i, j, W, H)
            assert -math.pi < phi < math.pi and -math.pi / 2 < theta < math.pi / 2
            u, v = oracle.sphere_to_pixel(phi, theta, W, H)
            assert abs(u - (i + 0.5)) < 1e-9 and abs(v - (j + 0.5)) < 1e-9


def test_eq2_forward_known_points(oracle):
    # Eq.2 itself: phi=0,theta=0 is the image centre; phi=pi/2 a quarter turn right; theta=pi/2 the top row
    W, H = 2048, 1024
    assert oracle.sphere_to_pixel(0.0, 0.0, W, H) == (W / 2, H / 2)
    u, v = oracle.sphere_to_pixel(math.pi / 2, 0.0, W, H)
    assert abs(u - 3 * W / 4) < 1e-9
    u, v = oracle.sphere_to_pixel(0.0, math.pi / 2, W, H)
    assert abs(v - 0.0) < 1e-9
    u, v = oracle.sphere_to_pixel(-math.pi, -math.pi / 2, W, H)
    assert abs(u) < 1e-9 and abs(v - H) < 1e-9


def test_directions_unit_norm_and_cardinals(oracle):
    W, H = 2048, 1024
    ident = np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], np.float32)
    rng = np.random.default_rng(0)
    for i, j in zip(rng.integers(0, W, 500), rng.integers(0, H, 500)):
        o, d = oracle.ray(ident, W, H, int(i), int(j))
        assert abs(float(np.linalg.norm(d.astype(np.float64))) - 1.0) <= 4e-7
        assert np.all(o == 0)
    tol = 2.5 * math.pi / W
    # Eq.3: phi=0,theta=0 -> +z (forward); phi=+pi/2 -> +x (right); theta=+pi/2 (top row) -> -y (y is down)
    _, d = oracle.ray(ident, W, H, W // 2, H // 2)
    assert np.allclose(d, [0, 0, 1], atol=tol)
    _, d = oracle.ray(ident, W, H, 3 * W // 4, H // 2)
    assert np.allclose(d, [1, 0, 0], atol=tol)
    _, d = oracle.ray(ident, W, H, W // 4, H // 2)
    assert np.allclose(d, [-1, 0, 0], atol=tol)
    _, d = oracle.ray(ident, W, H, 0, H // 2)
    assert np.allclose(d, [0, 0, -1], atol=tol)
    _, d = oracle.ray(ident, W, H, W // 2, 0)
    assert np.allclose(d, [0, -1, 0], atol=tol)
    _, d = oracle.ray(ident, W, H, W // 2, H - 1)
    assert np.allclose(d, [0, 1, 0], atol=tol)
    # octant: phi = pi/4 (right of centre), theta = pi/4 (above the horizon): x>0, y<0, z>0, equal |x| and z
    _, d = oracle.ray(ident, W, H, W // 2 + W // 8, H // 4)
    assert d[0] > 0 and d[1] < 0 and d[2] > 0 and abs(d[0] - d[2]) < 2 * tol
    assert abs(d[1] + math.sin(math.pi / 4)) < 2 * tol


def test_pose_rotates_and_translates(oracle):
    W, H = 512, 256
    # camera -> world: x_cam -> -y_w, y_cam -> -z_w, z_cam -> +x_w (the gravity-aligned R0 of scenegen)
    pose = np.array([0, 0, 1, 1.5, -1, 0, 0, -2.5, 0, -1, 0, 0.25], np.float32)
    o, d = oracle.ray(pose, W, H, W // 2, H // 2)
    assert np.all(o == np.array([1.5, -2.5, 0.25], np.float32))
    tol = 2.5 * math.pi / W
    assert np.allclose(d, [1, 0, 0], atol=tol)          # forward
    _, d = oracle.ray(pose, W, H, W // 2, 0)
    assert np.allclose(d, [0, 0, 1], atol=tol)          # top row looks up (world +z)
    _, d = oracle.ray(pose, W, H, 3 * W // 4, H // 2)
    assert np.allclose(d, [0, -1, 0], atol=tol)         # right of the camera


def test_trig_tables_match_libm(oracle):
    W, H = 640, 320
    sp, cp, st, ct = oracle.trig_tables(W, H)
    i = np.arange(W, dtype=np.float64)
    j = np.arange(H, dtype=np.float64)
    phi = (i + 0.5 - W / 2) * 2 * np.pi / W
    th = -(j + 0.5 - H / 2) * np.pi / H
    assert np.abs(sp - np.sin(phi)).max() < 1e-7 and np.abs(cp - np.cos(phi)).max() < 1e-7
    assert np.abs(st - np.sin(th)).max() < 1e-7 and np.abs(ct - np.cos(th)).max() < 1e-7
    # symmetry of the pixel grid: phi_i = -phi_{W-1-i}
    assert np.all(sp == -sp[::-1]) and np.all(cp == cp[::-1])
    assert np.all(st == -st[::-1]) and np.all(ct == ct[::-1])
