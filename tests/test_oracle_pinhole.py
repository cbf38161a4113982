"""Pins for the oracle's pinhole view (reading P in DESIGN.md; the paper's perspective display, PAPER.md:206,
gives no camera model).  The direction must be a unit vector, must project back to the pixel centre, and must
agree with Eq. 3 evaluated at the longitude / latitude of the same direction."""
import math

import numpy as np
import pytest

IDENT = np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], np.float32)


@pytest.mark.parametrize("W,H,fx,fy", [(1280, 720, 640.0, 640.0), (64, 36, 20.0, 30.0), (33, 17, 25.5, 19.25)])
def test_pinhole_unit_norm_and_round_trip(oracle, W, H, fx, fy):
    cx, cy = W / 2.0 + 0.25, H / 2.0 - 1.5
    rng = np.random.default_rng(1)
    for i, j in zip(rng.integers(0, W, 300), rng.integers(0, H, 300)):
        o, d = oracle.ray_pinhole(IDENT, fx, fy, cx, cy, int(i), int(j))
        d = d.astype(np.float64)
        assert np.all(o == 0)
        assert abs(np.linalg.norm(d) - 1.0) <= 4e-7
        assert d[2] > 0
        # projection of the direction lands on the pixel centre
        assert abs(fx * d[0] / d[2] + cx - (i + 0.5)) < 1e-3
        assert abs(fy * d[1] / d[2] + cy - (j + 0.5)) < 1e-3


def test_pinhole_principal_axis_and_frame(oracle):
    # the pixel whose centre is the principal point looks exactly along camera +z; x grows to the right,
    # y grows DOWNWARDS (the camera frame of Eq.3)
    _, d = oracle.ray_pinhole(IDENT, 500.0, 500.0, 100.5, 50.5, 100, 50)
    assert np.array_equal(d, np.array([0, 0, 1], np.float32))
    _, d = oracle.ray_pinhole(IDENT, 500.0, 500.0, 100.5, 50.5, 180, 50)
    assert d[0] > 0 and d[1] == 0
    _, d = oracle.ray_pinhole(IDENT, 500.0, 500.0, 100.5, 50.5, 100, 90)
    assert d[1] > 0 and d[0] == 0
    # 90 degree horizontal field of view: fx = W/2; the left image edge is 45 degrees off axis
    W = 1000
    _, d = oracle.ray_pinhole(IDENT, W / 2.0, W / 2.0, W / 2.0, 0.5, 0, 0)
    assert abs(math.degrees(math.atan2(-d[0], d[2])) - 45.0) < 0.06
    # a rotated, translated pose: third column of R is the viewing axis
    pose = np.array([0, 0, 1, 1.5, -1, 0, 0, -2.5, 0, -1, 0, 0.25], np.float32)
    o, d = oracle.ray_pinhole(pose, 500.0, 500.0, 100.5, 50.5, 100, 50)
    assert np.array_equal(o, np.array([1.5, -2.5, 0.25], np.float32))
    assert np.array_equal(d, np.array([1, 0, 0], np.float32))


def test_pinhole_agrees_with_eq3(oracle):
    # Eq.3: (x,y,z) = (cos th sin ph, -sin th, cos th cos ph).  The pinhole direction of a pixel, read as
    # longitude ph = atan2(x, z) and latitude th = -asin(y), must give back itself through Eq.3, and the
    # equirectangular pixel Eq.2 assigns to (ph, th) must see (nearly) the same direction through r360o_ray
    W, H, f = 320, 200, 210.0
    We, He = 8192, 4096
    worst = 0.0
    for i in range(0, W, 37):
        for j in range(0, H, 29):
            _, d = oracle.ray_pinhole(IDENT, f, f, W / 2.0, H / 2.0, i, j)
            d = d.astype(np.float64)
            ph, th = math.atan2(d[0], d[2]), -math.asin(d[1])
            e3 = np.array([math.cos(th) * math.sin(ph), -math.sin(th), math.cos(th) * math.cos(ph)])
            assert np.abs(e3 - d).max() < 1e-6
            u, v = oracle.sphere_to_pixel(ph, th, We, He)
            _, de = oracle.ray(IDENT, We, He, int(u), int(v))
            worst = max(worst, float(np.abs(de.astype(np.float64) - d).max()))
    assert worst < 2 * math.pi / We          # within one equirectangular pixel


def test_pinhole_tables_and_scene_camera(oracle, scene1):
    # the bulk entry points with the scene camera set to pinhole see the same rays as r360o_ray_pinhole:
    # per-pixel sample lists agree bit for bit, and equirect is restored by set_camera("equirect")
    sc = scene1
    W, H, f = 48, 27, 30.0
    s = oracle.scene_from(sc)
    base_counts, _, _ = s.samples_rows(sc.poses[0], W, H)
    s.set_camera("pinhole", f, f, W / 2.0, H / 2.0)
    counts, t, sid = s.samples_rows(sc.poses[0], W, H)
    off = np.concatenate([[0], np.cumsum(counts.astype(np.int64))])
    for (i, j) in [(0, 0), (W - 1, H - 1), (W // 2, H // 2), (5, 20), (40, 3)]:
        o, d = oracle.ray_pinhole(sc.poses[0], f, f, W / 2.0, H / 2.0, i, j)
        vox, t_in, t_out = s.walk(o, d, only_occupied=True)
        q = j * W + i
        assert counts[q] == len(vox) * s.K
        tt = t[off[q]:off[q + 1]].reshape(-1, s.K)
        K = np.float32(s.K)
        for n in range(len(vox)):
            dl = np.float32(np.float32(t_out[n] - t_in[n]) / K)
            for k in range(s.K):
                expect = np.float32(np.float32(np.float32(k) + np.float32(0.5)) * dl)  # fma below
                assert abs(float(tt[n, k]) - float(t_in[n] + expect)) <= 2e-6 * max(1.0, float(t_in[n]))
    with pytest.raises(ValueError):
        s.set_camera("pinhole", 0.0, 1.0, 0.0, 0.0)
    s.set_camera("equirect")
    again, _, _ = s.samples_rows(sc.poses[0], W, H)
    assert np.array_equal(again, base_counts)
    s.close()


def test_pinhole_end_to_end_zero_weight_closed_form(oracle, scene1):
    # zero weights: sigma = softplus(1), rgb = 0.5 inside occupied voxels -> C = 0.5 (1 - exp(-sigma L_occ)),
    # L_occ from an independent binary64 slab computation along the pinhole ray
    from test_oracle_composite import _zero_net
    sc = scene1
    W, H, f = 40, 24, 22.0
    w = np.tile(_zero_net(sc.hidden_width, sc.n_hidden, 1.0), sc.n_subfields)
    s = oracle.scene(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
                     hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, samples_per_voxel=sc.samples_per_voxel,
                     t_threshold=0.0, density_activation=1, occ_threshold=sc.occ_threshold,
                     occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield, weights=w)
    s.set_camera("pinhole", f, f, W / 2.0, H / 2.0)
    # gravity-aligned pose (scenegen's R0) at the room centre: the view is a wall, floor and ceiling
    pose = np.array([0, 0, 1, 0.1, -1, 0, 0, -0.2, 0, -1, 0, 0.05], np.float32)
    r = s.render_rows(pose, W, H)
    sigma = math.log1p(math.exp(1.0))
    occ = sc.occupied_mask()
    nx, ny, nz = sc.dims
    bmin = np.array(sc.box_min)
    vs = (np.array(sc.box_max) - bmin) / np.array(sc.dims)
    lin = np.flatnonzero(occ)
    lo = bmin + np.stack([lin % nx, (lin // nx) % ny, lin // (nx * ny)], 1) * vs
    hi = lo + vs
    worst = 0.0
    for j in range(0, H, 3):
        for i in range(0, W, 3):
            o, d = oracle.ray_pinhole(pose, f, f, W / 2.0, H / 2.0, i, j)
            o64, d64 = o.astype(np.float64), d.astype(np.float64)
            with np.errstate(divide="ignore", invalid="ignore"):
                ta, tb = (lo - o64) / d64, (hi - o64) / d64
            L = np.clip(np.maximum(ta, tb).min(1) - np.maximum(np.minimum(ta, tb).max(1), 0.0), 0, None).sum()
            expect = 0.5 * (1 - math.exp(-sigma * L))
            worst = max(worst, float(np.abs(r["rgb"][j * W + i] - expect).max()))
    assert worst < 2e-5
    s.close()
