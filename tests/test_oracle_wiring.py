"""Pins for the oracle's WIRING: the functions that produce every reference image (render_pixels / render_rows,
oracle/r360_oracle.c: render_visit, render_pixel) and every reference sample list (samples_rows) are checked
against the separately pinned building blocks -- r360o_ray (Eq.2-3), r360o_ray_samples (readings C, D),
r360o_field (Eq.1, Table 4) and r360o_composite (Eq.4-5) -- with RANDOM weights and several subfields, so that
a wrong label k, a wrong position p, a wrong direction d or a skipped sample inside the render loop fails
(with zero-weight networks, the only end-to-end pin before, every subfield and every position gives the same
sigma and colour).  PAPER.md:174 (per-voxel MLP label), :91-99 (Eq.4-5); SURVEY.md 8(c) C1-C5, D, G."""
import ctypes

import numpy as np
import pytest

from scenegen import make_nondyadic_scene, mlp_param_count, weight_layout

F = np.float32
_libm = ctypes.CDLL("libm.so.6")
_libm.fmaf.restype = ctypes.c_float
_libm.fmaf.argtypes = [ctypes.c_float] * 3


def _fmaf(a, b, c):
    """IEEE binary32 fused multiply-add from libm (not the oracle's own call)."""
    return F(_libm.fmaf(float(a), float(b), float(c)))


def _compose_from_parts(oracle, s, pose, W, H, i, j, tau, pinhole=None):
    """One pixel from the pinned parts: ray -> samples -> field per sample -> Eq.4-5."""
    if pinhole is None:
        o, d = oracle.ray(pose, W, H, i, j)
    else:
        o, d = oracle.ray_pinhole(pose, *pinhole, i, j)
    t, dl, sid = s.ray_samples(pose, W, H, i, j)
    sig = np.empty(len(t))
    rgb = np.empty((len(t), 3))
    for q in range(len(t)):
        p = np.array([_fmaf(t[q], d[a], o[a]) for a in range(3)], F)       # reading D: p = fma(t, d, o)
        f = s.field(int(sid[q]), p, d)
        sig[q], rgb[q] = f[0], f[1:]
    out, full, amb = oracle.composite(sig, rgb, t, dl, float(F(tau)))     # the scene stores tau as binary32
    return out, full, amb, len(t)


def _three_subfield_scene(oracle, tau):
    """4 x 3 x 2 grid, three occupied voxels with three different networks in a row along +x, random weights
    with random biases: a ray along +x crosses all three in a known order."""
    rng = np.random.default_rng(4)
    dims = (4, 3, 2)
    occ = np.zeros(24, np.uint8)
    lab = np.full(24, -1, np.int32)
    for x, k in ((1, 2), (2, 0), (3, 1)):            # voxel (x, 1, 0) -> network k
        occ[(0 * 3 + 1) * 4 + x] = 1
        lab[(0 * 3 + 1) * 4 + x] = k
    parts = []
    for name, fo, fi in weight_layout(32, 2):
        a = np.sqrt(6.0 / (fi + fo))
        parts.append(rng.uniform(-a, a, (3, fo * fi)))
        parts.append(rng.uniform(-0.3, 0.3, (3, fo)) + (2.0 if name == "density" else 0.0))
    w = np.concatenate(parts, 1).astype(F).reshape(-1)
    assert w.size == 3 * mlp_param_count(32, 2)
    return oracle.scene(dims=dims, box_min=(0.0, 0.0, 0.0), box_max=(2.0, 1.5, 1.0), n_subfields=3, hidden_width=32,
                        n_hidden=2, samples_per_voxel=3, t_threshold=tau, density_activation=1, occ_threshold=1,
                        occupancy=occ, voxel_subfield=lab, weights=w)


def _check_pixels(oracle, s, pose, W, H, pix, tau, pinhole=None):
    px = np.array([p[0] for p in pix], np.int32)
    py = np.array([p[1] for p in pix], np.int32)
    r = s.render_pixels(pose, W, H, px, py)
    n_nonempty = 0
    for q, (i, j) in enumerate(pix):
        out, full, amb, n = _compose_from_parts(oracle, s, pose, W, H, i, j, tau, pinhole)
        n_nonempty += n > 0
        assert r["n_emitted"][q] == n
        assert r["n_used"][q] == int(out[5])
        # the render loop and r360o_composite run the same binary64 recurrence: identical after the one rounding
        # to binary32 on output (1e-12 would already separate a wrong label, position or direction: those move
        # sigma and colour by 1e-2 and more with random weights)
        assert np.allclose(r["rgb"][q], out[:3], rtol=0, atol=1e-12 + 6e-8 * np.abs(out[:3]).max())
        assert np.array_equal(r["rgb"][q], out[:3].astype(F))
        assert np.array_equal(r["rgb_full"][q], full[:3].astype(F))
        assert r["depth"][q] == F(out[3]) and r["depth_full"][q] == F(full[3])
        if n:
            assert r["ambiguity"][q] == F(amb)
    return r, n_nonempty


@pytest.mark.parametrize("tau", [1e-3, 0.3])
def test_render_pixels_equals_composite_of_field_over_ray_samples_config1(oracle, scene1, tau):
    # config 1 with its random Xavier weights, 16 subfields.  tau = 0.3 makes many rays stop early, so the
    # stopped / continued pair and n_used are exercised too.
    sc = scene1
    s = oracle.scene(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
                     hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, samples_per_voxel=sc.samples_per_voxel,
                     t_threshold=tau, density_activation=1, occ_threshold=sc.occ_threshold,
                     occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield, weights=sc.weights)
    rng = np.random.default_rng(8)
    pix = [(int(rng.integers(0, sc.W)), int(rng.integers(0, sc.H))) for _ in range(40)] + [(0, 0), (sc.W - 1, sc.H - 1)]
    r, n_nonempty = _check_pixels(oracle, s, sc.poses[0], sc.W, sc.H, pix, tau)
    assert n_nonempty == len(pix)
    if tau == 0.3:
        assert (r["n_used"] < r["n_emitted"]).any()
    # rows entry point = pixel-list entry point, all outputs
    rows = s.render_rows(sc.poses[0], sc.W, sc.H, 5, 7)
    pp = s.render_pixels(sc.poses[0], sc.W, sc.H, np.tile(np.arange(sc.W, dtype=np.int32), 2),
                         np.repeat(np.array([5, 6], np.int32), sc.W))
    for key in ("rgb", "depth", "rgb_full", "depth_full", "ambiguity", "n_emitted", "n_used"):
        assert np.array_equal(rows[key], pp[key]), key
    s.close()


def test_render_pixels_three_subfields_in_known_order(oracle):
    tau = 0.05
    s = _three_subfield_scene(oracle, tau)
    # pinhole looking along +x from x = 0.2 through the row of three occupied voxels (y in [0.5,1], z in [0,0.5])
    W, H, f = 9, 7, 20.0
    cam = (f, f, W / 2.0, H / 2.0)
    s.set_camera("pinhole", *cam)
    pose = np.array([0, 0, 1, 0.2, 1, 0, 0, 0.77, 0, 1, 0, 0.21], F)     # camera z -> world +x
    i, j = W // 2, H // 2
    t, dl, sid = s.ray_samples(pose, W, H, i, j)
    assert list(sid) == [2, 2, 2, 0, 0, 0, 1, 1, 1]                        # labels in crossing order
    pix = [(i, j), (i - 1, j), (i + 1, j + 1), (0, 0), (W - 1, H - 1), (i, j - 1)]
    r, n_nonempty = _check_pixels(oracle, s, pose, W, H, pix, tau, pinhole=cam)
    assert n_nonempty >= 4
    # the three networks really differ along this ray (otherwise a wrong label would go unnoticed)
    o, d = oracle.ray_pinhole(pose, *cam, i, j)
    p = np.array([_fmaf(t[4], d[a], o[a]) for a in range(3)], F)
    f0, f1, f2 = (s.field(k, p, d) for k in range(3))
    assert np.abs(f0 - f1).max() > 1e-2 and np.abs(f0 - f2).max() > 1e-2 and np.abs(f1 - f2).max() > 1e-2
    s.close()


def test_render_pixels_nondyadic_scene(oracle):
    sc = make_nondyadic_scene()
    s = oracle.scene_from(sc)
    rng = np.random.default_rng(12)
    for b in range(3):                                # free space, inside an occupied voxel, outside the box
        pix = [(int(rng.integers(0, sc.W)), int(rng.integers(0, sc.H))) for _ in range(12)]
        counts, _, _ = s.samples_rows(sc.poses[b], sc.W, sc.H)
        hit = np.flatnonzero(counts)                  # and pixels whose ray crosses occupied voxels
        pix += [(int(q % sc.W), int(q // sc.W)) for q in rng.choice(hit, 14, replace=False)]
        _, n_nonempty = _check_pixels(oracle, s, sc.poses[b], sc.W, sc.H, pix, sc.t_threshold)
        assert n_nonempty >= 14
    s.close()


@pytest.mark.parametrize("which", ["config1", "nondyadic0", "nondyadic1", "nondyadic2"])
def test_samples_rows_equirect_equals_ray_samples(oracle, scene1, which):
    # the bulk tap every bit-exact GPU sampler test is compared with (r360o_samples_rows: camera_tables /
    # camera_dir) against the per-pixel r360o_ray_samples (r360o_ray: pinned by tests/test_oracle_rays.py),
    # equirectangular camera: counts, t bits and subfield ids of every ray of the image
    if which == "config1":
        sc, pose = scene1, scene1.poses[0]
    else:
        sc = make_nondyadic_scene()
        pose = sc.poses[int(which[-1])]
    s = oracle.scene_from(sc)
    counts, t, sid = s.samples_rows(pose, sc.W, sc.H)
    off = np.concatenate([[0], np.cumsum(counts.astype(np.int64))])
    assert off[-1] == len(t) == len(sid)
    for j in range(sc.H):
        for i in range(sc.W):
            q = j * sc.W + i
            tt, _, ss = s.ray_samples(pose, sc.W, sc.H, i, j)
            assert counts[q] == len(tt)
            assert np.array_equal(t[off[q]:off[q + 1]].view(np.uint32), tt.view(np.uint32))
            assert np.array_equal(sid[off[q]:off[q + 1]], ss)
    # a row range is the matching slice
    c2, t2, s2 = s.samples_rows(pose, sc.W, sc.H, 3, 6)
    assert np.array_equal(c2, counts[3 * sc.W:6 * sc.W])
    assert np.array_equal(t2.view(np.uint32), t[off[3 * sc.W]:off[6 * sc.W]].view(np.uint32))
    assert np.array_equal(s2, sid[off[3 * sc.W]:off[6 * sc.W]])
    s.close()
