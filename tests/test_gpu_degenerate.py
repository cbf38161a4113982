"""-m gpu: parity cases the BASELINE.json configs cannot show ("parity tests never leave dyadic
grids"): a non-dyadic anisotropic grid whose planes are not representable in binary32 (a contracted or reordered
plane / distance formula in the CUDA walk would change bits there), rays parallel to one and to TWO grid axes,
a camera inside an occupied voxel, a camera outside the box, and 1-pixel-wide / 1-pixel-high pinhole images.
Bars as everywhere: counts, t bits and subfield ids exact; fp32 1e-4; bf16 2e-3 (BASELINE.json north_star).
Readings C1-C5, D."""
import numpy as np
import pytest

from conftest import get_scene
from gpu_util import AMB_BAND, check_image, ray_major_index

pytestmark = pytest.mark.gpu
F = np.float32


@pytest.fixture(scope="module")
def r360():
    import torch
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def _samples_equal(gpu, ora, pose, W, H):
    counts, offsets, t, sid = gpu.debug_samples(pose, W, H)
    oc, ot, osid = ora.samples_rows(pose, W, H)
    counts, offsets = counts.cpu().numpy().view(np.uint32), offsets.cpu().numpy().view(np.uint32)
    assert np.array_equal(counts, oc)
    idx = ray_major_index(counts, offsets)
    assert np.array_equal(t.cpu().numpy().view(np.uint32)[idx], ot.view(np.uint32))
    assert np.array_equal(sid.cpu().numpy()[idx], osid)
    return oc


def _images_within_bars(gpu, ora, sc, pose, W, H):
    ref = ora.render_rows(pose, W, H)
    gpu.set_precision("fp32")
    rgb, depth = gpu.render(pose, W, H)
    assert gpu.stats().samples_emitted == int(ref["n_emitted"].sum())
    e32 = check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 1e-4)
    gpu.set_precision("bf16")
    rgb, depth = gpu.render(pose, W, H)
    t_max = float(np.linalg.norm(np.array(sc.box_max) - np.array(sc.box_min)))
    e16 = check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 2e-3, amb_band=AMB_BAND["bf16"], depth_tol=2e-3 * t_max)
    gpu.set_precision("fp32")
    return e32, e16


@pytest.mark.parametrize("K", [5, 8, 12])
def test_nondyadic_scene_equirect(r360, oracle, K):
    """Box [-1.3, 2.07] x [0.2, 3.9] x [-0.7, 1.13], 37 x 29 x 11 voxels, scattered occupancy, general rotation;
    pose 0 in free space, pose 1 inside an occupied voxel, pose 2 outside the box.  K = 5 and 12 take the
    division in delta = (t_out - t_in) / K, K = 8 the product with the exact reciprocal."""
    from scenegen import make_nondyadic_scene
    sc = make_nondyadic_scene(K=K)
    gpu, ora = r360.scene_from(sc), oracle.scene_from(sc)
    for b in range(3):
        oc = _samples_equal(gpu, ora, sc.poses[b], sc.W, sc.H)
        assert oc.sum() > 0
        if b == 1:
            # inside an occupied voxel: every ray starts with a hit at t_in = 0
            counts, offsets, t, sid = gpu.debug_samples(sc.poses[b], sc.W, sc.H)
            assert int(counts.min()) >= K
        e32, e16 = _images_within_bars(gpu, ora, sc, sc.poses[b], sc.W, sc.H)
        print(f"nondyadic K={K} pose {b}: fp32 {e32[0]:.2e}/{e32[1]:.2e}  bf16 {e16[0]:.2e}")
    # ragged sizes and the chunked path on the same grid
    for (W, H) in [(1, 1), (53, 7), (3, 121)]:
        _samples_equal(gpu, ora, sc.poses[0], W, H)
    gpu.set_chunk_rays(700)
    _samples_first = gpu.render(sc.poses[0], sc.W, sc.H)[0].clone()
    gpu.set_chunk_rays(1 << 22)
    import torch
    assert torch.equal(_samples_first, gpu.render(sc.poses[0], sc.W, sc.H)[0])
    gpu.close()
    ora.close()


def test_nondyadic_scene_pinhole_and_wavefront(r360, oracle):
    from scenegen import make_nondyadic_scene
    sc = make_nondyadic_scene()
    gpu, ora = r360.scene_from(sc), oracle.scene_from(sc)
    cam = ("pinhole", 61.3, 58.9, 40.2, 22.7)
    gpu.set_camera(*cam)
    ora.set_camera(*cam)
    for b in range(3):
        _samples_equal(gpu, ora, sc.poses[b], 80, 45)
        _images_within_bars(gpu, ora, sc, sc.poses[b], 80, 45)
    rgb, depth = gpu.render(sc.poses[1], 80, 45)
    rgb, depth = rgb.clone(), depth.clone()
    gpu.set_wavefront(True)
    rgb_w, depth_w = gpu.render(sc.poses[1], 80, 45)
    import torch
    assert torch.equal(rgb, rgb_w) and torch.equal(depth, depth_w)
    gpu.close()
    ora.close()


# camera z (the optical axis) mapped to the six world axis directions: column 2 of R
_AXIS_R = {
    "+z": [[1, 0, 0], [0, 1, 0], [0, 0, 1]],
    "-z": [[-1, 0, 0], [0, 1, 0], [0, 0, -1]],
    "+x": [[0, 0, 1], [1, 0, 0], [0, 1, 0]],
    "-x": [[0, 0, -1], [0, 1, 0], [1, 0, 0]],
    "+y": [[1, 0, 0], [0, 0, 1], [0, -1, 0]],
    "-y": [[0, 1, 0], [0, 0, -1], [-1, 0, 0]],
}


@pytest.mark.parametrize("axis", sorted(_AXIS_R))
@pytest.mark.parametrize("which", ["config1_on_lattice", "config1_off_lattice", "nondyadic"])
def test_rays_parallel_to_two_axes(r360, oracle, which, axis):
    """Pinhole with cx = i + 1/2, cy = j + 1/2 and an axis-permutation R: the centre pixel's direction is exactly a
    world axis (parallel to the two others, reading C1: tn = -inf, tf = +inf there), the centre row and column are
    parallel to one axis.  'on_lattice' puts the origin exactly ON grid planes of the parallel axes."""
    from scenegen import make_nondyadic_scene
    if which == "nondyadic":
        sc = make_nondyadic_scene()
        o = sc.poses[0].reshape(3, 4)[:, 3]
    else:
        sc = get_scene(1)
        o = np.array([0.0, 0.0, 0.0] if which == "config1_on_lattice" else [0.337, -1.113, 0.291])
    W, H = 33, 17
    cam = ("pinhole", 20.0, 20.0, 16.5, 8.5)
    pose = np.concatenate([np.array(_AXIS_R[axis], np.float64), np.asarray(o, np.float64).reshape(3, 1)], 1).astype(F).reshape(12)
    gpu, ora = r360.scene_from(sc), oracle.scene_from(sc)
    gpu.set_camera(*cam)
    ora.set_camera(*cam)
    _, d = oracle.ray_pinhole(pose, *cam[1:], 16, 8)
    assert sorted(np.abs(d).tolist()) == [0.0, 0.0, 1.0]           # exactly along a world axis
    _, d = oracle.ray_pinhole(pose, *cam[1:], 3, 8)
    assert int((d == 0).sum()) == 1                                  # the centre row: parallel to one axis
    oc = _samples_equal(gpu, ora, pose, W, H)
    if which != "nondyadic":
        assert oc[8 * W + 16] > 0                                    # the axis ray ends in the room shell
    _images_within_bars(gpu, ora, sc, pose, W, H)
    gpu.close()
    ora.close()


def test_camera_inside_an_occupied_voxel_config1(r360, oracle, scene1):
    sc = scene1
    nx, ny, nz = sc.dims
    occ = np.flatnonzero(sc.occupied_mask())
    vs = (np.array(sc.box_max) - np.array(sc.box_min)) / np.array(sc.dims)
    gpu, ora = r360.scene_from(sc), oracle.scene_from(sc)
    for lin, frac in ((int(occ[len(occ) // 2]), (0.31, 0.57, 0.73)), (int(occ[7]), (0.5, 0.5, 0.5)),
                      (int(occ[-3]), (0.0, 0.25, 0.999))):               # the last one sits ON a voxel face
        idx = np.array([lin % nx, (lin // nx) % ny, lin // (nx * ny)], np.float64)
        o = np.array(sc.box_min) + (idx + np.array(frac)) * vs
        pose = sc.poses[0].copy()
        pose[3], pose[7], pose[11] = o
        oc = _samples_equal(gpu, ora, pose, 64, 32)
        if frac[0] > 0:
            assert oc.min() >= sc.samples_per_voxel                  # every ray starts inside an occupied voxel
        _images_within_bars(gpu, ora, sc, pose, 64, 32)
    gpu.close()
    ora.close()


@pytest.mark.parametrize("W,H", [(1, 1), (1, 64), (97, 1), (1, 2)])
def test_pinhole_one_pixel_wide_or_high(r360, oracle, scene1, W, H):
    sc = scene1
    cam = ("pinhole", 30.0, 25.0, W / 2.0, H / 2.0)
    gpu, ora = r360.scene_from(sc), oracle.scene_from(sc)
    gpu.set_camera(*cam)
    ora.set_camera(*cam)
    pose = get_scene(2).poses[0].copy()          # a gravity-aligned pose (config 2's), inside config 1's room
    pose[3], pose[7], pose[11] = 0.4, -0.3, 0.1
    oc = _samples_equal(gpu, ora, pose, W, H)
    assert oc.sum() > 0
    _images_within_bars(gpu, ora, sc, pose, W, H)
    gpu.close()
    ora.close()
