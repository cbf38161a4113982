"""-m gpu: r360_occupancy_fuse against the oracle.  Flags and a minimum decide every voxel, then one binary32 add and
a clamp: the grids must be equal bit for bit."""
import numpy as np
import pytest

from conftest import get_scene

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def r360():
    import torch
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def _eq(a, b):
    return np.array_equal(np.asarray(a, np.float32).view(np.uint32), np.asarray(b, np.float32).view(np.uint32))


def test_corridor_and_saturation(r360, oracle):
    from oracle.fusion import fuse
    pose = np.array([0, 0, 1, 0.5, -1, 0, 0, 0.0, 0, -1, 0, 0.0], np.float32)
    dims, bmin, bmax, W, H = (8, 1, 1), (0.0, -0.5, -0.5), (8.0, 0.5, 0.5), 2048, 1024
    d = np.zeros((H, W), np.float32)
    d[H // 2, W // 2] = 4.2
    d[H // 2, W // 2 - 1] = 6.3
    d[0, 0] = np.nan
    d[1, 1] = -1.0
    Lg = Lo = np.zeros(8, np.float32)
    for _ in range(6):
        Lo = fuse(oracle, Lo, dims, bmin, bmax, pose, W, H, d)
        Lg = r360.occupancy_fuse(Lg, dims, bmin, bmax, pose, W, H, d)
        assert _eq(Lg, Lo)
    assert Lg[4] == 3.5 and Lg[0] == -2.0


@pytest.mark.parametrize("seed", [0, 1])
def test_random_depths_and_uncertainty(r360, oracle, seed):
    from oracle.fusion import fuse
    rng = np.random.default_rng(seed)
    dims, bmin, bmax = (20, 14, 9), (-2.0, -1.5, -1.0), (2.1, 1.4, 0.9)
    W, H = 96, 48
    yaw = rng.uniform(0, 6.28)
    c, s = np.cos(yaw), np.sin(yaw)
    R0 = np.array([[0, 0, 1], [-1, 0, 0], [0, -1, 0]], np.float64)
    R = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]]) @ R0
    o = rng.uniform(-0.5, 0.5, 3)
    pose = np.concatenate([R, o[:, None]], 1).astype(np.float32).reshape(12)
    L0 = rng.uniform(-2, 3.5, dims[0] * dims[1] * dims[2]).astype(np.float32)
    depth = rng.uniform(0.2, 3.0, (H, W)).astype(np.float32)
    depth[rng.random((H, W)) < 0.1] = 0.0                     # missing measurements
    depth[rng.random((H, W)) < 0.05] = 40.0                   # beyond the box
    unc = rng.uniform(-0.2, 1.2, (H, W)).astype(np.float32)   # clamped to [0, 1] by both sides
    for u in (None, unc):
        ref = fuse(oracle, L0, dims, bmin, bmax, pose, W, H, depth, u)
        got = r360.occupancy_fuse(L0, dims, bmin, bmax, pose, W, H, depth, u)
        assert _eq(got, ref)
        assert (got != L0).sum() > 500


def test_recovers_the_scene_from_its_own_depth(r360, oracle):
    """Stage I on a synthetic stand-in: the depth of the FIRST surface seen from a few poses inside config 1's room
    (computed with the oracle's walk) is fused; after six observations the voxels above the 0.97 threshold are all
    truly occupied and include the first-hit voxels of the first pose."""
    from oracle.fusion import L_OCC_THRESHOLD
    sc = get_scene(1, with_weights=False)
    ora = oracle.scene_from(get_scene(1))
    W, H = 128, 64
    occ = np.asarray(sc.occupancy).reshape(-1) >= sc.occ_threshold
    base = np.asarray(sc.poses[0], np.float32).reshape(3, 4)
    L = np.zeros(occ.size, np.float32)
    first_hits = None
    for k in range(6):
        pose = base.copy()
        pose[:, 3] += np.array([0.3 * (k % 3 - 1), 0.25 * (k // 3), 0.0], np.float32)
        depth = np.zeros((H, W), np.float32)
        hits = []
        for j in range(H):
            for i in range(W):
                o, d = oracle.ray(pose.reshape(12), W, H, i, j)
                vox, t_in, t_out = ora.walk(o, d, only_occupied=True, cap=4096)
                if len(vox):
                    depth[j, i] = np.float32(0.5) * (t_in[0] + t_out[0])      # inside the first occupied voxel
                    hits.append(int(vox[0]))
        if first_hits is None:
            first_hits = np.unique(hits)
        L = r360.occupancy_fuse(L, sc.dims, sc.box_min, sc.box_max, pose.reshape(12), W, H, depth)
    found = L > L_OCC_THRESHOLD
    assert found.sum() > 300 and occ[found].all()             # no false positives
    assert (L[first_hits] > 0).all()                          # everything the first pose saw carries occupied evidence
    assert (L[~occ] <= 0).all()
    ora.close()


def test_resident_grid_equals_repeated_single_observations(r360, oracle):
    """r360_fusion_*: the grid stays on the device over a sequence of observations; the result equals the oracle's
    observation-by-observation fusion bit for bit, and the thresholded occupancy is reading O5."""
    from oracle.fusion import L_OCC_THRESHOLD, fuse
    rng = np.random.default_rng(4)
    dims, bmin, bmax = (24, 18, 10), (-2.0, -1.5, -1.0), (2.1, 1.4, 0.9)
    W, H = 80, 40
    R0 = np.array([[0, 0, 1], [-1, 0, 0], [0, -1, 0]], np.float64)
    fu = r360.Fusion(dims, bmin, bmax)
    Lo = np.zeros(dims[0] * dims[1] * dims[2], np.float32)
    for k in range(5):
        yaw = rng.uniform(0, 6.28)
        c, s = np.cos(yaw), np.sin(yaw)
        R = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]]) @ R0
        pose = np.concatenate([R, rng.uniform(-0.4, 0.4, 3)[:, None]], 1).astype(np.float32).reshape(12)
        depth = rng.uniform(0.3, 2.5, (H, W)).astype(np.float32)
        unc = rng.uniform(0, 1, (H, W)).astype(np.float32) if k % 2 else None
        fu.fuse(pose, W, H, depth, unc)
        Lo = fuse(oracle, Lo, dims, bmin, bmax, pose, W, H, depth, unc)
    Lg, occ = fu.read(occupancy=True)
    assert _eq(Lg, Lo)
    assert np.array_equal(occ, np.where(Lo > np.float32(L_OCC_THRESHOLD), 255, 0).astype(np.uint8))
    # an initial grid, and a second image size on the same handle
    fu2 = r360.Fusion(dims, bmin, bmax, logodds_init=Lo)
    depth = rng.uniform(0.3, 2.5, (33, 70)).astype(np.float32)
    fu2.fuse(pose, 70, 33, depth)
    assert _eq(fu2.read(), fuse(oracle, Lo, dims, bmin, bmax, pose, 70, 33, depth))
    fu.close()
    fu2.close()


def test_fusion_fed_by_the_renderers_own_depth(r360, oracle):
    """the renderer's depth output (a DEVICE buffer, Eq. 4's radial distance) goes straight into
    the fusion (r360_fusion_fuse_device) -- the synthetic stand-in for 360NeRF's depth panoramas.  Same grid as
    fusing the image after a round trip through the host."""
    from oracle.fusion import fuse
    sc = get_scene(1)
    gpu = r360.scene_from(sc)
    W, H = 128, 64
    rgb, depth = gpu.render(sc.poses[0], W, H)
    import torch
    torch.cuda.synchronize()
    fu = r360.Fusion(sc.dims, sc.box_min, sc.box_max)
    fu.fuse(sc.poses[0], W, H, depth.contiguous())
    ref = fuse(oracle, np.zeros(int(np.prod(sc.dims)), np.float32), sc.dims, sc.box_min, sc.box_max, sc.poses[0], W, H,
               depth.cpu().numpy())
    assert _eq(fu.read(), ref)
    assert (ref != 0).sum() > 1000
    fu.close()
    gpu.close()
