"""-m gpu: r360_fusion_fuse_static, the allocation-free form of the Eq. 6 fusion step, against the existing
r360_fusion handle path.

Why the entry point exists: some users of this library cannot let it call cudaMalloc -- their process has given the
whole GPU to its own pool, or they run in a frame loop where an allocation's device-wide stall is not acceptable, or
allocation is forbidden at that moment.  The static variant keeps its per-voxel scratch, tables and pose in one fixed
device array inside libr360.so instead, so it has a size limit and all calls on a device share that array.

What is checked: the same kernels run on both paths, so the log-odds grids must be equal bit for bit (the tolerance
of tests/test_gpu_fusion.py), and they must stay equal over calls IN A ROW -- the second call finds the first call's
leftovers in the shared array (other grid size, other image size, with and without an uncertainty image), which is
what the per-call reset has to deal with.  This file sorts last on purpose: pytest -x stops at the first failure,
and a failure here must not hide the other tests.  It does not depend on their state (it passes alone in a fresh
process, where the first call also does the per-device set-up, and after the others)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

R0 = np.array([[0, 0, 1], [-1, 0, 0], [0, -1, 0]], np.float64)     # camera looking along world +x, z up


@pytest.fixture(scope="module")
def r360():
    import torch
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def _pose(rng):
    yaw = rng.uniform(0, 6.28)
    c, s = np.cos(yaw), np.sin(yaw)
    R = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]]) @ R0
    return np.concatenate([R, rng.uniform(-0.4, 0.4, 3)[:, None]], 1).astype(np.float32).reshape(12)


def _observation(rng, W, H, with_unc):
    depth = rng.uniform(0.3, 2.5, (H, W)).astype(np.float32)
    depth[rng.random((H, W)) < 0.1] = 0.0                          # missing measurements are skipped
    unc = rng.uniform(-0.2, 1.2, (H, W)).astype(np.float32) if with_unc else None
    return depth, unc


def _bits(a):
    return np.ascontiguousarray(a, np.float32).view(np.uint32)


def test_two_calls_in_a_row_equal_the_handle_path(r360):
    import torch
    rng = np.random.default_rng(11)
    bmin, bmax = (-2.0, -1.5, -1.0), (2.1, 1.4, 0.9)
    # (grid, image size, uncertainty image?) of consecutive calls: the big grid first, so the small one that follows
    # runs over scratch the big one has used; then the image size changes back (tables rebuilt twice)
    plan = [((40, 30, 17), (96, 48), True), ((40, 30, 17), (96, 48), False),
            ((24, 18, 10), (70, 33), True), ((24, 18, 10), (96, 48), False)]
    grids = {}
    for dims, (W, H), with_unc in plan:
        N = dims[0] * dims[1] * dims[2]
        if dims not in grids:
            L0 = rng.uniform(-2, 3.5, N).astype(np.float32)
            grids[dims] = (torch.from_numpy(L0).cuda(), r360.Fusion(dims, bmin, bmax, logodds_init=L0), L0)
        L_static, handle, L0 = grids[dims]
        pose = _pose(rng)
        depth, unc = _observation(rng, W, H, with_unc)
        d_dev = torch.from_numpy(depth).cuda()
        u_dev = None if unc is None else torch.from_numpy(unc).cuda()
        r360.fusion_fuse_static(L_static, dims, bmin, bmax, pose, W, H, d_dev, u_dev)    # default stream, like the handle
        handle.fuse(pose, W, H, d_dev, u_dev)
        torch.cuda.synchronize()
        got, ref = L_static.cpu().numpy(), handle.read()
        assert np.array_equal(_bits(got), _bits(ref)), (dims, W, H, with_unc)
        assert (got != L0).sum() > 500                              # the observation did change the grid
    for _, handle, _ in grids.values():
        handle.close()


def test_same_observation_twice_accumulates_like_the_handle(r360):
    """Back-to-back calls with nothing in between (no synchronisation, same stream): the second starts from the
    first one's result and from a scratch array the first has just used."""
    import torch
    rng = np.random.default_rng(12)
    dims, bmin, bmax, W, H = (20, 14, 9), (-2.0, -1.5, -1.0), (2.1, 1.4, 0.9), 64, 32
    pose = _pose(rng)
    depth, unc = _observation(rng, W, H, True)
    d_dev, u_dev = torch.from_numpy(depth).cuda(), torch.from_numpy(unc).cuda()
    L = torch.zeros(dims[0] * dims[1] * dims[2], device="cuda")
    handle = r360.Fusion(dims, bmin, bmax)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    for _ in range(2):
        r360.fusion_fuse_static(L, dims, bmin, bmax, pose, W, H, d_dev, u_dev, stream=s)
        handle.fuse(pose, W, H, d_dev, u_dev)
    s.synchronize()
    torch.cuda.synchronize()
    ref = handle.read()
    assert np.array_equal(_bits(L.cpu().numpy()), _bits(ref))
    assert ref.max() > 1.6 and ref.min() < -0.8                    # both observations counted (one gives 0.85 / -0.41)
    handle.close()


def test_sizes_beyond_the_static_scratch_are_refused(r360):
    import torch
    assert r360.STATIC_MAX_VOXELS == 8 << 20 and (r360.STATIC_MAX_W, r360.STATIC_MAX_H) == (4096, 2048)
    bmin, bmax = (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    pose = np.concatenate([R0, np.zeros((3, 1))], 1).astype(np.float32).reshape(12)

    class Fake:                                                     # sizes only: the call must refuse before any access
        is_cuda = True

        def __init__(self, n, ptr):
            self._n, self._p = n, ptr

        def is_contiguous(self): return True
        def numel(self): return self._n
        def element_size(self): return 4
        def data_ptr(self): return self._p

    small = torch.zeros(64, device="cuda")
    p = small.data_ptr()
    for dims, (W, H) in [((2049, 64, 64), (8, 8)), ((4, 4, 4), (4097, 8)), ((4, 4, 4), (8, 2049))]:
        N = dims[0] * dims[1] * dims[2]
        with pytest.raises(r360.R360Error) as e:
            r360.fusion_fuse_static(Fake(N, p), dims, bmin, bmax, pose, W, H, Fake(W * H, p))
        assert e.value.status == 6 and "static scratch" in str(e.value) and "8388608" in str(e.value)
    torch.cuda.synchronize()
    assert float(small.abs().sum()) == 0.0                          # nothing was written
    # the largest grid that is allowed goes through (8 Mi voxels exactly), and touches nothing outside its inputs
    dims = (256, 256, 128)
    L = torch.zeros(dims[0] * dims[1] * dims[2], device="cuda")
    depth = torch.full((32 * 64,), 0.4, device="cuda")
    r360.fusion_fuse_static(L, dims, (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0), pose, 64, 32, depth)
    torch.cuda.synchronize()
    assert int((L > 0).sum()) > 100 and int((L < 0).sum()) > 1000
