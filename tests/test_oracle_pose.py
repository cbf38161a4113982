"""-m "not gpu": reading B5 -- which poses the render calls accept.  The oracle's r360o_pose_ok is pinned
to the linear algebra it stands for (numpy's SVD and determinant, rotations built from axis-angle), the oracle's walk
is checked to survive a zero direction, and the library's own check (capi.cu, reached through an entry point that
validates its pose before it touches CUDA) must take the same decision on every probe."""
import ctypes as C

import numpy as np
import pytest

F = np.float32


def _rot(rng):
    """A rotation from a random unit axis and angle (Rodrigues), binary64."""
    k = rng.normal(size=3)
    k /= np.linalg.norm(k)
    a = rng.uniform(-np.pi, np.pi)
    K = np.array([[0, -k[2], k[1]], [k[2], 0, -k[0]], [-k[1], k[0], 0]])
    return np.eye(3) + np.sin(a) * K + (1 - np.cos(a)) * (K @ K)


def _pose(M, o=(0.1, -0.2, 0.3)):
    return np.concatenate([np.asarray(M, np.float64), np.asarray(o, np.float64)[:, None]], 1).astype(F).reshape(12)


def _probes():
    rng = np.random.default_rng(5)
    out = []
    for _ in range(40):
        R = _rot(rng)
        out.append((_pose(R), True))                                            # rotations
        out.append((_pose(R * rng.uniform(0.01, 100.0)), True))                 # uniformly scaled
        out.append((_pose(R @ np.diag([1.0, 1.0, rng.uniform(0.05, 20.0)])), True))   # moderate anisotropy
        S = R @ np.diag([1.0, 1.0, 0.0])
        out.append((_pose(S), False))                                           # rank 2: the camera z axis is lost
        out.append((_pose(R @ np.diag([1.0, 1.0, 1e-7])), False))               # nearly singular
        out.append((_pose(np.outer(R[:, 0], R[0])), False))                     # rank 1
    out.append((_pose(np.zeros((3, 3))), False))
    out.append((_pose(np.eye(3) * 1e-6), False))                                # norm below 2^-16
    out.append((_pose(np.eye(3) * 1e6), False))                                 # norm above 2^16
    for bad in (np.nan, np.inf, -np.inf):
        p = _pose(np.eye(3))
        p[6] = bad
        out.append((p, False))
        p = _pose(np.eye(3))
        p[3] = bad                                                              # the centre must be finite too
        out.append((p, False))
    return out


def test_pose_ok_is_the_stated_rule(oracle):
    """|det M| >= 2^-16 |M|_F^3 and 2^-16 <= |M|_F <= 2^16, evaluated independently with numpy, and what the rule is
    for: the smallest singular value of an accepted matrix is at least 2^-16 |M|_F."""
    ok = oracle.lib.r360o_pose_ok
    ok.restype = C.c_int
    ok.argtypes = [C.POINTER(C.c_float)]
    rng = np.random.default_rng(6)
    n_acc = n_rej = 0
    probes = [p for p, _ in _probes()]
    for _ in range(300):                                                        # random matrices across the threshold
        U, V = _rot(rng), _rot(rng)
        sv = np.array([1.0, 10.0 ** rng.uniform(-3, 0), 10.0 ** rng.uniform(-7, 0)])
        probes.append(_pose(U @ np.diag(sv) @ V.T * 10.0 ** rng.uniform(-1, 1)))
    for p in probes:
        got = bool(ok(p.ctypes.data_as(C.POINTER(C.c_float))))
        if not np.isfinite(p).all():
            assert not got
            continue
        M = p.reshape(3, 4)[:, :3].astype(np.float64)
        f = np.linalg.norm(M)
        ratio = abs(np.linalg.det(M)) / f ** 3 if f > 0 else 0.0
        in_range = 2.0 ** -16 <= f <= 2.0 ** 16
        if in_range and abs(ratio / 2.0 ** -16 - 1) < 1e-9:
            continue                                                            # on the boundary: either answer
        want = in_range and ratio >= 2.0 ** -16
        assert got == want, (p, ratio, f)
        if got:
            assert np.linalg.svd(M, compute_uv=False).min() >= 2.0 ** -16 * f * (1 - 1e-12)
            n_acc += 1
        else:
            n_rej += 1
    assert n_acc > 100 and n_rej > 100


def test_probe_classes(oracle):
    ok = oracle.lib.r360o_pose_ok
    ok.restype = C.c_int
    ok.argtypes = [C.POINTER(C.c_float)]
    for p, want in _probes():
        assert bool(ok(p.ctypes.data_as(C.POINTER(C.c_float)))) == want, p


def test_accepted_poses_never_give_an_all_parallel_ray(oracle):
    """The point of the rule: for an accepted pose every generated direction keeps a component far above reading
    C1's 2^-100, on the whole pixel grid of a small panorama."""
    rng = np.random.default_rng(8)
    for _ in range(6):
        M = _rot(rng) @ np.diag([1.0, 1.0, 2.0 ** -14.0]) * 2.0 ** -15          # close to both limits
        p = _pose(M)
        assert oracle.lib.r360o_pose_ok(p.ctypes.data_as(C.POINTER(C.c_float)))
        f = np.linalg.norm(M)
        for j in range(0, 16):
            for i in range(0, 32):
                _, d = oracle.ray(p, 32, 16, i, j)
                assert np.abs(d).max() >= 2.0 ** -16 * f / np.sqrt(3) * 0.9


def test_oracle_refuses_and_survives(oracle, scene1):
    ora = oracle.scene_from(scene1)
    bad = _pose(np.diag([1.0, 1.0, 0.0]), scene1.poses[0].reshape(3, 4)[:, 3])
    with pytest.raises(ValueError):
        ora.render_rows(bad, 16, 8)
    with pytest.raises(ValueError):
        ora.render_pixels(bad, 16, 8, np.zeros(1, np.int32), np.zeros(1, np.int32))
    with pytest.raises(ValueError):
        ora.samples_rows(bad, 16, 8)
    with pytest.raises(ValueError):
        ora.ray_samples(bad, 16, 8, 0, 0)
    # a zero direction from inside the box: no voxel is crossed, nothing is indexed out of range
    o = scene1.poses[0].reshape(3, 4)[:, 3]
    for d in ((0, 0, 0), (1e-35, -1e-36, 0)):
        v, ti, to = ora.walk(o, np.array(d, F))
        assert len(v) == 0
    ora.close()


def test_library_takes_the_same_decision_before_touching_cuda():
    """r360_fusion_fuse_static checks its pose (capi.cu: r360_poses_ok, the check behind every pose argument of
    include/r360.h) before its size limit and before any CUDA call: with a grid over the limit a bad pose is
    R360_ERR_INVALID_ARG (1) and a good one R360_ERR_CAPACITY (6).  No device is needed or used."""
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as r360
    L = r360.lib()
    f32p = C.POINTER(C.c_float)
    fn = L.r360_fusion_fuse_static
    fn.restype = C.c_int
    fn.argtypes = [C.POINTER(C.c_int32), f32p, f32p, C.c_void_p, f32p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                   C.c_void_p]
    dims = (C.c_int32 * 3)(4096, 4096, 4)
    lo, hi = (C.c_float * 3)(0, 0, 0), (C.c_float * 3)(1, 1, 1)
    for p, want in _probes():
        st = fn(dims, lo, hi, 256, p.ctypes.data_as(f32p), 8, 8, 256, None, None)   # (the pointers are never touched)
        assert st == (6 if want else 1), (p, st)
