"""scenegen is data only: determinism and the stated structure of the synthetic scenes."""
import numpy as np

from scenegen import CONFIGS, SplitMix64, make_scene, mlp_param_count


def test_splitmix_is_counter_based():
    a = SplitMix64(3, 1).bits(10)
    r = SplitMix64(3, 1)
    b = np.concatenate([r.bits(4), r.bits(6)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, SplitMix64(3, 2).bits(10))
    u = SplitMix64(0).uniform(1000)
    assert u.min() >= 0 and u.max() < 1 and np.all(u * 2 ** 24 == np.floor(u * 2 ** 24))


def test_config1_structure(scene1):
    sc = scene1
    assert (sc.W, sc.H, sc.dims, sc.n_subfields) == (64, 32, (32, 32, 12), 16)
    occ = sc.occupied_mask().reshape(12, 32, 32)
    shell = np.zeros_like(occ)
    shell[[0, -1]] = shell[:, [0, -1]] = True
    shell[:, :, [0, -1]] = True
    assert np.all(occ[shell]) and shell.sum() == 3288 and occ.sum() > 3288
    lab = sc.voxel_subfield
    assert np.all((lab >= 0) == occ.reshape(-1)) and lab.max() == 15
    cnt = np.bincount(lab[lab >= 0])
    assert cnt.max() - cnt.min() <= 1                      # median kd-split
    assert sc.weights.size == 16 * mlp_param_count(32, 2) == 16 * 6212
    assert np.array_equal(sc.poses[0], np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], np.float32))


def test_deterministic_and_xavier_bounds(scene1):
    again = make_scene(1)
    assert np.array_equal(again.occupancy, scene1.occupancy)
    assert np.array_equal(again.voxel_subfield, scene1.voxel_subfield)
    assert np.array_equal(again.weights, scene1.weights)
    w = scene1.weights.reshape(16, -1)
    a1 = np.sqrt(6.0 / (63 + 32))
    assert np.abs(w[:, :63 * 32]).max() <= a1 and np.abs(w[:, :63 * 32]).max() > 0.95 * a1
    assert np.all(w[:, 63 * 32:63 * 32 + 32] == 0)          # biases zero
    dens_bias = 63 * 32 + 32 + 32 * 32 + 32 + 32
    assert np.all(w[:, dens_bias] == 1.0)


def test_config2_pose_is_free_and_gravity_aligned(scene2):
    sc = scene2
    m = sc.poses[0].reshape(3, 4).astype(np.float64)
    r = m[:, :3]
    assert np.allclose(r @ r.T, np.eye(3), atol=1e-6) and abs(np.linalg.det(r) - 1) < 1e-6
    assert np.allclose(r[:, 1], [0, 0, -1], atol=1e-7)       # camera y (down) = world -z
    assert -0.5 <= m[2, 3] <= 0.0
    frac = sc.occupied_mask().mean()
    assert 0.05 < frac < 0.12
    assert len(CONFIGS) == 5
