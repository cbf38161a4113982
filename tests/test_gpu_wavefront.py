"""-m gpu: wavefronted early termination (r360_set_wavefront).  Every ray sees the same sequence of operations as in
the single-pass path, so the images must be IDENTICAL bit for bit in both precisions; what changes is how many
samples reach the MLP."""
import numpy as np
import pytest

from conftest import get_scene
from gpu_util import check_image, with_density_bias

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def r360():
    import torch
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def _both(gpu, pose, W, H):
    gpu.set_wavefront(False)
    rgb0, d0 = gpu.render(pose, W, H)
    rgb0, d0 = rgb0.clone(), d0.clone()
    st0 = gpu.stats()
    gpu.set_wavefront(True)
    rgb1, d1 = gpu.render(pose, W, H)
    st1 = gpu.stats()
    assert np.array_equal(rgb0.cpu().numpy().view(np.uint32), rgb1.cpu().numpy().view(np.uint32))
    assert np.array_equal(d0.cpu().numpy().view(np.uint32), d1.cpu().numpy().view(np.uint32))
    assert st1.samples_emitted == st0.samples_emitted          # geometric count: unchanged
    assert st1.samples_used == st0.samples_used
    return st0, st1


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
@pytest.mark.parametrize("config", [1, 2])
def test_same_image_translucent(r360, config, precision):
    # BASELINE scenes: sigma ~ 1.3 behind thin walls, no ray terminates: every sample still reaches the MLP
    sc = get_scene(config)
    gpu = r360.scene_from(sc)
    gpu.set_precision(precision)
    st0, st1 = _both(gpu, sc.poses[0], sc.W, sc.H)
    assert st1.segments == st0.segments
    gpu.close()


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_opaque_scene_skips_mlp_work(r360, precision):
    # config 5's clutter (about 20 occupied voxels per ray, some rays beyond the hit buffer) made opaque (density
    # bias 40: T < tau after about three voxels): the passes retire the rays before the MLP sees the rest
    sc = get_scene(5)
    gpu = r360.scene_from(sc, weights=with_density_bias(sc, 40.0))
    gpu.set_precision(precision)
    st0, st1 = _both(gpu, sc.poses[0], 512, 256)
    print("opaque config 5 at 512x256:", precision, "segments to the MLP", st0.segments, "->", st1.segments)
    assert st1.segments < 0.4 * st0.segments
    assert st1.mlp_tiles < 0.5 * st0.mlp_tiles
    gpu.close()


def test_ragged_chunks_batch_and_long_rays(r360):
    sc = get_scene(1)
    gpu = r360.scene_from(sc, samples_per_voxel=5)
    for (W, H) in ((37, 19), (1, 1), (257, 3)):
        _both(gpu, sc.poses[0], W, H)
    gpu.set_chunk_rays(300)
    _both(gpu, sc.poses[0], 64, 32)
    gpu.close()
    # config 5 has rays with more crossings than the hit buffer holds (processed whole in the first pass)
    sc5 = get_scene(5)
    gpu = r360.scene_from(sc5)
    gpu.set_precision("bf16")
    st0, st1 = _both(gpu, sc5.poses[0], 512, 256)
    gpu.close()


def test_wavefront_against_oracle(r360, oracle):
    sc = get_scene(1)
    w = with_density_bias(sc, 40.0)
    gpu = r360.scene_from(sc, weights=w)
    gpu.set_wavefront(True)
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    okw = dict(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
               hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, pe_pos_levels=sc.pe_pos_levels,
               pe_dir_levels=sc.pe_dir_levels, samples_per_voxel=sc.samples_per_voxel, t_threshold=sc.t_threshold,
               density_activation=sc.density_activation, occ_threshold=sc.occ_threshold, occupancy=sc.occupancy,
               voxel_subfield=sc.voxel_subfield, weights=w)
    ref = oracle.scene(**okw).render_rows(sc.poses[0], sc.W, sc.H)
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 1e-4)
    assert gpu.stats().samples_emitted == int(ref["n_emitted"].sum())
    gpu.close()


def test_automatic_mode_follows_the_scene(r360):
    """r360_set_wavefront(2): passes only once a finished frame has shown that most samples go unused."""
    import torch
    sc = get_scene(5)
    W, H = 512, 256
    for bias, expect_passes in ((None, False), (40.0, True)):
        gpu = r360.scene_from(sc) if bias is None else r360.scene_from(sc, weights=with_density_bias(sc, bias))
        gpu.set_precision("bf16")
        rgb0, d0 = gpu.render(sc.poses[0], W, H)
        rgb0, d0 = rgb0.clone(), d0.clone()
        gpu.set_wavefront("auto")
        launches = []
        for _ in range(3):
            rgb, depth = gpu.render(sc.poses[0], W, H)
            launches.append(gpu.stats().kernel_launches)            # synchronises: the next call sees this frame's ratio
            assert torch.equal(rgb, rgb0) and torch.equal(depth, d0)
        assert launches[0] == 5                                     # nothing known yet: single pass
        assert (launches[-1] > 5) == expect_passes
        gpu.close()
