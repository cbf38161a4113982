"""-m gpu: Algorithm 1 stage II (r360_assign_subfields) against the oracle: labels are integers, the bar is exact."""
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


def _cmp(r360, occ, dims, box_min, box_max, thr, n):
    from oracle.stage2 import assign_subfields
    ref = assign_subfields(occ, dims, box_min, box_max, thr, n)
    got = r360.assign_subfields(occ, dims, box_min, box_max, thr, n)
    assert np.array_equal(got, ref)
    return got


@pytest.mark.parametrize("seed,dims,n", [(0, (6, 5, 4), 7), (1, (8, 8, 2), 5), (2, (4, 4, 4), 1), (3, (9, 3, 3), 11),
                                         (4, (33, 17, 9), 40), (5, (64, 64, 8), 97)])
def test_random_grids(r360, seed, dims, n):
    rng = np.random.default_rng(seed)
    N = dims[0] * dims[1] * dims[2]
    occ = np.where(rng.random(N) < 0.4, 250, 10).astype(np.uint8)
    # a box whose voxel sizes are not powers of two: the binary32 rounding of d2 decides some orders
    _cmp(r360, occ, dims, (-1.3, 0.2, -0.7), (-1.3 + dims[0] * 0.07, 0.2 + dims[1] * 0.11, -0.7 + dims[2] * 0.05), 248, n)


def test_degenerate(r360):
    occ = np.full(5, 255, np.uint8)
    for n in (1, 2, 5):
        _cmp(r360, occ, (5, 1, 1), (0, 0, 0), (5, 1, 1), 128, n)
    with pytest.raises(r360.R360Error):
        r360.assign_subfields(occ, (5, 1, 1), (0, 0, 0), (5, 1, 1), 128, 6)
    with pytest.raises(r360.R360Error):
        r360.assign_subfields(np.zeros(5, np.uint8), (5, 1, 1), (0, 0, 0), (5, 1, 1), 128, 1)   # no occupied voxel


@pytest.mark.parametrize("config,n", [(1, 16), (2, 256)])
def test_baseline_scenes(r360, config, n):
    """The occupancy grids of BASELINE.json's configs 1 and 2 with the paper's assignment instead of the kd-split."""
    sc = get_scene(config, with_weights=False)
    lab = _cmp(r360, sc.occupancy, sc.dims, sc.box_min, sc.box_max, sc.occ_threshold, n)
    counts = np.bincount(lab[lab >= 0], minlength=n)
    assert counts.max() - counts.min() <= 1


def test_assignment_feeds_the_renderer(r360, oracle):
    """End to end: labels from the GPU assignment -> scene -> render, against the oracle with the same labels."""
    from gpu_util import check_image
    sc = get_scene(1)
    lab = r360.assign_subfields(sc.occupancy, sc.dims, sc.box_min, sc.box_max, sc.occ_threshold, sc.n_subfields)
    gpu = r360.scene_from(sc, voxel_subfield=lab)
    okw = dict(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
               hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, pe_pos_levels=sc.pe_pos_levels,
               pe_dir_levels=sc.pe_dir_levels, samples_per_voxel=sc.samples_per_voxel, t_threshold=sc.t_threshold,
               density_activation=sc.density_activation, occ_threshold=sc.occ_threshold, occupancy=sc.occupancy,
               voxel_subfield=lab, weights=sc.weights)
    ora = oracle.scene(**okw)
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ora.render_rows(sc.poses[0], sc.W, sc.H), 1e-4)
    gpu.close()
