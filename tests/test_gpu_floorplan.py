"""-m gpu: r360_floorplan against the oracle (byte image: exact)."""
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


def _free_seed(occ, dims, thr, rng):
    from oracle.floorplan import floorplan
    nx, ny, nz = dims
    for _ in range(200):
        s = (int(rng.integers(0, nx)), int(rng.integers(0, ny)))
        try:
            return s, floorplan(occ, dims, thr, s)
        except ValueError:
            continue
    raise AssertionError("no free seed found")


@pytest.mark.parametrize("seed,dims,p", [(0, (12, 10, 20), 0.02), (1, (70, 45, 24), 0.03), (2, (33, 97, 8), 0.05),
                                         (3, (130, 130, 40), 0.01)])
def test_random_grids(r360, seed, dims, p):
    rng = np.random.default_rng(seed)
    nx, ny, nz = dims
    occ = np.where(rng.random((nz, ny, nx)) < p, 250, 5).astype(np.uint8)
    occ[:, 0, :] = occ[:, -1, :] = 250          # a shell, random pillars and a few wall pieces inside
    occ[:, :, 0] = occ[:, :, -1] = 250
    occ[:, ny // 2, : nx // 2] = 250
    s, ref = _free_seed(occ, dims, 248, rng)
    got = r360.floorplan(occ, dims, 248, s)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("config", [1, 2, 3])
def test_baseline_scenes(r360, config):
    from oracle.floorplan import BOUNDARY, INTERIOR, floorplan
    sc = get_scene(config, with_weights=False)
    nx, ny, nz = sc.dims
    pose = np.asarray(sc.poses[0], np.float64).reshape(3, 4)
    vs = (np.array(sc.box_max) - np.array(sc.box_min)) / np.array(sc.dims)
    cell = np.floor((pose[:, 3] - np.array(sc.box_min)) / vs).astype(int)       # the camera's cell is the seed
    seed = (int(cell[0]), int(cell[1]))
    ref = floorplan(sc.occupancy, sc.dims, sc.occ_threshold, seed)
    got = r360.floorplan(sc.occupancy, sc.dims, sc.occ_threshold, seed)
    assert np.array_equal(got, ref)
    assert (got & INTERIOR).any() and (got & BOUNDARY).any()
    # other slices through the same entry point
    ref2 = floorplan(sc.occupancy, sc.dims, sc.occ_threshold, seed, upper=(0.5, 0.9), lower=(0.0, 0.5))
    got2 = r360.floorplan(sc.occupancy, sc.dims, sc.occ_threshold, seed, upper=(0.5, 0.9), lower=(0.0, 0.5))
    assert np.array_equal(got2, ref2)


def test_winding_region_is_filled_completely(r360):
    """A serpentine of 300 corridors on a 1200 x 1200 grid: the free region crosses 32 x 32 tile borders about
    11 000 times, more than the 4 (nx + ny) + 8 launches the flood fill used to stop after."""
    from oracle.floorplan import INTERIOR, floorplan
    nx = ny = 1200
    nz = 4
    occ = np.full((nz, ny, nx), 5, np.uint8)
    occ[:, 0, :] = occ[:, -1, :] = 250
    occ[:, :, 0] = occ[:, :, -1] = 250
    for k, x in enumerate(range(4, nx - 4, 4)):          # walls one cell thick, corridors three cells wide
        occ[:, :, x] = 250
        if k % 2 == 0:
            occ[:, ny - 4:ny - 1, x] = 5                  # door at the far end ...
        else:
            occ[:, 1:4, x] = 5                            # ... then at the near end
    ref = floorplan(occ, (nx, ny, nz), 248, (2, 2))
    got = r360.floorplan(occ, (nx, ny, nz), 248, (2, 2))
    assert np.array_equal(got, ref)
    assert (ref[:, nx - 3] & INTERIOR).any()              # the fill reached the last corridor


def test_errors(r360):
    occ = np.full((4, 6, 6), 255, np.uint8)
    with pytest.raises(r360.R360Error):
        r360.floorplan(occ, (6, 6, 4), 128, (2, 2))            # seed on a wall
    with pytest.raises(r360.R360Error):
        r360.floorplan(occ, (6, 6, 4), 128, (9, 2))            # seed outside
    with pytest.raises(r360.R360Error):
        r360.floorplan(np.zeros((4, 6, 6), np.uint8), (6, 6, 4), 128, (2, 2), upper=(0.7, 0.6))
