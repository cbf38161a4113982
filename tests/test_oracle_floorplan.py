"""Pins for the floorplan oracle: hand-built rooms whose plan can be written down by eye."""
import numpy as np
import pytest

from oracle.floorplan import BOUNDARY, INTERIOR, OBSTACLE, floorplan, slice_layers


def _room(nx=12, ny=10, nz=20):
    """A closed room: walls on the image border over the full height, one box on the floor (layers 0..7)."""
    occ = np.zeros((nz, ny, nx), np.uint8)
    occ[:, 0, :] = occ[:, -1, :] = 255
    occ[:, :, 0] = occ[:, :, -1] = 255
    occ[0:8, 4:6, 5:8] = 255                 # obstacle: y 4..5, x 5..7, below 40 % of the height
    return occ


def test_slice_layers():
    assert slice_layers(96, 0.60, 0.65) == [58, 59, 60, 61]          # centres 0.609 .. 0.641
    assert slice_layers(96, 0.20, 0.30) == list(range(19, 29))        # 0.203 .. 0.297
    assert slice_layers(20, 0.60, 0.65) == [12]                       # centre 0.625
    assert slice_layers(4, 0.60, 0.65) == [2]                         # centre 0.625
    assert slice_layers(3, 0.60, 0.65) == []                          # centres 0.167 0.5 0.833


def test_closed_room_by_hand():
    occ = _room()
    plan = floorplan(occ, (12, 10, 20), 128, (2, 2))
    interior = (plan & INTERIOR) > 0
    exp_int = np.zeros((10, 12), bool)
    exp_int[1:-1, 1:-1] = True                                        # everything inside the walls
    assert np.array_equal(interior, exp_int)
    exp_b = np.zeros((10, 12), bool)                                  # the ring of interior cells along the walls
    exp_b[1, 1:-1] = exp_b[-2, 1:-1] = True
    exp_b[1:-1, 1] = exp_b[1:-1, -2] = True
    assert np.array_equal((plan & BOUNDARY) > 0, exp_b)
    exp_o = np.zeros((10, 12), bool)
    exp_o[4:6, 5:8] = True                                            # the box shows up as an obstacle, not as wall
    assert np.array_equal((plan & OBSTACLE) > 0, exp_o)


def test_one_cell_gap_is_closed_two_rooms_are_separated():
    # an interior wall with a ONE-cell gap at the upper slice: the closing seals it, the seed's room is the interior
    occ = _room(16, 10, 20)
    occ[:, :, 8] = 255
    occ[:, 5, 8] = 0                                                  # the gap
    plan = floorplan(occ, (16, 10, 20), 128, (3, 3))
    interior = (plan & INTERIOR) > 0
    assert interior[1:-1, 1:8].all() and not interior[:, 8:].any()
    # a door three cells wide stays open (the closing only fills what a 3x3 square cannot enter)
    occ[:, 4:7, 8] = 0
    plan = floorplan(occ, (16, 10, 20), 128, (3, 3))
    interior = (plan & INTERIOR) > 0
    assert interior[5, 8] and interior[1:-1, 9:-1].all()


def test_head_jamb_above_the_slice_is_ignored_and_seed_checks():
    # a lintel above a door (layers 14..19 = above 70 %) does not close the door: the slice is 60-65 %
    occ = _room(16, 10, 20)
    occ[:, :, 8] = 255
    occ[0:14, 3:7, 8] = 0                                             # door up to 70 % of the height
    plan = floorplan(occ, (16, 10, 20), 128, (3, 3))
    assert ((plan & INTERIOR) > 0)[1:-1, 9:-1].all()
    with pytest.raises(ValueError):
        floorplan(occ, (16, 10, 20), 128, (0, 0))                     # seed on a wall
    with pytest.raises(ValueError):
        floorplan(occ, (16, 10, 20), 128, (40, 3))                    # seed outside


def test_baseline_scene_plan_is_consistent(scene1):
    sc = scene1
    nx, ny, nz = sc.dims
    plan = floorplan(sc.occupancy, sc.dims, sc.occ_threshold, (nx // 2, ny // 2))
    interior, boundary, obstacle = (plan & INTERIOR) > 0, (plan & BOUNDARY) > 0, (plan & OBSTACLE) > 0
    assert interior[ny // 2, nx // 2] and not interior[0].any() and not interior[:, 0].any()
    assert not (boundary & ~interior).any() and not (obstacle & ~interior).any()
    assert boundary.sum() >= 2 * (nx + ny) - 16                       # at least the ring along the shell
