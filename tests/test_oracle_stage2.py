"""Pins for the oracle of Algorithm 1, stage II: partition properties, degenerate cases,
a hand-checkable line of voxels, and a literal pure-Python transcription of the algorithm on tiny grids."""
import math

import numpy as np
import pytest

from oracle.stage2 import assign_subfields


def _literal(occ, dims, box_min, box_max, thr, n):
    """The algorithm word by word with Python lists and exact rational distances (no numpy, no float32)."""
    from fractions import Fraction
    nx, ny, nz = dims
    vs = [Fraction(float(np.float32(np.float32(box_max[a]) - np.float32(box_min[a])) / np.float32(dims[a]))) for a in range(3)]
    un = [v for v in range(nx * ny * nz) if occ[v] >= thr]          # unassigned, ascending "coordinate"
    S = len(un)
    labels = [-1] * (nx * ny * nz)
    q, r = divmod(S, n)
    for k in range(n):
        size = q + (1 if k < r else 0)
        a = un.pop(0)                                              # pop the minimum coordinate
        labels[a] = k
        ac = (a % nx, (a // nx) % ny, a // (nx * ny))

        def d2(v):
            c = (v % nx, (v // nx) % ny, v // (nx * ny))
            return sum(((c[i] - ac[i]) * vs[i]) ** 2 for i in range(3))
        near = sorted(un, key=lambda v: (d2(v), v))[:size - 1]     # s-1 nearest, ties to the smaller index
        for v in near:
            un.remove(v)
            labels[v] = k
    return np.array(labels, np.int32)


@pytest.mark.parametrize("seed,dims,n", [(0, (6, 5, 4), 7), (1, (8, 8, 2), 5), (2, (4, 4, 4), 1), (3, (9, 3, 3), 11)])
def test_matches_literal_transcription(seed, dims, n):
    rng = np.random.default_rng(seed)
    N = dims[0] * dims[1] * dims[2]
    occ = np.where(rng.random(N) < 0.45, 250, 10).astype(np.uint8)
    # power-of-two voxel sizes: binary32 distances are exact, so the float32 oracle must equal exact arithmetic
    box_min, box_max = (0.0, 0.0, 0.0), (dims[0] * 0.25, dims[1] * 0.25, dims[2] * 0.125)
    got = assign_subfields(occ, dims, box_min, box_max, 248, n)
    assert np.array_equal(got, _literal(occ, dims, box_min, box_max, 248, n))


def test_partition_properties(scene1):
    sc = scene1
    n = 16
    lab = assign_subfields(sc.occupancy, sc.dims, sc.box_min, sc.box_max, sc.occ_threshold, n)
    occ = np.asarray(sc.occupancy).reshape(-1) >= sc.occ_threshold
    assert np.all(lab[~occ] == -1) and np.all(lab[occ] >= 0)
    S = int(occ.sum())
    counts = np.bincount(lab[occ], minlength=n)
    assert counts.sum() == S and counts.max() - counts.min() <= 1           # "similar amount" (:157), reading S1
    assert np.array_equal(counts, [S // n + (1 if k < S % n else 0) for k in range(n)])
    # anchors: network k's smallest voxel index increases with k (each anchor is the minimum unassigned coordinate)
    firsts = [int(np.flatnonzero(lab == k)[0]) for k in range(n)]
    assert firsts == sorted(firsts)
    # locality: every network's voxels lie within the distance of its farthest member from the anchor, and no
    # voxel assigned LATER is strictly closer to the anchor than that farthest member (greedy nearest rule)
    nx, ny, nz = sc.dims
    vs = (np.array(sc.box_max) - np.array(sc.box_min)) / np.array(sc.dims)
    lin = np.flatnonzero(occ)
    c = np.stack([lin % nx, (lin // nx) % ny, lin // (nx * ny)], 1) * vs
    for k in range(n):
        mine = lab[lin] == k
        a = c[np.flatnonzero(mine)[0]]
        far = np.sqrt(((c[mine] - a) ** 2).sum(1)).max()
        later = lab[lin] > k
        assert np.sqrt(((c[later] - a) ** 2).sum(1)).min(initial=np.inf) >= far - 1e-6


def test_degenerate_cases():
    dims = (5, 1, 1)
    occ = np.full(5, 255, np.uint8)
    box = ((0, 0, 0), (5, 1, 1))
    assert np.array_equal(assign_subfields(occ, dims, *box, 128, 1), [0, 0, 0, 0, 0])
    assert np.array_equal(assign_subfields(occ, dims, *box, 128, 5), [0, 1, 2, 3, 4])
    # a line: anchors sweep from the low end, each network a contiguous run; 5 = 2*2 + 1 -> sizes 3, 2 (S1)
    assert np.array_equal(assign_subfields(occ, dims, *box, 128, 2), [0, 0, 0, 1, 1])
    with pytest.raises(ValueError):
        assign_subfields(occ, dims, *box, 128, 6)
    # an empty voxel in the line and a tie: anchor 0 has voxels 1 (d=1); then anchor 3: neighbours 4 (d=1)
    occ2 = np.array([255, 255, 0, 255, 255, 255], np.uint8)
    assert np.array_equal(assign_subfields(occ2, (6, 1, 1), (0, 0, 0), (6, 1, 1), 128, 2), [0, 0, -1, 0, 1, 1])


def test_tie_goes_to_smaller_index():
    # 3x3 plane, anchor = voxel 0; the two voxels at distance 1 are index 1 (x+1) and index 3 (y+1): with s = 2
    # the tie goes to index 1 (reading S4)
    occ = np.full(9, 255, np.uint8)
    lab = assign_subfields(occ, (3, 3, 1), (0, 0, 0), (3, 3, 1), 128, 4)   # sizes 3,2,2,2
    assert lab[0] == 0 and lab[1] == 0 and lab[3] == 0
    lab = assign_subfields(occ, (3, 3, 1), (0, 0, 0), (3, 3, 1), 128, 5)   # sizes 2,2,2,2,1
    assert lab[0] == 0 and lab[1] == 0 and lab[3] != 0
    # anisotropic voxels (y half as long as x): the y neighbour is nearer and wins without a tie
    lab = assign_subfields(occ, (3, 3, 1), (0, 0, 0), (3, 1.5, 1), 128, 5)
    assert lab[0] == 0 and lab[3] == 0 and lab[1] != 0
