"""Pins for the oracle's compositing (Eq. 4-5; readings E, G) and the end-to-end render."""
import math

import numpy as np
import pytest

from scenegen import mlp_param_count, weight_layout

F = np.float32
TAU = float(F(1e-3))


def _segments(rng, n_seg, K):
    """n_seg disjoint segments with gaps; K midpoints each (reading D)."""
    edges = np.sort(rng.uniform(0.5, 6.0, 2 * n_seg))
    t, dl = [], []
    for a, b in zip(edges[0::2], edges[1::2]):
        d = (b - a) / K
        t += [a + (j + 0.5) * d for j in range(K)]
        dl += [d] * K
    return np.array(t, F), np.array(dl, F), float((edges[1::2] - edges[0::2]).sum())


@pytest.mark.parametrize("K", [1, 3, 8, 12])
def test_constant_density_slab_closed_form(oracle, K):
    # constant sigma over occupied length d: T_end = exp(-sigma d) for any K, any gaps (reading E)
    rng = np.random.default_rng(K)
    t, dl, length = _segments(rng, 5, K)
    sigma = 0.7
    length = float(dl.astype(np.float64).sum())            # binary32 strata as given
    out, full, amb = oracle.composite(np.full(t.size, sigma), np.tile([0.2, 0.5, 0.9], (t.size, 1)), t, dl, 0.0)
    T_end = math.exp(-sigma * length)
    assert abs(out[4] - T_end) < 1e-13
    assert np.allclose(out[:3], np.array([0.2, 0.5, 0.9]) * (1 - T_end), atol=1e-13)   # constant colour x opacity
    assert out[5] == t.size


def test_telescoping_weights_and_depth(oracle):
    rng = np.random.default_rng(5)
    t, dl, _ = _segments(rng, 6, 8)
    sigma = rng.uniform(0, 3, t.size)
    rgb = rng.uniform(0, 1, (t.size, 3))
    out, full, amb = oracle.composite(sigma, rgb, t, dl, 0.0)
    # sum_i w_i = 1 - T_end with white colour
    out1, _, _ = oracle.composite(sigma, np.ones((t.size, 3)), t, dl, 0.0)
    assert abs(out1[0] - (1 - out1[4])) < 1e-13
    # Eq.5 written literally: w_i = exp(-sum_{k<i} sigma_k delta_k) (1 - exp(-sigma_i delta_i))
    sd = sigma * dl.astype(np.float64)
    w = np.exp(-np.concatenate([[0], np.cumsum(sd)[:-1]])) * (1 - np.exp(-sd))
    assert np.allclose(out[:3], (w[:, None] * rgb).sum(0), atol=1e-13)
    assert abs(out[3] - (w * t.astype(np.float64)).sum()) < 1e-12                      # Eq.4 depth
    assert abs(out[4] - math.exp(-sd.sum())) < 1e-13


def test_constant_sigma_depth_geometric_sum(oracle):
    # one slab [a, a+K*d], constant sigma: D = sum_j e^{-sigma j d}(1-e^{-sigma d}) (a+(j+1/2)d)
    a, d, K, sigma = 1.25, 0.03125, 16, 2.0
    t = np.array([a + (j + 0.5) * d for j in range(K)], F)
    out, _, _ = oracle.composite(np.full(K, sigma), np.ones((K, 3)), t, np.full(K, d, F), 0.0)
    q = math.exp(-sigma * d)
    expect = sum(q ** j * (1 - q) * (a + (j + 0.5) * d) for j in range(K))
    assert abs(out[3] - expect) < 1e-13


def test_early_out_semantics(oracle):
    # sigma*delta = ln 2 per sample: T halves each sample; T < 1e-3 first after sample 10 (2^-10 = 9.77e-4)
    n = 30
    dl = np.full(n, 0.125, F)
    sigma = np.full(n, math.log(2) / 0.125)
    t = (np.arange(n) + 0.5).astype(F) * F(0.125)
    rgb = np.ones((n, 3))
    out, full, amb = oracle.composite(sigma, rgb, t, dl, TAU)
    assert out[5] == 10 and abs(out[4] - 2.0 ** -10) < 1e-15    # the crossing sample is included
    assert abs(out[0] - (1 - 2.0 ** -10)) < 1e-13
    assert full[5] == n and abs(full[0] - (1 - 2.0 ** -n)) < 1e-13
    assert np.all(full[:4] >= out[:4]) and np.all(full[:3] - out[:3] <= TAU)   # early-out costs at most tau
    assert abs(amb - abs(2.0 ** -10 - TAU) / TAU) < 1e-12
    # no samples: black, zero depth, T = 1
    out, full, amb = oracle.composite(np.zeros(0), np.zeros((0, 3)), np.zeros(0, F), np.zeros(0, F), TAU)
    assert np.all(out[:4] == 0) and out[4] == 1.0 and out[5] == 0


def _zero_net(width, n_hidden, sigma_bias):
    w, o = np.zeros(mlp_param_count(width, n_hidden), F), 0
    for name, fo, fi in weight_layout(width, n_hidden):
        if name == "density":
            w[o + fo * fi] = sigma_bias
        o += fo * fi + fo
    return w


@pytest.mark.parametrize("sigma_bias", [1.0, 6.0])
def test_end_to_end_zero_weight_closed_form(oracle, scene1, sigma_bias):
    # zero weights: sigma = softplus(bias), rgb = 0.5 inside occupied voxels, so
    # C = 0.5 (1 - exp(-sigma L_occ)) with L_occ from an independent binary64 slab computation
    sc = scene1
    w = np.tile(_zero_net(sc.hidden_width, sc.n_hidden, sigma_bias), sc.n_subfields)
    s = oracle.scene(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
                     hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, samples_per_voxel=sc.samples_per_voxel,
                     t_threshold=0.0, density_activation=1, occ_threshold=sc.occ_threshold,
                     occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield, weights=w)
    r = s.render_rows(sc.poses[0], sc.W, sc.H)
    sigma = math.log1p(math.exp(sigma_bias))
    occ = sc.occupied_mask()
    nx, ny, nz = sc.dims
    bmin = np.array(sc.box_min)
    vs = (np.array(sc.box_max) - bmin) / np.array(sc.dims)
    lin = np.flatnonzero(occ)
    lo = bmin + np.stack([lin % nx, (lin // nx) % ny, lin // (nx * ny)], 1) * vs
    hi = lo + vs
    worst = 0.0
    for j in range(0, sc.H, 3):
        for i in range(0, sc.W, 5):
            o, d = oracle.ray(sc.poses[0], sc.W, sc.H, i, j)
            o64, d64 = o.astype(np.float64), d.astype(np.float64)
            ta, tb = (lo - o64) / d64, (hi - o64) / d64
            L = np.clip(np.maximum(ta, tb).min(1) - np.maximum(np.minimum(ta, tb).max(1), 0.0), 0, None).sum()
            expect = 0.5 * (1 - math.exp(-sigma * L))
            worst = max(worst, float(np.abs(r["rgb"][j * sc.W + i] - expect).max()))
    assert worst < 2e-5
    assert np.array_equal(r["n_emitted"], r["n_used"])


def test_render_early_out_bounds(oracle, scene1):
    # dense medium (density bias 40): rays stop early; stopped result within tau of the continued one
    sc = scene1
    w = sc.weights.copy().reshape(sc.n_subfields, -1)
    o = 0
    for name, fo, fi in weight_layout(sc.hidden_width, sc.n_hidden):
        if name == "density":
            w[:, o + fo * fi] = 40.0
        o += fo * fi + fo
    s = oracle.scene(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
                     hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, samples_per_voxel=sc.samples_per_voxel,
                     t_threshold=1e-3, density_activation=1, occ_threshold=sc.occ_threshold,
                     occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield, weights=w.reshape(-1))
    r = s.render_rows(sc.poses[0], sc.W, sc.H)
    assert (r["n_used"] < r["n_emitted"]).mean() > 0.5
    assert np.all(r["rgb_full"] >= r["rgb"]) and np.all(r["rgb_full"] - r["rgb"] <= 1e-3 + 1e-7)
    assert np.all(r["depth_full"] >= r["depth"])
    # pixel-list entry point agrees with the row entry point
    px = np.array([3, 17, 60], np.int32)
    py = np.array([2, 9, 30], np.int32)
    rp = s.render_pixels(sc.poses[0], sc.W, sc.H, px, py)
    assert np.array_equal(rp["rgb"], r["rgb"][py * sc.W + px])
    assert np.array_equal(rp["n_used"], r["n_used"][py * sc.W + px])
