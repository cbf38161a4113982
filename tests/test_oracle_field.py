"""Pins for the oracle's tiny-MLP field (Eq. 1; Table 4 :434-444; :413; readings A1-A5)."""
import math
import os

import numpy as np
import pytest
import torch

from scenegen import mlp_param_count, weight_layout

F = np.float32
GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_parameter_counts_match_paper(oracle):
    g = _gold()
    # 6212 parameters <=> 63->32, 32->32, 32->(1+32), (32+27)->32, 32->3 (reading A1)
    assert oracle.params_per_subfield(hidden_width=32, n_hidden=2) == int(g["tiny_mlp_params"]) == 6212
    assert mlp_param_count(32, 2) == 6212
    # Table 4 as printed (60->32, 32->1, 32->32, (32+24)->32, 32->3) does NOT give 6212:
    assert (60 * 32 + 32) + 33 + (32 * 32 + 32) + (56 * 32 + 32) + (32 * 3 + 3) == 4964
    # 360Roam-200 has "about 1.2M parameters"
    assert abs(200 * 6212 - g["roam200_params_approx"]) / g["roam200_params_approx"] < 0.05
    # Table 3 / :413: 360NeRF has 0.596M parameters only if the PE includes the raw input (63 / 27)
    def nerf360(pp, pd):
        n = pp * 256 + 256 + 3 * (256 * 256 + 256) + (256 + pp) * 256 + 256 + 3 * (256 * 256 + 256)
        return n + (256 + 1) + (256 * 256 + 256) + (256 + pd) * 128 + 128 + 128 * 3 + 3
    assert nerf360(63, 27) == 595844 and round(nerf360(63, 27) / 1e3) == round(g["nerf360_params_approx"] / 1e3)
    assert nerf360(60, 24) == 593924
    assert oracle.params_per_subfield(hidden_width=32, n_hidden=3) == 7268
    assert oracle.params_per_subfield(hidden_width=64, n_hidden=3) == 22724


def _tiny_scene(oracle, weights, n_hidden=2, width=32, act=1, dims=(4, 4, 4)):
    """One subfield owning voxels (1..2, 1..3, 2..2): AABB [0.25,0.75]x[0.25,1.0]x[0.5,0.75] in a unit box."""
    nx, ny, nz = dims
    occ = np.zeros((nz, ny, nx), np.uint8)
    occ[2, 1:4, 1:3] = 255
    lab = np.where(occ > 0, 0, -1).astype(np.int32)
    return oracle.scene(dims=dims, box_min=(0, 0, 0), box_max=(1, 1, 1), n_subfields=1, hidden_width=width,
                        n_hidden=n_hidden, samples_per_voxel=4, density_activation=act, occ_threshold=128,
                        occupancy=occ, voxel_subfield=lab, weights=weights)


def _offsets(width, n_hidden):
    off, o = {}, 0
    for name, fo, fi in weight_layout(width, n_hidden):
        off[name] = (o, fo, fi)
        o += fo * fi + fo
    return off, o


def test_subfield_frame_is_voxel_face_aabb(oracle):
    off, P = _offsets(32, 2)
    s = _tiny_scene(oracle, np.zeros(P, F))
    c, ih = s.subfield_frame(0)
    assert np.allclose(c, [0.5, 0.625, 0.625]) and np.allclose(ih, [4.0, 1 / 0.375, 8.0])


def test_zero_weight_network_constants(oracle):
    off, P = _offsets(32, 2)
    w = np.zeros(P, F)
    o, fo, fi = off["density"]
    w[o + fo * fi] = 1.0                                   # density bias +1
    s = _tiny_scene(oracle, w)
    f = s.field(0, np.array([0.4, 0.5, 0.6], F), np.array([0, 0, 1], F))
    assert abs(f[0] - 1.3132616875182228) < 1e-12          # softplus(1) = ln(1+e)
    assert np.allclose(f[1:], 0.5, atol=1e-15)             # sigmoid(0)
    s = _tiny_scene(oracle, w, act=0)
    assert s.field(0, np.array([0.4, 0.5, 0.6], F), np.array([0, 0, 1], F))[0] == 1.0   # ReLU(1)
    w[o + fo * fi] = -3.0
    s = _tiny_scene(oracle, w, act=0)
    assert s.field(0, np.array([0.4, 0.5, 0.6], F), np.array([0, 0, 1], F))[0] == 0.0   # ReLU(-3)


def _pe_hand(x, f):
    """Feature f of F(x) under reading A2, written from the definition: index -> (level, sin/cos, axis)."""
    if f < 3:
        return x[f]
    l, r = divmod(f - 3, 6)
    fn = math.sin if r < 3 else math.cos
    return fn((2.0 ** l) * x[r % 3])


def test_position_pe_one_hot_probes(oracle):
    # trunk-1 row 0 selects +/- one PE feature; trunk-2 passes channel 0; density head reads channel 0
    off, P = _offsets(32, 2)
    p = np.array([0.31, 0.77, 0.58], F)
    c, h = np.array([0.5, 0.625, 0.625]), np.array([0.25, 0.375, 0.125])
    q = ((p - c.astype(F)) * (F(1) / h.astype(F))).astype(np.float64)
    for f in range(63):
        vals = {}
        for sign in (+1.0, -1.0):
            w = np.zeros(P, F)
            w[off["trunk1"][0] + f] = sign
            w[off["trunk2"][0]] = 1.0
            w[off["density"][0]] = 1.0
            s = _tiny_scene(oracle, w, act=0)
            vals[sign] = s.field(0, p, np.array([0, 0, 1], F), raw=True)[0]
        got = vals[+1.0] - vals[-1.0]                      # relu(x) - relu(-x) = x
        assert abs(got - _pe_hand(q, f)) < 1e-12, f


def test_direction_pe_one_hot_probes(oracle):
    off, P = _offsets(32, 2)
    d = np.array([0.36, -0.48, 0.8], F)
    for f in range(27):
        vals = {}
        for sign in (+1.0, -1.0):
            w = np.zeros(P, F)
            w[off["colour"][0] + 32 + f] = sign           # colour row 0, input [feature(32), F(d)]
            w[off["rgb"][0] + 32] = 1.0                    # green reads colour channel 0
            s = _tiny_scene(oracle, w)
            vals[sign] = s.field(0, np.array([0.4, 0.5, 0.6], F), d, raw=True)[2]
        assert abs(vals[+1.0] - vals[-1.0] - _pe_hand(d.astype(np.float64), f)) < 1e-12, f


def test_feature_layer_has_no_activation_and_feeds_colour(oracle):
    # feature = -2 (bias) must reach the colour layer unclipped: colour row0 = -1 * feature0 -> relu(2) = 2
    off, P = _offsets(32, 2)
    w = np.zeros(P, F)
    o, fo, fi = off["feature"]
    w[o + fo * fi] = -2.0
    w[off["colour"][0]] = -1.0
    w[off["rgb"][0] + 2 * 32] = 1.0                        # blue reads colour channel 0
    s = _tiny_scene(oracle, w)
    raw = s.field(0, np.array([0.4, 0.5, 0.6], F), np.array([0, 0, 1], F), raw=True)
    assert raw[3] == 2.0 and raw[1] == 0.0 and raw[2] == 0.0


@pytest.mark.parametrize("width,n_hidden,act", [(32, 2, 1), (32, 3, 1), (64, 3, 0)])
def test_field_matches_float64_torch(oracle, width, n_hidden, act):
    off, P = _offsets(width, n_hidden)
    rng = np.random.default_rng(width + n_hidden)
    w = (rng.uniform(-0.4, 0.4, P)).astype(F)
    s = _tiny_scene(oracle, w, n_hidden=n_hidden, width=width, act=act)
    c, ih = s.subfield_frame(0)
    tw = torch.from_numpy(w.astype(np.float64))

    def lin(name, x):
        o, fo, fi = off[name]
        return torch.nn.functional.linear(x, tw[o:o + fo * fi].reshape(fo, fi), tw[o + fo * fi:o + fo * fi + fo])

    def pe(x, L):
        out = [x]
        for l in range(L):
            out += [torch.sin(2.0 ** l * x), torch.cos(2.0 ** l * x)]
        return torch.cat(out)

    for _ in range(20):
        p = rng.uniform(0.2, 0.9, 3).astype(F)
        d = rng.normal(size=3)
        d = (d / np.linalg.norm(d)).astype(F)
        q = torch.from_numpy((((p - c) * ih).astype(F)).astype(np.float64))
        x = pe(q, 10)
        for l in range(1, n_hidden + 1):
            x = torch.relu(lin(f"trunk{l}", x))
        sig = lin("density", x)
        sig = torch.nn.functional.softplus(sig, threshold=20.0) if act == 1 else torch.relu(sig)
        feat = lin("feature", x)
        col = torch.relu(lin("colour", torch.cat([feat, pe(torch.from_numpy(d.astype(np.float64)), 4)])))
        rgb = torch.sigmoid(lin("rgb", col))
        got = s.field(0, p, d)
        assert abs(got[0] - float(sig)) < 1e-11
        assert np.abs(got[1:] - rgb.numpy()).max() < 1e-12


def test_create_rejects_bad_inputs(oracle):
    off, P = _offsets(32, 2)
    occ = np.full(8, 255, np.uint8)
    lab = np.zeros(8, np.int32)
    kw = dict(dims=(2, 2, 2), box_min=(0, 0, 0), box_max=(1, 1, 1), n_subfields=1, occ_threshold=128)
    with pytest.raises(ValueError):
        oracle.scene(occupancy=occ, voxel_subfield=lab + 1, weights=np.zeros(P, F), **kw)   # label out of range
    w = np.zeros(P, F)
    w[5] = np.nan
    with pytest.raises(ValueError):
        oracle.scene(occupancy=occ, voxel_subfield=lab, weights=w, **kw)
    with pytest.raises(ValueError):
        oracle.scene(occupancy=occ, voxel_subfield=lab, weights=np.zeros(P, F),
                     **{**kw, "box_max": (1, 0, 1)})
