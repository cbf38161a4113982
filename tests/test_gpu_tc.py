"""-m gpu: the tensor-core MLP path (tcgen05; bfloat16 operands = BASELINE.json's "bf16 tensor-core variant", and
the same kernel with binary16 operands) against the oracle: RGB within 2e-3 absolute, max over pixels
(BASELINE.json north_star).  Depth is a sum of w_i * t_i with t up to the scene diagonal, so its bound scales
with the ray length: 2e-3 * t_max."""
import numpy as np
import pytest

from conftest import get_scene
from gpu_util import AMB_BAND, check_image, with_density_bias

pytestmark = pytest.mark.gpu
F = np.float32
TOL = 2e-3


@pytest.fixture(scope="module")
def r360():
    import torch
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def _t_max(sc):
    return float(np.linalg.norm(np.array(sc.box_max) - np.array(sc.box_min)))


def _cmp(r360, oracle, sc, weights=None, amb_band=None, px=None, py=None, tol=TOL, precision="bf16", pose=None,
         **desc_over):
    amb_band = AMB_BAND[precision] if amb_band is None else amb_band
    over = dict(desc_over)
    if weights is not None:
        over["weights"] = weights
    gpu = r360.scene_from(sc, **over)
    gpu.set_precision(precision)
    pose = sc.poses[0] if pose is None else pose
    okw = dict(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
               hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, pe_pos_levels=sc.pe_pos_levels,
               pe_dir_levels=sc.pe_dir_levels, samples_per_voxel=sc.samples_per_voxel,
               t_threshold=sc.t_threshold, density_activation=sc.density_activation,
               occ_threshold=sc.occ_threshold, occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield,
               weights=sc.weights if weights is None else weights)
    okw.update(desc_over)
    ora = oracle.scene(**okw)
    rgb, depth = gpu.render(pose, sc.W, sc.H)
    st = gpu.stats()
    rgb, depth = rgb.cpu().numpy(), depth.cpu().numpy()
    if px is None:
        ref = ora.render_rows(pose, sc.W, sc.H)
        assert st.samples_emitted == int(ref["n_emitted"].sum())
    else:
        ref = ora.render_pixels(pose, sc.W, sc.H, px, py)
        rgb, depth = rgb[py, px], depth[py, px]
    depth_tol = tol * _t_max(sc) if precision != "fp32" else tol
    res = check_image(rgb, depth, ref, tol, amb_band=amb_band, depth_tol=depth_tol)
    gpu.close()
    return res


def test_sass_has_tcgen05_and_tma():
    import subprocess
    import paper_2208_02705_b200 as m
    sass = subprocess.run(["cuobjdump", "-sass", m.lib_path()], capture_output=True, text=True).stdout
    assert "UTCHMMA" in sass and "LDTM" in sass and "STTM" in sass and "UBLKCP" in sass


TC = pytest.mark.parametrize("prec", ["bf16", "f16"])


@TC
def test_render_tc_config1(r360, oracle, scene1, prec):
    e_rgb, e_d, n_amb = _cmp(r360, oracle, scene1, precision=prec)
    print("config1", prec, "max rgb err", e_rgb, "depth", e_d)


@TC
def test_render_tc_config2(r360, oracle, scene2, prec):
    e_rgb, e_d, n_amb = _cmp(r360, oracle, scene2, precision=prec)
    print("config2", prec, "max rgb err", e_rgb, "depth", e_d)


@TC
@pytest.mark.parametrize("over", [dict(samples_per_voxel=12), dict(samples_per_voxel=5),
                                  dict(samples_per_voxel=1), dict(samples_per_voxel=16),
                                  dict(samples_per_voxel=128),
                                  dict(density_activation=0), dict(t_threshold=0.0)])
def test_render_tc_variants(r360, oracle, scene1, over, prec):
    _cmp(r360, oracle, scene1, precision=prec, **over)


@TC
def test_render_tc_width64(r360, oracle, prec):
    from scenegen import mlp_param_count, weight_layout
    sc = get_scene(1)
    rng = np.random.default_rng(11)
    parts = []
    for name, fo, fi in weight_layout(64, 3):
        a = np.sqrt(6.0 / (fi + fo))
        parts.append(rng.uniform(-a, a, (sc.n_subfields, fo * fi)))
        b = rng.uniform(-0.1, 0.1, (sc.n_subfields, fo))
        if name == "density":
            b += 1.0
        parts.append(b)
    w = np.concatenate(parts, 1).astype(F).reshape(-1)
    assert w.size == sc.n_subfields * mlp_param_count(64, 3)
    _cmp(r360, oracle, sc, weights=w, hidden_width=64, n_hidden=3, precision=prec)


BF16_SINGLE_SAMPLE_BOUND = 4e-3
# Rays inside the threshold-ambiguity band (reading G4; gpu_util.check_image) are held to an interval that is at most
# tau * max|rgb| = 1e-3 wider than the tolerance, not to the tolerance itself: on the opaque scenes they must stay a
# minority, or the image comparison would say little.  Measured on the density-bias-40 scene (T falls by e^-1.25 per
# sample, so the threshold is crossed between two samples of most rays): 233 of 2048 rays (11.4 %) lie inside
# bfloat16's band of 0.06, 74 (3.6 %) inside binary16's 0.02; none on the saturating-density scenes.
MAX_AMBIGUOUS_FRACTION = {"bf16": 0.15, "f16": 0.05}


def test_bfloat16_operands_on_opaque_scenes_stay_within_their_format_limit(r360, oracle, scene1):
    """NOT a north_star claim: a characterisation of mode 1 (bfloat16 operands) on scenes whose pixels are the colour
    of their first one or two samples (density bias 40; density beyond binary16's range, stored clamped to 65504).
    A sample's colour through five layers of 8-bit-significand operands is off by up to 2.7e-3
    (tests/test_rounding_budget.py: weights and activations contribute equally, no layer dominates), and with one
    sample per pixel nothing averages it out: measured 2.4e-3 / 2.6e-3 here, above north_star's 2e-3.  The bound
    asserted is that format limit with margin, 4e-3; the mode that meets 2e-3 on these scenes is binary16 operands
    (test_render_f16_opaque_scenes below: 3.3e-4 / 4.5e-4).  On all five BASELINE.json configs, where a pixel
    averages 35-290 samples, mode 1 is within 2e-3 (tests above and below)."""
    n_rays = scene1.W * scene1.H
    e_rgb, e_d, n_amb = _cmp(r360, oracle, scene1, weights=with_density_bias(scene1, 40.0), tol=BF16_SINGLE_SAMPLE_BOUND)
    print("dense stress bf16 max rgb err", e_rgb, "ambiguous", n_amb, "of", n_rays)
    assert n_amb <= MAX_AMBIGUOUS_FRACTION["bf16"] * n_rays
    for act in (0, 1):
        e_rgb, e_d, n_amb = _cmp(r360, oracle, scene1, weights=with_density_bias(scene1, 1.0e6),
                                 tol=BF16_SINGLE_SAMPLE_BOUND, density_activation=act)
        print("saturating density bf16 act", act, "max rgb err", e_rgb, "ambiguous", n_amb, "of", n_rays)
        assert n_amb <= MAX_AMBIGUOUS_FRACTION["bf16"] * n_rays


def test_render_f16_opaque_scenes(r360, oracle, scene1):
    """The scene class the method is for (trained scenes: opaque surfaces end rays early) at
    north_star's bar, 2e-3, on the binary16-operand tensor path: density bias 40 (every pixel is the colour of its
    first one or two samples) and density far beyond binary16's range (sigma stored clamped to 65504, alpha = 1).
    Ambiguity band: gpu_util.AMB_BAND."""
    n_rays = scene1.W * scene1.H
    e_rgb, e_d, n_amb = _cmp(r360, oracle, scene1, weights=with_density_bias(scene1, 40.0),
                             tol=TOL, precision="f16")
    print("dense stress f16 max rgb err", e_rgb, "ambiguous", n_amb, "of", n_rays)
    assert n_amb <= MAX_AMBIGUOUS_FRACTION["f16"] * n_rays
    for act in (0, 1):
        e_rgb, e_d, n_amb = _cmp(r360, oracle, scene1, weights=with_density_bias(scene1, 1.0e6),
                                 tol=TOL, density_activation=act, precision="f16")
        print("saturating density f16 act", act, "max rgb err", e_rgb, "ambiguous", n_amb, "of", n_rays)
        assert n_amb <= MAX_AMBIGUOUS_FRACTION["f16"] * n_rays


def test_f16_refused_when_a_weight_exceeds_binary16(r360, scene1):
    sc = scene1
    w = sc.weights.copy()
    w[5] = 7.0e4                      # a first-layer weight beyond 65504
    gpu = r360.scene_from(sc, weights=w)
    gpu.set_precision("bf16")         # bfloat16 has binary32's range
    with pytest.raises(r360.R360Error):
        gpu.set_precision("f16")
    gpu.close()


def test_tensor_path_refused_when_the_weights_exceed_shared_memory(r360, scene1):
    # refused at r360_set_precision, not by a failing launch at render time
    from scenegen import mlp_param_count
    sc = scene1
    for width, n_hidden, ok in ((32, 6, True), (32, 7, False), (64, 3, True), (64, 4, False)):
        P = mlp_param_count(width, n_hidden)
        gpu = r360.scene_from(sc, weights=np.zeros(sc.n_subfields * P, F), hidden_width=width, n_hidden=n_hidden)
        if ok:
            gpu.set_precision("bf16")
            gpu.render(sc.poses[0], 16, 8)
        else:
            with pytest.raises(r360.R360Error):
                gpu.set_precision("bf16")
        gpu.close()


def test_bf16_refused_for_other_pe_sizes(r360, scene1):
    from scenegen import mlp_param_count
    sc = scene1
    P = mlp_param_count(32, 2, 6, 4)
    gpu = r360.scene_from(sc, weights=np.zeros(sc.n_subfields * P, F), pe_pos_levels=6)
    with pytest.raises(r360.R360Error):
        gpu.set_precision("bf16")


@TC
def test_full_size_config3_tc_sampled(r360, oracle, prec):
    sc = get_scene(3)
    rng = np.random.default_rng(5)
    px = rng.integers(0, sc.W, 3000).astype(np.int32)
    py = rng.integers(0, sc.H, 3000).astype(np.int32)
    e_rgb, e_d, n_amb = _cmp(r360, oracle, sc, px=px, py=py, precision=prec)
    print("config3", prec, "sampled max rgb err", e_rgb, "depth", e_d)


@TC
@pytest.mark.parametrize("n_hidden", [2, 3])
def test_render_tc_random_biases(r360, oracle, n_hidden, prec):
    # every bias path of the tensor kernel: the single bf16 bias row of the first layer, the hi/lo rows of
    # the hidden layers, the bias of the folded feature+colour layer, the fp32 biases of the two heads
    from scenegen import mlp_param_count, weight_layout
    sc = get_scene(1)
    rng = np.random.default_rng(23 + n_hidden)
    parts = []
    for name, fo, fi in weight_layout(32, n_hidden):
        a = np.sqrt(6.0 / (fi + fo))
        parts.append(rng.uniform(-a, a, (sc.n_subfields, fo * fi)))
        b = rng.uniform(-0.5, 0.5, (sc.n_subfields, fo))
        if name == "density":
            b += 1.0
        parts.append(b)
    w = np.concatenate(parts, 1).astype(F).reshape(-1)
    assert w.size == sc.n_subfields * mlp_param_count(32, n_hidden)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, weights=w, n_hidden=n_hidden, precision=prec)
    print("random biases, n_hidden", n_hidden, prec, "max rgb err", e_rgb)
    if prec == "bf16":
        _cmp(r360, oracle, sc, weights=w, n_hidden=n_hidden, precision="fp32", tol=1e-4, amb_band=1e-3)


def _sampled(sc, n, seed):
    rng = np.random.default_rng(seed)
    return rng.integers(0, sc.W, n).astype(np.int32), rng.integers(0, sc.H, n).astype(np.int32)


def test_full_size_config5_sampled(r360, oracle):
    """BASELINE.json config 5 (load imbalance, density bias -2, ~290 samples per ray) at full size, both paths,
    on pixels the oracle renders one by one."""
    sc = get_scene(5)
    px, py = _sampled(sc, 1200, 7)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, px=px, py=py)
    print("config5 bf16 sampled max rgb err", e_rgb, "depth", e_d)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, px=px, py=py, precision="f16")
    print("config5 f16 sampled max rgb err", e_rgb, "depth", e_d)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, px=px, py=py, precision="fp32", tol=1e-4, amb_band=1e-3)
    print("config5 fp32 sampled max rgb err", e_rgb, "depth", e_d)


def test_full_size_config4_one_pose_sampled(r360, oracle):
    """BASELINE.json config 4 (width 64, K = 12, 4096 subfields, 4096x2048) -- one pose of the batch of 8, in two
    ray chunks, both paths, on sampled pixels."""
    sc = get_scene(4)
    px, py = _sampled(sc, 1200, 9)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, px=px, py=py, pose=sc.poses[3])
    print("config4 bf16 sampled max rgb err", e_rgb, "depth", e_d)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, px=px, py=py, pose=sc.poses[3], precision="f16")
    print("config4 f16 sampled max rgb err", e_rgb, "depth", e_d)
    e_rgb, e_d, _ = _cmp(r360, oracle, sc, px=px, py=py, pose=sc.poses[3], precision="fp32", tol=1e-4, amb_band=1e-3)
    print("config4 fp32 sampled max rgb err", e_rgb, "depth", e_d)
