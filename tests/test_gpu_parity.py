"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element.

Bars (BASELINE.json north_star): sample counts / subfield ids / t bit-exact; fp32 RGB and depth
within 1e-4 absolute; bf16 tensor-core RGB within 2e-3 absolute (tests/test_gpu_tc.py)."""
import numpy as np
import pytest

from conftest import get_scene
from gpu_util import AMB_BAND, check_image, ray_major_index, with_density_bias

pytestmark = pytest.mark.gpu
F = np.float32


@pytest.fixture(scope="module")
def r360():
    import torch
    assert torch.cuda.is_available()
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def _cmp_samples(r360, oracle, sc, pose, W, H, **override):
    gpu = r360.scene_from(sc, **override)
    kw = {k: v for k, v in override.items()}
    ora = oracle.scene_from(sc) if not kw else None
    assert ora is not None
    counts, offsets, t, sid = gpu.debug_samples(pose, W, H)
    oc, ot, osid = ora.samples_rows(pose, W, H)
    counts, offsets = counts.cpu().numpy().view(np.uint32), offsets.cpu().numpy().view(np.uint32)
    assert np.array_equal(counts, oc)                                           # bit-exact counts
    idx = ray_major_index(counts, offsets)                                      # valid layout, any ray order
    assert np.array_equal(t.cpu().numpy().view(np.uint32)[idx], ot.view(np.uint32))  # bit-exact distances
    assert np.array_equal(sid.cpu().numpy()[idx], osid)                         # exact subfield ids
    gpu.close()
    return int(oc.sum())


def test_sampler_bit_exact_config1(r360, oracle, scene1):
    n = _cmp_samples(r360, oracle, scene1, scene1.poses[0], scene1.W, scene1.H)
    assert n == 39808


def test_sampler_bit_exact_config2(r360, oracle, scene2):
    _cmp_samples(r360, oracle, scene2, scene2.poses[0], scene2.W, scene2.H)


@pytest.mark.parametrize("W,H", [(1, 1), (37, 19), (257, 3), (2, 200)])
def test_sampler_ragged_sizes(r360, oracle, scene1, W, H):
    _cmp_samples(r360, oracle, scene1, scene1.poses[0], W, H)


def test_sampler_camera_outside_and_rotated(r360, oracle, scene1):
    # outside the box (t0 > 0 for rays that enter, no samples for rays that miss), tilted pose
    a, b = 0.3, -0.7
    ra = np.array([[1, 0, 0], [0, np.cos(a), -np.sin(a)], [0, np.sin(a), np.cos(a)]])
    rb = np.array([[np.cos(b), 0, np.sin(b)], [0, 1, 0], [-np.sin(b), 0, np.cos(b)]])
    pose = np.concatenate([ra @ rb, np.array([[7.3], [-1.1], [0.4]])], 1).astype(F).reshape(12)
    n = _cmp_samples(r360, oracle, scene1, pose, 96, 48)
    assert n > 0


def _render_cmp(r360, oracle, sc, tol=1e-4, precision="fp32", weights=None, W=None, H=None, **desc_over):
    W = W or sc.W
    H = H or sc.H
    over = dict(desc_over)
    if weights is not None:
        over["weights"] = weights
    gpu = r360.scene_from(sc, **over)
    gpu.set_precision(precision)
    okw = dict(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
               hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, pe_pos_levels=sc.pe_pos_levels,
               pe_dir_levels=sc.pe_dir_levels, samples_per_voxel=sc.samples_per_voxel,
               t_threshold=sc.t_threshold, density_activation=sc.density_activation,
               occ_threshold=sc.occ_threshold, occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield,
               weights=sc.weights if weights is None else weights)
    okw.update(desc_over)
    ora = oracle.scene(**okw)
    rgb, depth = gpu.render(sc.poses[0], W, H)
    ref = ora.render_rows(sc.poses[0], W, H)
    st = gpu.stats()
    assert st.samples_emitted == int(ref["n_emitted"].sum())
    assert st.rays == W * H
    res = check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, tol)
    gpu.close()
    return res, st, ref


def test_render_fp32_config1(r360, oracle, scene1):
    (e_rgb, e_d, n_amb), st, ref = _render_cmp(r360, oracle, scene1)
    assert st.samples_used == st.samples_emitted == 39808
    assert st.kernel_launches == 5


def test_render_fp32_config2(r360, oracle, scene2):
    _render_cmp(r360, oracle, scene2)


def test_render_fp32_early_out(r360, oracle, scene1):
    # dense medium: most rays stop early; the stopping sample must match the oracle's
    w = with_density_bias(scene1, 40.0)
    (e_rgb, e_d, n_amb), st, ref = _render_cmp(r360, oracle, scene1, weights=w)
    assert st.samples_used < st.samples_emitted
    amb = ref["ambiguity"] < 1e-3
    if not amb.any():
        assert st.samples_used == int(ref["n_used"].sum())


@pytest.mark.parametrize("over", [dict(samples_per_voxel=12), dict(samples_per_voxel=5),
                                  dict(samples_per_voxel=1), dict(samples_per_voxel=128),
                                  dict(density_activation=0), dict(t_threshold=0.0)])
def test_render_fp32_variants(r360, oracle, scene1, over):
    _render_cmp(r360, oracle, scene1, **over)


def test_render_fp32_width64_hidden3(r360, oracle):
    from scenegen import mlp_param_count
    sc = get_scene(1)
    P = mlp_param_count(64, 3)
    rng = np.random.default_rng(7)
    w = rng.uniform(-0.25, 0.25, sc.n_subfields * P).astype(F)
    _render_cmp(r360, oracle, sc, weights=w, hidden_width=64, n_hidden=3)


def test_empty_scene_is_black(r360, scene1):
    import torch
    sc = scene1
    gpu = r360.scene_from(sc, occupancy=np.zeros_like(sc.occupancy))
    rgb, depth = gpu.render(sc.poses[0], 64, 32)
    assert torch.all(rgb == 0) and torch.all(depth == 0)
    assert gpu.stats().samples_emitted == 0


def test_chunked_and_batched_equal_single(r360, scene1):
    import torch
    sc = scene1
    gpu = r360.scene_from(sc)
    rgb0, d0 = gpu.render(sc.poses[0], 64, 32)
    rgb0, d0 = rgb0.clone(), d0.clone()
    gpu.set_chunk_rays(300)                                     # 7 ragged chunks
    rgb1, d1 = gpu.render(sc.poses[0], 64, 32)
    assert gpu.stats().chunks == 7
    assert torch.equal(rgb0, rgb1) and torch.equal(d0, d1)
    pose2 = sc.poses[0].copy()
    pose2[3] += 0.4
    poses = np.stack([sc.poses[0], pose2])
    rgbb, db = gpu.render_batch(poses, 64, 32)
    gpu.set_chunk_rays(1 << 22)
    rgb2, d2 = gpu.render(pose2, 64, 32)
    assert torch.equal(rgbb[0], rgb0) and torch.equal(rgbb[1], rgb2) and torch.equal(db[1], d2)
    h_rgb, h_d = gpu.render_batch_host(poses, 64, 32)
    assert np.array_equal(h_rgb, rgbb.cpu().numpy()) and np.array_equal(h_d, db.cpu().numpy())
    gpu.set_chunk_rays(300)                                     # 14 chunks, each copied to the host behind the next
    h_rgb2, h_d2 = gpu.render_batch_host(poses, 64, 32)
    assert gpu.stats().chunks == 14
    assert np.array_equal(h_rgb2, h_rgb) and np.array_equal(h_d2, h_d)


def test_render_rejects_bad_arguments(r360, scene1):
    gpu = r360.scene_from(scene1)
    bad = scene1.poses[0].copy()
    bad[5] = np.nan
    with pytest.raises(r360.R360Error) as e:
        gpu.render(bad, 64, 32)
    assert e.value.status == 1
    L = r360.lib()
    assert L.r360_render(gpu._h, None, 64, 32, None, None) == 1
    # reading B5: a (nearly) singular 3x3 part maps some pixel's unit direction to ~zero -- refused by both sides
    for scale_z in (0.0, 1e-7):
        flat = scene1.poses[0].copy().reshape(3, 4)
        flat[:, 2] *= scale_z
        with pytest.raises(r360.R360Error) as e:
            gpu.render(flat.reshape(12), 64, 32)
        assert e.value.status == 1
        with pytest.raises(r360.R360Error):
            gpu.render_batch(np.stack([scene1.poses[0], flat.reshape(12)]), 64, 32)
        with pytest.raises(r360.R360Error):
            gpu.debug_samples(flat.reshape(12), 64, 32)
    rgb, depth = gpu.render(scene1.poses[0] * np.array([2, 2, 2, 1] * 3, F), 64, 32)   # a scaled rotation is fine
    assert float(depth.max()) > 0


def test_full_size_config3_sampled(r360, oracle):
    """BASELINE config 3 in the launch configuration bench.py times: 2048x1024, ~1k subfields.
    The oracle renders a sample of pixels one by one; counts are compared on whole rows."""
    sc = get_scene(3)
    gpu = r360.scene_from(sc)
    ora = oracle.scene_from(sc)
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    st = gpu.stats()
    rng = np.random.default_rng(3)
    px = rng.integers(0, sc.W, 3000).astype(np.int32)
    py = rng.integers(0, sc.H, 3000).astype(np.int32)
    ref = ora.render_pixels(sc.poses[0], sc.W, sc.H, px, py)
    g_rgb = rgb.cpu().numpy()[py, px]
    g_d = depth.cpu().numpy()[py, px]
    check_image(g_rgb, g_d, ref, 1e-4)
    counts, offsets, t, sid = gpu.debug_samples(sc.poses[0], sc.W, sc.H)
    counts = counts.cpu().numpy().view(np.uint32).reshape(sc.H, sc.W)
    offsets = offsets.cpu().numpy().view(np.uint32).reshape(sc.H, sc.W)
    ray_major_index(counts, offsets)
    t_np, sid_np = t.cpu().numpy().view(np.uint32), sid.cpu().numpy()
    assert int(counts.sum()) == st.samples_emitted
    assert np.array_equal(counts[py, px], ref["n_emitted"])
    for row in (0, 511, 1023):
        oc, ot, osid = ora.samples_rows(sc.poses[0], sc.W, sc.H, row, row + 1)
        assert np.array_equal(counts[row], oc)
        oc64 = oc.astype(np.int64)
        idx = np.repeat(offsets[row].astype(np.int64), oc64) + (np.arange(int(oc64.sum())) - np.repeat(np.cumsum(oc64) - oc64, oc64))
        assert np.array_equal(t_np[idx], ot.view(np.uint32))
        assert np.array_equal(sid_np[idx], osid)


@pytest.mark.parametrize("config,W,H,f", [(1, 160, 90, 80.0), (2, 320, 180, 200.0), (1, 37, 19, 11.5)])
def test_pinhole_view(r360, oracle, config, W, H, f):
    """The roaming (perspective) view, reading P: samples bit-exact, fp32 image within 1e-4, bf16 within 2e-3."""
    sc = get_scene(config)
    cam = ("pinhole", f, f * 1.1, W / 2.0 + 0.25, H / 2.0 - 0.5)
    ora = oracle.scene_from(sc)
    ora.set_camera(*cam)
    gpu = r360.scene_from(sc)
    gpu.set_camera(*cam)
    pose = sc.poses[0]
    counts, offsets, t, sid = gpu.debug_samples(pose, W, H)
    oc, ot, osid = ora.samples_rows(pose, W, H)
    counts, offsets = counts.cpu().numpy().view(np.uint32), offsets.cpu().numpy().view(np.uint32)
    assert np.array_equal(counts, oc)
    idx = ray_major_index(counts, offsets)
    assert np.array_equal(t.cpu().numpy().view(np.uint32)[idx], ot.view(np.uint32))
    assert np.array_equal(sid.cpu().numpy()[idx], osid)
    ref = ora.render_rows(pose, W, H)
    rgb, depth = gpu.render(pose, W, H)
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 1e-4)
    gpu.set_precision("bf16")
    rgb, depth = gpu.render(pose, W, H)
    t_max = float(np.linalg.norm(np.array(sc.box_max) - np.array(sc.box_min)))
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 2e-3, amb_band=AMB_BAND["bf16"], depth_tol=2e-3 * t_max)
    # back to the panorama: the tables are rebuilt for the other camera
    gpu.set_camera("equirect")
    gpu.set_precision("fp32")
    ora.set_camera("equirect")
    rgb, depth = gpu.render(pose, 64, 32)
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ora.render_rows(pose, 64, 32), 1e-4)
    with pytest.raises(r360.R360Error):
        gpu.set_camera("pinhole", -1.0, 1.0, 0.0, 0.0)
    gpu.close()
    ora.close()


def test_more_subfields_than_the_shared_memory_histogram_holds(r360, oracle):
    """n_subfields > 8192: the sampler's per-block histograms and cursors do not fit shared memory and every bin
    update goes through the global counters (bin_ovf / bin_cursor).  Samples bit-exact, fp32 and bf16 images within
    their bars, wavefront passes identical to the single pass."""
    from scenegen import mlp_param_count, weight_layout
    sc = get_scene(1)
    n = 8200
    occ = np.asarray(sc.occupancy).reshape(-1) >= sc.occ_threshold
    lab = np.asarray(sc.voxel_subfield).reshape(-1).copy()
    v = np.flatnonzero(occ)
    lab[v] = (lab[v].astype(np.int64) * 512 + v % 512) % n
    rng = np.random.default_rng(77)
    parts = []
    for name, fo, fi in weight_layout(sc.hidden_width, sc.n_hidden):
        a = np.sqrt(6.0 / (fi + fo))
        parts.append(rng.uniform(-a, a, (n, fo * fi)))
        parts.append(np.full((n, fo), 1.0 if name == "density" else 0.0))
    w = np.concatenate(parts, 1).astype(F).reshape(-1)
    assert w.size == n * mlp_param_count(sc.hidden_width, sc.n_hidden)
    over = dict(n_subfields=n, voxel_subfield=lab, weights=w)
    gpu = r360.scene_from(sc, **over)
    okw = dict(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, hidden_width=sc.hidden_width,
               n_hidden=sc.n_hidden, pe_pos_levels=sc.pe_pos_levels, pe_dir_levels=sc.pe_dir_levels,
               samples_per_voxel=sc.samples_per_voxel, t_threshold=sc.t_threshold,
               density_activation=sc.density_activation, occ_threshold=sc.occ_threshold, occupancy=sc.occupancy, **over)
    ora = oracle.scene(**okw)
    pose, W, H = sc.poses[0], sc.W, sc.H
    counts, offsets, t, sid = gpu.debug_samples(pose, W, H)
    oc, ot, osid = ora.samples_rows(pose, W, H)
    counts, offsets = counts.cpu().numpy().view(np.uint32), offsets.cpu().numpy().view(np.uint32)
    assert np.array_equal(counts, oc)
    idx = ray_major_index(counts, offsets)
    assert np.array_equal(t.cpu().numpy().view(np.uint32)[idx], ot.view(np.uint32))
    assert np.array_equal(sid.cpu().numpy()[idx], osid)
    ref = ora.render_rows(pose, W, H)
    rgb, depth = gpu.render(pose, W, H)
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 1e-4)
    gpu.set_wavefront(True)
    rgb_w, depth_w = gpu.render(pose, W, H)
    assert np.array_equal(rgb.cpu().numpy().view(np.uint32), rgb_w.cpu().numpy().view(np.uint32))
    assert np.array_equal(depth.cpu().numpy().view(np.uint32), depth_w.cpu().numpy().view(np.uint32))
    gpu.set_wavefront(False)
    gpu.set_precision("bf16")
    rgb, depth = gpu.render(pose, W, H)
    t_max = float(np.linalg.norm(np.array(sc.box_max) - np.array(sc.box_min)))
    check_image(rgb.cpu().numpy(), depth.cpu().numpy(), ref, 2e-3, amb_band=AMB_BAND["bf16"], depth_tol=2e-3 * t_max)
    gpu.close()
    ora.close()


def _rows_bit_exact(gpu, ora, pose, W, H, rows):
    """Whole-image layout check plus (count, t bits, subfield id) of every sample of the given rows against the
    oracle; the sample arrays stay on the device (hundreds of millions of samples), only the rows' entries come back.
    Returns the per-ray counts [H, W]."""
    import torch
    counts, offsets, t, sid = gpu.debug_samples(pose, W, H)
    c = counts.cpu().numpy().view(np.uint32).astype(np.int64)
    o = offsets.cpu().numpy().view(np.uint32).astype(np.int64)
    total = int(c.sum())
    assert total == t.numel() == sid.numel()
    # the per-ray ranges [offset, offset + count) are disjoint and cover [0, total), in any ray order
    live = np.flatnonzero(c)
    order = live[np.argsort(o[live], kind="stable")]
    assert o[order[0]] == 0 and np.array_equal(o[order[1:]], (o[order] + c[order])[:-1])
    assert o[order[-1]] + c[order[-1]] == total
    c, o = c.reshape(H, W), o.reshape(H, W)
    t_bits = t.view(torch.int32)
    rows = sorted({int(np.unravel_index(int(c.argmax()), c.shape)[0]) if r == "longest" else r for r in rows})
    for row in rows:
        oc, ot, osid = ora.samples_rows(pose, W, H, row, row + 1)
        assert np.array_equal(c[row], oc), row                                   # bit-exact counts
        oc64 = oc.astype(np.int64)
        idx = np.repeat(o[row], oc64) + (np.arange(int(oc64.sum())) - np.repeat(np.cumsum(oc64) - oc64, oc64))
        idx = torch.from_numpy(idx).cuda()
        assert np.array_equal(t_bits[idx].cpu().numpy(), ot.view(np.int32)), row  # bit-exact distances
        assert np.array_equal(sid[idx].cpu().numpy(), osid), row                  # exact subfield ids
    return c, rows


def test_sampler_bit_exact_config5_rows(r360, oracle):
    """BASELINE config 5 (30 % occupancy) at full size: rows 0, H/2, H-1 and the row of the longest ray, every sample.
    Rays that cross more than kHitCap = 64 occupied voxels leave k_count's per-ray hit buffer and are walked again
    by k_emit (sampler.cu): at least one compared ray must be of that kind, so that branch is held to the oracle
    bit for bit and not only through an image tolerance (north_star: counts and ids bit-exact)."""
    sc = get_scene(5)
    gpu = r360.scene_from(sc)
    ora = oracle.scene_from(sc)
    K = sc.samples_per_voxel
    c, rows = _rows_bit_exact(gpu, ora, sc.poses[0], sc.W, sc.H, (0, sc.H // 2, sc.H - 1, "longest"))
    segs = c[rows] // K
    assert segs.max() > 64 and (segs > 64).sum() >= 10, "no compared ray takes the re-walk branch"
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    assert gpu.stats().samples_emitted == int(c.sum())                           # the render agrees with the tap
    gpu.close()
    ora.close()


def test_sampler_bit_exact_config4_rows_and_pose_boundary(r360, oracle):
    """BASELINE config 4 (512 x 512 x 96 grid: skip distances saturate at 255; K = 12; 4096 x 2048): three rows of
    pose 3, every sample; then two poses in one batch with a ray chunk that straddles the pose boundary, each image
    equal bit for bit to its single render."""
    import torch
    sc = get_scene(4)
    gpu = r360.scene_from(sc)
    ora = oracle.scene_from(sc)
    assert sc.samples_per_voxel == 12 and tuple(sc.dims) == (512, 512, 96)
    _rows_bit_exact(gpu, ora, sc.poses[3], sc.W, sc.H, (0, sc.H // 2, sc.H - 1))
    ora.close()
    gpu.set_precision("bf16")
    singles = []
    for p in (sc.poses[3], sc.poses[4]):
        rgb, depth = gpu.render(p, sc.W, sc.H)
        singles.append((rgb.clone(), depth.clone()))
    assert gpu.stats().samples_emitted > 0
    rays = sc.W * sc.H
    gpu.set_chunk_rays(3 << 20)                                                  # chunk 2 = rays [6 Mi, 9 Mi): both poses
    assert (2 * (3 << 20)) < rays < (3 * (3 << 20))
    rgb2, d2 = gpu.render_batch(np.stack([sc.poses[3], sc.poses[4]]), sc.W, sc.H)
    assert gpu.stats().chunks == (2 * rays + (3 << 20) - 1) // (3 << 20)
    for b in range(2):
        assert torch.equal(rgb2[b], singles[b][0]) and torch.equal(d2[b], singles[b][1])
    assert not torch.equal(rgb2[0], rgb2[1])
    gpu.close()
