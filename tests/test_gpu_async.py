"""-m gpu: the asynchronous frame pipeline (render.cu): no host wait in the middle of a frame, buffers sized from a
learnt capacity with a re-render of chunks that outgrow it, row bands (r360_render_rows), the 5-byte output format,
CUDA graph capture, host-output bands, a stereoscopic pair in one batch.  Every variant must give the SAME pixels
bit for bit as the plain call, which tests/test_gpu_parity.py compares with the oracle.
SURVEY.md 8(b) ("asynchronous with respect to the host"), 8(e) (row bands), 8(f)1 (stereo)."""
import numpy as np
import pytest

from conftest import get_scene

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


def _far_pose(sc):
    """A pose far outside the box: most rays miss it, so the segments-per-ray ratio is tiny."""
    pose = sc.poses[0].copy()
    pose[3] = sc.box_max[0] + 40.0
    return pose


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_render_returns_before_the_gpu_finishes(r360, precision):
    import torch
    sc = get_scene(3)
    gpu = r360.scene_from(sc)
    gpu.set_precision(precision)
    W, H = (sc.W, sc.H) if precision == "bf16" else (sc.W // 2, sc.H // 2)
    rgb, depth = gpu.render(sc.poses[0], W, H)            # first frame: exact sizing
    ref_rgb, ref_d = rgb.clone(), depth.clone()
    torch.cuda.synchronize()
    not_ready = 0
    for _ in range(5):
        done = torch.cuda.Event()
        gpu.render(sc.poses[0], W, H, rgb, depth, wait=False)
        done.record()
        not_ready += not done.query()                     # asked right after the call returned
        torch.cuda.synchronize()
    assert not_ready >= 4, "r360_render waited for the GPU"
    assert torch.equal(rgb, ref_rgb) and torch.equal(depth, ref_d)
    st = gpu.stats()
    assert st.retries == 0 and st.kernel_launches == 5
    gpu.close()


@pytest.mark.parametrize("wavefront", [False, True])
@pytest.mark.parametrize("precision", ["fp32", "f16"])
def test_chunk_that_outgrows_the_buffers_is_rendered_again(r360, scene2, precision, wavefront):
    import torch
    sc = scene2
    ref = r360.scene_from(sc)
    ref.set_precision(precision)
    rgb0, d0 = ref.render(sc.poses[0], sc.W, sc.H)
    n_samples = ref.stats().samples_emitted
    gpu = r360.scene_from(sc)
    gpu.set_precision(precision)
    gpu.set_wavefront(wavefront)
    gpu.render(_far_pose(sc), sc.W, sc.H)                 # learns a tiny capacity
    assert gpu.stats().retries == 0
    rgb1, d1 = gpu.render(sc.poses[0], sc.W, sc.H)        # far more samples per ray: overflow, re-render in wait()
    st = gpu.stats()
    assert st.retries == 1 and st.samples_emitted == n_samples
    assert torch.equal(rgb0, rgb1) and torch.equal(d0, d1)
    rgb2, d2 = gpu.render(sc.poses[0], sc.W, sc.H)        # now it fits
    assert gpu.stats().retries == 1
    assert torch.equal(rgb0, rgb2) and torch.equal(d0, d2)
    # several chunks, some of which overflow; host-output path re-copies them
    gpu2 = r360.scene_from(sc)
    gpu2.set_precision(precision)
    gpu2.set_wavefront(wavefront)
    gpu2.set_chunk_rays(sc.W * 37)
    gpu2.render(_far_pose(sc), sc.W, sc.H)
    h_rgb, h_d = gpu2.render_batch_host(sc.poses[0], sc.W, sc.H)
    assert gpu2.stats().retries >= 1
    assert np.array_equal(h_rgb[0], rgb0.cpu().numpy()) and np.array_equal(h_d[0], d0.cpu().numpy())
    for s in (ref, gpu, gpu2):
        s.close()


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_row_bands_equal_the_full_frame(r360, scene2, precision):
    import torch
    sc = scene2
    gpu = r360.scene_from(sc)
    gpu.set_precision(precision)
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    rgb, depth = rgb.clone(), depth.clone()
    full_rgb = torch.zeros_like(rgb)
    full_d = torch.zeros_like(depth)
    for r0, r1 in ((0, 100), (100, 101), (101, 256)):     # ragged bands, rendered in place into a full frame
        gpu.render_rows(sc.poses[0], sc.W, sc.H, r0, r1, full_rgb[r0:r1], full_d[r0:r1])
        assert gpu.stats().rays == (r1 - r0) * sc.W
    assert torch.equal(full_rgb, rgb) and torch.equal(full_d, depth)
    band_rgb, band_d = gpu.render_rows(sc.poses[0], sc.W, sc.H, 17, 60)
    assert tuple(band_rgb.shape) == (43, sc.W, 3) and torch.equal(band_rgb, rgb[17:60]) and torch.equal(band_d, depth[17:60])
    # shard.row_band partition of two ranks covers the frame
    from paper_2208_02705_b200.shard import row_band
    parts = [gpu.render_rows(sc.poses[0], sc.W, sc.H, *row_band(sc.H, r, 3))[0].clone() for r in range(3)]
    assert torch.equal(torch.cat(parts, 0), rgb)
    for bad in ((-1, 4), (4, 4), (10, sc.H + 1)):
        with pytest.raises(r360.R360Error):
            gpu.render_rows(sc.poses[0], sc.W, sc.H, *bad)
    gpu.close()


def test_rgb8_d16_output(r360, oracle, scene2):
    import torch
    sc = scene2
    gpu = r360.scene_from(sc)
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    rgb, depth = rgb.cpu().numpy(), depth.cpu().numpy()
    gpu.set_output_format("rgb8_d16")
    rgb8, d16 = gpu.render(sc.poses[0], sc.W, sc.H)
    assert rgb8.dtype == torch.uint8 and d16.dtype == torch.float16
    # exactly the rounding include/r360.h states, applied to the fp32 image
    assert np.array_equal(rgb8.cpu().numpy(), np.rint(np.clip(rgb, 0, 1) * F(255)).astype(np.uint8))
    assert np.array_equal(d16.cpu().numpy(), depth.astype(np.float16))
    # and against the oracle: 1e-4 + half a level
    ref = oracle.scene_from(sc).render_rows(sc.poses[0], sc.W, sc.H, 100, 104)
    err = np.abs(rgb8.cpu().numpy()[100:104].reshape(-1, 3).astype(np.float64) / 255.0 - ref["rgb"])
    assert err.max() <= 1e-4 + 0.5 / 255
    h_rgb, h_d = gpu.render_batch_host(sc.poses[0], sc.W, sc.H)
    assert h_rgb.dtype == np.uint8 and np.array_equal(h_rgb[0], rgb8.cpu().numpy())
    assert np.array_equal(h_d[0], d16.cpu().numpy())
    band_rgb, band_d = gpu.render_rows(sc.poses[0], sc.W, sc.H, 30, 50)
    assert torch.equal(band_rgb, rgb8[30:50]) and torch.equal(band_d, d16[30:50])
    gpu.set_output_format("f32")
    with pytest.raises(r360.R360Error):
        gpu.set_output_format(7)
    gpu.close()


@pytest.mark.parametrize("bands", [1, 2, 4, 7])
def test_host_bands_equal_single_copy(r360, scene2, bands):
    sc = scene2
    gpu = r360.scene_from(sc)
    gpu.set_precision("bf16")
    rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H)
    gpu.set_host_bands(bands)
    h_rgb, h_d = gpu.render_batch_host(sc.poses[0], sc.W, sc.H)
    assert gpu.stats().chunks == (bands if sc.W * sc.H >= 65536 * bands else 1)
    assert np.array_equal(h_rgb[0], rgb.cpu().numpy()) and np.array_equal(h_d[0], depth.cpu().numpy())
    gpu.close()


def test_streaming_host_output(r360, scene2):
    """r360_render_batch_host_async: frames of a roaming path enqueued back to back, each copied to its own host
    buffer behind the next frame's kernels; after r360_host_sync every buffer holds exactly the frame of the
    synchronous call.  The third frame outgrows the buffers learnt from the first two (re-rendered, re-copied)."""
    import torch
    sc = scene2
    gpu = r360.scene_from(sc)
    gpu.set_precision("bf16")
    poses = [_far_pose(sc), _far_pose(sc)]
    for k in range(4):
        p = sc.poses[0].copy()
        p[3] += 0.15 * k
        poses.append(p)
    refs = []
    ref_scene = r360.scene_from(sc)
    ref_scene.set_precision("bf16")
    for p in poses:
        rgb, depth = ref_scene.render(p, sc.W, sc.H)
        refs.append((rgb.cpu().numpy(), depth.cpu().numpy()))
    bufs = [(torch.empty((1, sc.H, sc.W, 3), dtype=torch.float32).pin_memory(),
             torch.empty((1, sc.H, sc.W), dtype=torch.float32).pin_memory()) for _ in poses]
    for b in bufs:
        b[0].fill_(-1.0); b[1].fill_(-1.0)
    for k, (p, (h_rgb, h_d)) in enumerate(zip(poses, bufs)):
        gpu.render_batch_host(p, sc.W, sc.H, h_rgb.numpy(), h_d.numpy(), sync=False)
        if k >= 2:
            # include/r360.h: once the second-next call has returned, a frame is in its host buffers -- read at once,
            # no r360_host_sync (frame 2 is the one that was re-rendered and re-copied)
            assert np.array_equal(bufs[k - 2][0].numpy()[0], refs[k - 2][0]), k
            assert np.array_equal(bufs[k - 2][1].numpy()[0], refs[k - 2][1]), k
    gpu.host_sync()
    assert gpu.stats().retries >= 1
    for (h_rgb, h_d), (rgb, depth) in zip(bufs, refs):
        assert np.array_equal(h_rgb.numpy()[0], rgb) and np.array_equal(h_d.numpy()[0], depth)
    gpu.close()
    ref_scene.close()


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_stereo_pair_in_one_batch(r360, scene2, precision):
    """Stereoscopic mode: two eyes 65 mm apart along the camera's x axis, binned in ONE chunk
    (a subfield's weights are staged once for both eyes); each eye bit-identical to its own mono render."""
    import torch
    sc = scene2
    gpu = r360.scene_from(sc)
    gpu.set_precision(precision)
    from paper_2208_02705_b200.shard import stereo_poses
    pair = stereo_poses(sc.poses[0], 0.065)
    assert np.allclose(np.linalg.norm(pair[0].reshape(3, 4)[:, 3] - pair[1].reshape(3, 4)[:, 3]), 0.065, atol=1e-6)
    rgb2, d2 = gpu.render_batch(pair, sc.W, sc.H)
    st = gpu.stats()
    assert st.chunks == 1 and st.kernel_launches == 5
    rgb2, d2 = rgb2.clone(), d2.clone()
    for e in range(2):
        rgb, depth = gpu.render(pair[e], sc.W, sc.H)
        assert torch.equal(rgb2[e], rgb) and torch.equal(d2[e], depth)
    assert not torch.equal(rgb2[0], rgb2[1])
    gpu.close()


def test_cuda_graph_capture_and_replay(r360, scene2):
    import torch
    sc = scene2
    gpu = r360.scene_from(sc)
    gpu.set_precision("bf16")
    pose_b = sc.poses[0].copy()
    pose_b[3] += 0.3
    ref_a = [t.clone() for t in gpu.render(sc.poses[0], sc.W, sc.H)]
    ref_b = [t.clone() for t in gpu.render(pose_b, sc.W, sc.H)]
    rgb = torch.zeros((1, sc.H, sc.W, 3), dtype=torch.float32, device="cuda")
    depth = torch.zeros((1, sc.H, sc.W), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        gpu.use_current_torch_stream()
        gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth)           # warm on the capture stream
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth, wait=False)
        rgb.zero_(); depth.zero_()
        graph.replay()
        gpu.graph_status()
        assert torch.equal(rgb[0], ref_a[0]) and torch.equal(depth[0], ref_a[1])
        gpu.set_graph_poses(pose_b)                                  # another pose, same graph
        graph.replay()
        gpu.graph_status()
        assert torch.equal(rgb[0], ref_b[0]) and torch.equal(depth[0], ref_b[1])
        # a replay whose samples outgrow the captured buffers reports it instead of truncating
        gpu2 = r360.scene_from(sc)
        gpu2.use_current_torch_stream()
        gpu2.render(_far_pose(sc), sc.W, sc.H, rgb, depth)
        torch.cuda.synchronize()
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=side):
            gpu2.render(_far_pose(sc), sc.W, sc.H, rgb, depth, wait=False)
        g2.replay()
        gpu2.graph_status()
        gpu2.set_graph_poses(sc.poses[0])
        g2.replay()
        with pytest.raises(r360.R360Error) as e:
            gpu2.graph_status()
        assert e.value.status == 6
        torch.cuda.synchronize()
    del graph, g2
    gpu.close()
    gpu2.close()


def test_stale_graph_is_reported(r360, scene2):
    """A captured graph holds raw buffer addresses and capacities.  A later call outside the capture that frees or
    reallocates one of them (here: a frame four times as large) makes the graph stale: r360_graph_status and
    r360_set_graph_poses report R360_ERR_CAPACITY until the frame is captured again."""
    import torch
    sc = scene2
    gpu = r360.scene_from(sc)
    rgb = torch.zeros((1, sc.H, sc.W, 3), dtype=torch.float32, device="cuda")
    depth = torch.zeros((1, sc.H, sc.W), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        gpu.use_current_torch_stream()
        ref = [t.clone() for t in gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth)]
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth, wait=False)
        graph.replay()
        gpu.graph_status()
        gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth)               # same size: nothing moves, the graph stays valid
        gpu.graph_status()
        gpu.set_graph_poses(sc.poses[0])
        gpu.render(sc.poses[0], 2 * sc.W, 2 * sc.H)                   # other tables, larger chunk buffers
        torch.cuda.synchronize()
        for call in (gpu.graph_status, lambda: gpu.set_graph_poses(sc.poses[0])):
            with pytest.raises(r360.R360Error) as e:
                call()
            assert e.value.status == 6
        gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth)               # builds the tables of this size again
        torch.cuda.synchronize()
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=side):
            gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth, wait=False)
        rgb.zero_(); depth.zero_()
        g2.replay()
        gpu.graph_status()
        assert torch.equal(rgb[0], ref[0]) and torch.equal(depth[0], ref[1])
        torch.cuda.synchronize()
    del graph, g2
    gpu.close()


def test_capture_behind_an_unsettled_frame_is_refused(r360, scene2):
    """A frame whose chunks nobody has verified (no r360_wait) may still need a re-render, which a capture cannot do
    and would silently drop: the captured call is refused (INVALID_ARG); after r360_wait the frame is complete."""
    import torch
    sc = scene2
    ref = r360.scene_from(sc)
    want = [t.clone() for t in ref.render(sc.poses[0], sc.W, sc.H)]
    gpu = r360.scene_from(sc)
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        gpu.use_current_torch_stream()
        gpu.render(_far_pose(sc), sc.W, sc.H)                          # learns a tiny capacity
        rgb, depth = gpu.render(sc.poses[0], sc.W, sc.H, wait=False)   # overflows; not yet re-rendered
        graph = torch.cuda.CUDAGraph()
        with pytest.raises(r360.R360Error) as e:
            with torch.cuda.graph(graph, stream=side, capture_error_mode="thread_local"):
                gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth, wait=False)
        assert e.value.status == 1
        gpu.wait()
        torch.cuda.synchronize()
        assert gpu.stats().retries == 1
        assert torch.equal(rgb, want[0]) and torch.equal(depth, want[1])
    gpu.close()
    ref.close()


def test_capture_of_a_cold_scene_is_refused(r360, scene1):
    import torch
    sc = scene1
    gpu = r360.scene_from(sc)
    side = torch.cuda.Stream()
    rgb = torch.zeros((1, sc.H, sc.W, 3), dtype=torch.float32, device="cuda")
    depth = torch.zeros((1, sc.H, sc.W), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        gpu.use_current_torch_stream()
        graph = torch.cuda.CUDAGraph()
        with pytest.raises(r360.R360Error) as e:
            with torch.cuda.graph(graph, stream=side, capture_error_mode="thread_local"):
                gpu.render(sc.poses[0], sc.W, sc.H, rgb, depth, wait=False)
        assert e.value.status == 6
    torch.cuda.synchronize()
    gpu.close()
