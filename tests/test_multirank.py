"""World-size-2 gloo test (CPU) of the multi-GPU host logic: rank -> pose, rank -> row band, and the
gather of row bands into one image.  The render itself needs a GPU and is covered by -m gpu tests."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2208_02705_b200.shard import gather_rows, rank_pose, render_sharded, row_band, stereo_poses


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, H, W, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    r0, r1 = row_band(H, rank, world)
    rows = torch.arange(r0, r1, dtype=torch.float32)[:, None, None]
    band = rows * 1000 + torch.arange(W, dtype=torch.float32)[None, :, None] + torch.tensor([0.0, 0.25, 0.5])
    full = gather_rows(band, H, rank, world, dist)

    # the function bench.py --scaling strong calls, with a stand-in for Scene.render_rows that writes the same
    # synthetic pixels (the render itself needs a GPU): every rank must end up with the whole frame
    def fake_render_rows(pose, W_, H_, row0, row1, out_rgb, out_depth):
        rr = torch.arange(row0, row1, dtype=torch.float32)[:, None]
        cc = torch.arange(W_, dtype=torch.float32)[None, :]
        out_rgb.copy_((rr * 1000 + cc)[:, :, None] + torch.tensor([0.0, 0.25, 0.5]))
        out_depth.copy_(rr * 7 + cc)
    full_rgb = torch.full((H, W, 3), -1.0)
    full_d = torch.full((H, W), -1.0)
    rows = render_sharded(fake_render_rows, None, W, H, rank, world, dist, full_rgb, full_d)
    assert rows == (r0, r1)
    assert torch.equal(full_rgb, full)
    assert torch.equal(full_d, torch.arange(H, dtype=torch.float32)[:, None] * 7 + torch.arange(W, dtype=torch.float32)[None, :])
    # max-over-ranks timing reduction used by bench.py
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    q.put((rank, full.numpy(), float(t.item())))
    dist.destroy_process_group()


def test_row_bands_partition_every_size():
    for H in (1, 2, 7, 32, 1024, 1025):
        for world in (1, 2, 3, 8):
            bands = [row_band(H, r, world) for r in range(world)]
            assert bands[0][0] == 0 and bands[-1][1] == H
            assert all(bands[i][1] == bands[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in bands]
            assert max(sizes) - min(sizes) <= 1


def test_rank_pose_is_a_yaw_about_world_up():
    pose = np.array([0, 0, 1, 1.5, -1, 0, 0, -2.5, 0, -1, 0, 0.25], np.float32)
    assert np.array_equal(rank_pose(pose, 0, 4), pose)
    p1 = rank_pose(pose, 1, 4).reshape(3, 4)
    r = p1[:, :3].astype(np.float64)
    assert np.allclose(r @ r.T, np.eye(3), atol=1e-6)
    assert np.allclose(p1[:, 3], [1.5, -2.5, 0.25])
    assert np.allclose(r[:, 2], [0, 1, 0], atol=1e-6)       # forward (+x) turned by 90 degrees to +y
    assert np.allclose(r[:, 1], [0, 0, -1], atol=1e-6)      # camera down stays world -z


def test_stereo_poses_are_one_eye_distance_apart_along_camera_x():
    pose = np.array([0, 0, 1, 1.5, -1, 0, 0, -2.5, 0, -1, 0, 0.25], np.float32)    # camera x = world -y
    pair = stereo_poses(pose, 0.065).reshape(2, 3, 4)
    assert np.array_equal(pair[0][:, :3], pose.reshape(3, 4)[:, :3]) and np.array_equal(pair[1][:, :3], pair[0][:, :3])
    assert np.allclose(pair[1][:, 3] - pair[0][:, 3], [0, -0.065, 0], atol=1e-7)
    assert np.allclose(0.5 * (pair[0][:, 3] + pair[1][:, 3]), [1.5, -2.5, 0.25], atol=1e-7)


import pytest


@pytest.mark.parametrize("H", [33, 32])
def test_two_gloo_ranks_gather_a_ragged_image(H):
    world, W = 2, 8
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, H, W, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    expect = (np.arange(H, dtype=np.float32)[:, None, None] * 1000 + np.arange(W, dtype=np.float32)[None, :, None]
              + np.array([0.0, 0.25, 0.5], np.float32))
    for rank, full, tmax in res:
        assert np.array_equal(full, expect)
        assert tmax == 2.0
