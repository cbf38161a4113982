"""Multi-GPU host logic (one process per GPU): rays are independent, the scene is replicated, so the
path shards by poses (bench.py: one pose per rank, weak scaling) or by image row bands (strong
scaling of one frame) with no data-path collective; only the assembled image is gathered."""
import numpy as np


def rank_pose(pose, rank: int, world: int) -> np.ndarray:
    """Pose of rank r: pose 0 yawed by 2*pi*r/world about the world up axis (z)."""
    m = np.asarray(pose, np.float32).reshape(3, 4).copy()
    if world > 1 and rank:
        a = 2.0 * np.pi * rank / world
        rz = np.array([[np.cos(a), -np.sin(a), 0.0], [np.sin(a), np.cos(a), 0.0], [0.0, 0.0, 1.0]])
        m[:, :3] = (rz @ m[:, :3].astype(np.float64)).astype(np.float32)
    return m.reshape(12)


def row_band(H: int, rank: int, world: int):
    """Contiguous band [row0, row1) of image rows owned by `rank`; bands differ by at most one row."""
    base, rem = divmod(H, world)
    row0 = rank * base + min(rank, rem)
    return row0, row0 + base + (1 if rank < rem else 0)


def stereo_poses(pose, eye_distance: float = 0.065) -> np.ndarray:
    """Left and right eye of a stereoscopic pair (Fig. 5): the camera centre moved by
    -/+ eye_distance / 2 along the camera's x axis (right), same rotation.  float32 [2, 12]; render
    both in one r360_render_batch call."""
    m = np.asarray(pose, np.float64).reshape(3, 4)
    out = []
    for sgn in (-0.5, 0.5):
        e = m.copy()
        e[:, 3] = m[:, 3] + sgn * eye_distance * m[:, 0]
        out.append(e.astype(np.float32).reshape(12))
    return np.stack(out)


def render_sharded(render_rows, pose, W: int, H: int, rank: int, world: int, dist, full_rgb, full_depth):
    """Strong scaling of ONE frame: this rank renders its band of rows in place into the
    full-size frame (`render_rows(pose, W, H, row0, row1, out_rgb, out_depth)` = Scene.render_rows), then the bands
    are all-gathered so that every rank holds the whole image.  Rays are independent and the scene is replicated:
    the gather of the finished pixels is the only exchange.  Returns (row0, row1)."""
    r0, r1 = row_band(H, rank, world)
    render_rows(pose, W, H, r0, r1, full_rgb[r0:r1], full_depth[r0:r1])
    if world > 1:
        gather_rows_inplace(full_rgb, H, rank, world, dist)
        gather_rows_inplace(full_depth, H, rank, world, dist)
    return r0, r1


def gather_rows_inplace(full, H: int, rank: int, world: int, dist):
    """All-gather of row bands inside a full [H, ...] tensor whose band `row_band(H, rank, world)` this rank has
    filled.  Equal bands: one in-place all-gather (NCCL writes every peer's band at its place); ragged bands: the
    padded gather of gather_rows, copied back."""
    r0, r1 = row_band(H, rank, world)
    if H % world == 0:
        dist.all_gather_into_tensor(full, full[r0:r1])
    else:
        full.copy_(gather_rows(full[r0:r1], H, rank, world, dist))
    return full


def gather_rows(band, H: int, rank: int, world: int, dist=None):
    """All-gather row bands (torch tensors [rows, ...]) into the full [H, ...] image on every rank."""
    import torch
    if world == 1:
        return band
    base, rem = divmod(H, world)
    pad_rows = base + (1 if rem else 0)
    padded = torch.zeros((pad_rows,) + tuple(band.shape[1:]), dtype=band.dtype, device=band.device)
    padded[:band.shape[0]] = band
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded)
    out = []
    for r in range(world):
        r0, r1 = row_band(H, r, world)
        out.append(parts[r][:r1 - r0])
    return torch.cat(out, 0)
