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
