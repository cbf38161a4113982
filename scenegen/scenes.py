"""The five synthetic scenes of BASELINE.json (seed = config index - 1).

Generator rules (restated in DESIGN.md "Input recipe"):

* grid ``occupancy[(iz*Ny+iy)*Nx+ix]`` uint8.  Occupied voxels carry a quantised
  probability in [248,255], empty ones in [0,40]; ``occ_threshold`` = 248
  (0.97*255, the paper's occupancy threshold).
* shell  = every voxel with an index on the grid boundary.
* rooms  = interior walls 1 voxel thick, full height, on a ``rx x ry`` room grid;
  every wall segment shared by two rooms gets one door gap 0.9 m x 2.1 m at a
  seeded offset.
* boxes  = axis-aligned boxes; footprint U(0.3,1.5) m, height U(0.3,2.0) m,
  resting on the floor, hollow (1-voxel surface; boxes are drawn in order, a later
  box's hollow interior clears whatever an earlier one put there) (config 5: solid,
  footprint U(0.5,1.5), height U(0.3,1.0), floating anywhere).
* labels = recursive kd-split of the occupied voxels (BASELINE.json's stand-in
  for Algorithm 1 stage II): split on the longest metric
  bounding-box axis (ties: lowest axis) of the voxels sorted by (coordinate,
  linear index); leaf budget split floor(m/2):ceil(m/2); voxels cut in the
  same proportion (config 5: in proportion to summed Pareto(1.2) leaf weights).
* weights = Xavier-uniform per layer, biases 0 except the density bias.
* poses  = camera->world [R|o], row-major 3x4 float32.
"""
from dataclasses import dataclass, field
import math

import numpy as np

from .rng import SplitMix64

OCC_THRESHOLD = 248

# name -> parameters.  `rooms` = (rx, ry) room grid or None; `n_boxes`; `n` = subfields.
CONFIGS = {
    1: dict(name="smoke", W=64, H=32, n_poses=1, dims=(32, 32, 12),
            box_min=(-4.0, -4.0, -1.5), box_max=(4.0, 4.0, 1.5), rooms=None, n_boxes=3,
            n=16, width=32, n_hidden=2, K=8, sigma_bias=1.0, pareto=False, clutter=False,
            pose="centre"),
    2: dict(name="room", W=512, H=256, n_poses=1, dims=(128, 128, 48),
            box_min=(-4.0, -4.0, -1.5), box_max=(4.0, 4.0, 1.5), rooms=None, n_boxes=12,
            n=256, width=32, n_hidden=3, K=8, sigma_bias=1.0, pareto=False, clutter=False,
            pose="free"),
    3: dict(name="floor", W=2048, H=1024, n_poses=1, dims=(256, 256, 96),
            box_min=(-8.0, -8.0, -1.5), box_max=(8.0, 8.0, 1.5), rooms=(3, 2), n_boxes=40,
            n=1024, width=32, n_hidden=3, K=8, sigma_bias=1.0, pareto=False, clutter=False,
            pose="free", max_leaf=1500),
    4: dict(name="roaming", W=4096, H=2048, n_poses=8, dims=(512, 512, 96),
            box_min=(-16.0, -16.0, -1.5), box_max=(16.0, 16.0, 1.5), rooms=(4, 3), n_boxes=80,
            n=4096, width=64, n_hidden=3, K=12, sigma_bias=1.0, pareto=False, clutter=False,
            pose="path"),
    5: dict(name="imbalance", W=2048, H=1024, n_poses=1, dims=(256, 256, 96),
            box_min=(-8.0, -8.0, -1.5), box_max=(8.0, 8.0, 1.5), rooms=None, n_boxes=400,
            n=2048, width=32, n_hidden=3, K=8, sigma_bias=-2.0, pareto=True, clutter=True,
            pose="free"),
}

# stream ids of the PRNG, one per purpose, so that draw counts do not couple
_S_OCCVAL, _S_DOORS, _S_BOXES, _S_POSE, _S_PARETO, _S_WEIGHTS = range(6)


def weight_layout(width: int, n_hidden: int, pe_pos_levels: int = 10, pe_dir_levels: int = 4):
    """Blob order per subfield: list of (name, fan_out, fan_in).  Each layer is
    stored as W[out][in] row-major followed by b[out] (include/r360.h)."""
    pe_p = 3 + 6 * pe_pos_levels
    pe_d = 3 + 6 * pe_dir_levels
    layers = [("trunk1", width, pe_p)]
    for i in range(2, n_hidden + 1):
        layers.append((f"trunk{i}", width, width))
    layers.append(("density", 1, width))
    layers.append(("feature", width, width))
    layers.append(("colour", width, width + pe_d))
    layers.append(("rgb", 3, width))
    return layers


def mlp_param_count(width: int, n_hidden: int, pe_pos_levels: int = 10, pe_dir_levels: int = 4) -> int:
    return sum(o * i + o for _, o, i in weight_layout(width, n_hidden, pe_pos_levels, pe_dir_levels))


@dataclass
class Scene:
    config: int
    name: str
    W: int
    H: int
    dims: tuple
    box_min: tuple
    box_max: tuple
    n_subfields: int
    hidden_width: int
    n_hidden: int
    pe_pos_levels: int
    pe_dir_levels: int
    samples_per_voxel: int
    t_threshold: float
    density_activation: int
    occ_threshold: int
    occupancy: np.ndarray = field(repr=False)      # uint8 [N]
    voxel_subfield: np.ndarray = field(repr=False)  # int32 [N], -1 where empty
    weights: np.ndarray = field(repr=False)         # float32 [n*P]
    poses: np.ndarray = field(repr=False)           # float32 [B,12]

    @property
    def n_voxels(self):
        return int(self.dims[0] * self.dims[1] * self.dims[2])

    @property
    def params_per_subfield(self):
        return mlp_param_count(self.hidden_width, self.n_hidden, self.pe_pos_levels, self.pe_dir_levels)

    def occupied_mask(self):
        return self.occupancy >= self.occ_threshold


# --------------------------------------------------------------------------- geometry

def _build_occupied(cfg, seed):
    nx, ny, nz = cfg["dims"]
    bmin = np.array(cfg["box_min"], dtype=np.float64)
    bmax = np.array(cfg["box_max"], dtype=np.float64)
    vs = (bmax - bmin) / np.array([nx, ny, nz], dtype=np.float64)
    occ = np.zeros((nz, ny, nx), dtype=bool)
    # shell
    occ[0, :, :] = occ[-1, :, :] = True
    occ[:, 0, :] = occ[:, -1, :] = True
    occ[:, :, 0] = occ[:, :, -1] = True
    # interior walls with door gaps
    if cfg["rooms"] is not None:
        rx, ry = cfg["rooms"]
        rng = SplitMix64(seed, _S_DOORS)
        xs = [0] + [int(round(nx * i / rx)) for i in range(1, rx)] + [nx - 1]
        ys = [0] + [int(round(ny * i / ry)) for i in range(1, ry)] + [ny - 1]
        gap_z = int(math.ceil(2.1 / vs[2]))
        for i in range(1, rx):                       # walls normal to x
            occ[:, :, xs[i]] = True
        for j in range(1, ry):                       # walls normal to y
            occ[:, ys[j], :] = True
        for i in range(1, rx):
            gap = int(math.ceil(0.9 / vs[1]))
            for j in range(ry):                      # segment between rooms (i-1,j),(i,j)
                lo, hi = ys[j] + 1, ys[j + 1] - gap
                a = rng.randint(lo, max(lo + 1, hi))
                occ[1:1 + gap_z, a:a + gap, xs[i]] = False
        for j in range(1, ry):
            gap = int(math.ceil(0.9 / vs[0]))
            for i in range(rx):
                lo, hi = xs[i] + 1, xs[i + 1] - gap
                a = rng.randint(lo, max(lo + 1, hi))
                occ[1:1 + gap_z, ys[j], a:a + gap] = False
    # boxes
    rng = SplitMix64(seed, _S_BOXES)
    for _ in range(cfg["n_boxes"]):
        u = rng.uniform(6)
        if cfg["clutter"]:
            fx, fy = 0.5 + u[0] * 1.0, 0.5 + u[1] * 1.0
            hz = 0.3 + u[2] * 0.7
        else:
            fx, fy = 0.3 + u[0] * 1.2, 0.3 + u[1] * 1.2
            hz = 0.3 + u[2] * 1.7
        ex = max(1, int(round(fx / vs[0])))
        ey = max(1, int(round(fy / vs[1])))
        ez = max(1, int(round(hz / vs[2])))
        ex, ey, ez = min(ex, nx - 2), min(ey, ny - 2), min(ez, nz - 2)
        x0 = 1 + int(u[3] * (nx - 1 - ex))
        y0 = 1 + int(u[4] * (ny - 1 - ey))
        z0 = 1 + int(u[5] * (nz - 1 - ez)) if cfg["clutter"] else 1
        occ[z0:z0 + ez, y0:y0 + ey, x0:x0 + ex] = True
        if not cfg["clutter"] and ex > 2 and ey > 2 and ez > 2:
            # configs 1-4: 1-voxel-thick surface only (an occupancy map fused from
            # depth maps sees surfaces); keeps occupancy near the
            # "about 5-6 %" BASELINE.json states.  Config 5's clutter boxes are solid.
            occ[z0 + 1:z0 + ez - 1, y0 + 1:y0 + ey - 1, x0 + 1:x0 + ex - 1] = False
    return occ, vs


def _free_position(occ, cfg, vs, rng, fixed_xy=None):
    """Camera position with z in [-0.5,0] and >= 2 voxels of clearance."""
    nz, ny, nx = occ.shape
    bmin = np.array(cfg["box_min"], dtype=np.float64)
    bmax = np.array(cfg["box_max"], dtype=np.float64)
    for _ in range(100000):
        u = rng.uniform(3)
        p = np.array([bmin[0] + u[0] * (bmax[0] - bmin[0]),
                      bmin[1] + u[1] * (bmax[1] - bmin[1]),
                      -0.5 + 0.5 * u[2]])
        if _is_free(occ, p, bmin, vs):
            return p
    raise RuntimeError("no free camera position found")


def _is_free(occ, p, bmin, vs):
    nz, ny, nx = occ.shape
    c = np.floor((p - bmin) / vs).astype(int)
    if not (2 <= c[0] < nx - 2 and 2 <= c[1] < ny - 2 and 2 <= c[2] < nz - 2):
        return False
    return not occ[c[2] - 2:c[2] + 3, c[1] - 2:c[1] + 3, c[0] - 2:c[0] + 3].any()


def _pose(yaw, o):
    """Gravity-aligned camera->world pose.  R = Rz(yaw) * R0, R0 maps camera
    (x right, y down, z forward) to world (-y, -z, +x) (world z up)."""
    c, s = math.cos(yaw), math.sin(yaw)
    rz = np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])
    r0 = np.array([[0.0, 0.0, 1.0], [-1.0, 0.0, 0.0], [0.0, -1.0, 0.0]])
    r = rz @ r0
    m = np.concatenate([r, np.asarray(o, dtype=np.float64).reshape(3, 1)], axis=1)
    return m.astype(np.float32).reshape(12)


def _build_poses(occ, cfg, vs, seed):
    rng = SplitMix64(seed, _S_POSE)
    bmin = np.array(cfg["box_min"], dtype=np.float64)
    if cfg["pose"] == "centre":
        m = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)
        c = 0.5 * (np.array(cfg["box_min"]) + np.array(cfg["box_max"]))
        m[:, 3] = c
        return m.astype(np.float32).reshape(1, 12)
    if cfg["pose"] == "free":
        p = _free_position(occ, cfg, vs, rng)
        yaw = rng.uniform1() * 2.0 * math.pi
        return _pose(yaw, p).reshape(1, 12)
    # path: consecutive poses 0.25 m apart, heading re-drawn when blocked
    poses = []
    for _attempt in range(1000):
        poses = []
        p = _free_position(occ, cfg, vs, rng)
        heading = rng.uniform1() * 2.0 * math.pi
        ok = True
        for _k in range(cfg["n_poses"]):
            poses.append(_pose(heading, p))
            moved = False
            for _try in range(64):
                q = p + 0.25 * np.array([math.cos(heading), math.sin(heading), 0.0])
                if _is_free(occ, q, bmin, vs):
                    p = q
                    moved = True
                    break
                heading = rng.uniform1() * 2.0 * math.pi
            if not moved:
                ok = False
                break
        if ok:
            break
    return np.stack(poses).astype(np.float32)


# --------------------------------------------------------------------------- kd-split

def _kd_split(occ, vs, n_leaves, leaf_weights=None):
    """Labels in [0,n_leaves) for the occupied voxels, -1 elsewhere (int32 [N])."""
    nz, ny, nx = occ.shape
    lin = np.flatnonzero(occ.reshape(-1)).astype(np.int64)
    ix = (lin % nx).astype(np.int32)
    iy = ((lin // nx) % ny).astype(np.int32)
    iz = (lin // (nx * ny)).astype(np.int32)
    coords = np.stack([ix, iy, iz], axis=1)
    if n_leaves > lin.size:
        raise ValueError("more subfields than occupied voxels")
    if leaf_weights is None:
        leaf_weights = np.ones(n_leaves, dtype=np.float64)
    cum = np.concatenate([[0.0], np.cumsum(leaf_weights)])
    labels = np.full(nz * ny * nx, -1, dtype=np.int32)
    stack = [(np.arange(lin.size), 0, n_leaves)]
    while stack:
        sel, l0, l1 = stack.pop()
        nl = l1 - l0
        if nl == 1:
            labels[lin[sel]] = l0
            continue
        c = coords[sel]
        ext = (c.max(axis=0) - c.min(axis=0) + 1).astype(np.float64) * vs
        axis = int(np.argmax(ext))                    # ties -> lowest axis
        order = np.lexsort((lin[sel], c[:, axis]))
        sel = sel[order]
        ll = nl // 2
        lr = nl - ll
        wl = cum[l0 + ll] - cum[l0]
        wt = cum[l1] - cum[l0]
        m = sel.size
        ml = int(math.floor(m * (wl / wt)))
        ml = min(max(ml, ll), m - lr)
        stack.append((sel[ml:], l0 + ll, l1))
        stack.append((sel[:ml], l0, l0 + ll))
    return labels


# --------------------------------------------------------------------------- weights

def _build_weights(cfg, seed, n):
    width, n_hidden = cfg["width"], cfg["n_hidden"]
    layers = weight_layout(width, n_hidden)
    scale = []
    shift = []
    for name, fo, fi in layers:
        a = np.float32(math.sqrt(6.0 / (fi + fo)))
        scale.append(np.full(fo * fi, a, dtype=np.float32))
        scale.append(np.zeros(fo, dtype=np.float32))
        shift.append(np.zeros(fo * fi, dtype=np.float32))
        b = np.zeros(fo, dtype=np.float32)
        if name == "density":
            b[:] = np.float32(cfg["sigma_bias"])
        shift.append(b)
    scale = np.concatenate(scale)
    shift = np.concatenate(shift)
    P = scale.size
    rng = SplitMix64(seed, _S_WEIGHTS)
    out = np.empty(n * P, dtype=np.float32)
    chunk = max(1, (1 << 24) // P)
    for k0 in range(0, n, chunk):
        k1 = min(n, k0 + chunk)
        u = rng.uniform((k1 - k0) * P).astype(np.float32).reshape(k1 - k0, P)
        w = (np.float32(2.0) * u - np.float32(1.0)) * scale[None, :] + shift[None, :]
        out[k0 * P:k1 * P] = w.reshape(-1)
    return out


# --------------------------------------------------------------------------- entry

def make_scene(config: int, with_weights: bool = True) -> Scene:
    cfg = CONFIGS[config]
    seed = config - 1
    occ, vs = _build_occupied(cfg, seed)
    n = cfg["n"]
    lw = None
    if cfg["pareto"]:
        u = SplitMix64(seed, _S_PARETO).uniform(n)
        lw = (1.0 - u) ** (-1.0 / 1.2)
    labels = _kd_split(occ, vs, n, lw)
    if "max_leaf" in cfg:
        assert np.bincount(labels[labels >= 0]).max() <= cfg["max_leaf"]
    # quantised occupancy probabilities
    r = SplitMix64(seed, _S_OCCVAL).bits(occ.size)
    flat = occ.reshape(-1)
    val = np.where(flat, OCC_THRESHOLD + (r % np.uint64(8)), r % np.uint64(41)).astype(np.uint8)
    poses = _build_poses(occ, cfg, vs, seed)
    if with_weights:
        weights = _build_weights(cfg, seed, n)
    else:
        weights = np.zeros(0, dtype=np.float32)
    return Scene(config=config, name=cfg["name"], W=cfg["W"], H=cfg["H"], dims=tuple(cfg["dims"]),
                 box_min=tuple(cfg["box_min"]), box_max=tuple(cfg["box_max"]), n_subfields=n,
                 hidden_width=cfg["width"], n_hidden=cfg["n_hidden"], pe_pos_levels=10, pe_dir_levels=4,
                 samples_per_voxel=cfg["K"], t_threshold=1e-3, density_activation=1,
                 occ_threshold=OCC_THRESHOLD, occupancy=val, voxel_subfield=labels, weights=weights,
                 poses=poses)


# --------------------------------------------------------------------------- parity-test scene (not a BASELINE.json config)

def make_nondyadic_scene(seed: int = 100, K: int = 5, n: int = 7, occupancy_fraction: float = 0.12,
                         W: int = 96, H: int = 48) -> Scene:
    """Non-dyadic, anisotropic test scene: box [-1.3, 2.07] x [0.2, 3.9] x [-0.7, 1.13], grid 37 x 29 x 11
    (voxel sizes 0.0911 / 0.1276 / 0.1664 m, none a power of two, box_min not representable in binary32), random
    scattered occupancy (no shell: many rays leave the grid through empty space), kd-split labels, Xavier
    weights, a camera that sits on no lattice plane with a general (not gravity-aligned) rotation, and K = 5
    (not a power of two).  The BASELINE.json configs all have power-of-two voxel sizes and exactly
    representable planes, which would hide a contracted or reordered plane formula in a walk; this one does not.
    Pose 0: camera in free space; pose 1: camera inside an occupied voxel; pose 2: camera outside the box."""
    dims = (37, 29, 11)
    box_min, box_max = (-1.3, 0.2, -0.7), (2.07, 3.9, 1.13)
    nx, ny, nz = dims
    vs = (np.array(box_max) - np.array(box_min)) / np.array(dims, dtype=np.float64)
    rng = SplitMix64(seed, _S_BOXES)
    occ = (rng.uniform(nx * ny * nz) < occupancy_fraction).reshape(nz, ny, nx)
    # a few solid blobs so that rays cross runs of adjacent occupied voxels as well as isolated ones
    for _ in range(6):
        u = rng.uniform(6)
        e = 1 + (u[:3] * np.array([6, 5, 3])).astype(int)
        x0, y0, z0 = (u[3:] * (np.array(dims) - e)).astype(int)
        occ[z0:z0 + e[2], y0:y0 + e[1], x0:x0 + e[0]] = True
    labels = _kd_split(occ, vs, n)
    r = SplitMix64(seed, _S_OCCVAL).bits(occ.size)
    val = np.where(occ.reshape(-1), OCC_THRESHOLD + (r % np.uint64(8)), r % np.uint64(41)).astype(np.uint8)
    cfg = dict(width=32, n_hidden=2, sigma_bias=1.0)
    weights = _build_weights(cfg, seed, n)
    # general rotation from a seeded unit quaternion
    pr = SplitMix64(seed, _S_POSE)
    q = pr.uniform(4) * 2.0 - 1.0
    q /= np.linalg.norm(q)
    a, b, c, d = q
    R = np.array([[a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)],
                  [2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)],
                  [2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d]])
    flat = occ.reshape(-1)
    free = np.flatnonzero(~flat)
    full = np.flatnonzero(flat)

    def centre_of(lin, frac):
        idx = np.array([lin % nx, (lin // nx) % ny, lin // (nx * ny)], dtype=np.float64)
        return np.array(box_min) + (idx + frac) * vs

    o_free = centre_of(int(free[int(pr.uniform1() * free.size)]), np.array([0.37, 0.61, 0.43]))
    o_occ = centre_of(int(full[int(pr.uniform1() * full.size)]), np.array([0.53, 0.29, 0.71]))
    o_out = np.array([box_min[0] - 0.77, box_max[1] + 0.31, 0.5 * (box_min[2] + box_max[2]) + 0.113])
    poses = np.stack([np.concatenate([R, o.reshape(3, 1)], axis=1).astype(np.float32).reshape(12)
                      for o in (o_free, o_occ, o_out)])
    return Scene(config=0, name="nondyadic", W=W, H=H, dims=dims, box_min=box_min, box_max=box_max, n_subfields=n,
                 hidden_width=32, n_hidden=2, pe_pos_levels=10, pe_dir_levels=4, samples_per_voxel=K,
                 t_threshold=1e-3, density_activation=1, occ_threshold=OCC_THRESHOLD, occupancy=val,
                 voxel_subfield=labels, weights=weights, poses=poses)
