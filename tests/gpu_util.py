"""Helpers of the -m gpu parity tests: compare the CUDA path (through the C ABI binding) with the oracle."""
import numpy as np

from scenegen import weight_layout


def with_density_bias(sc, bias):
    """Copy of a scenegen scene's weights with the density bias replaced (data only)."""
    w = sc.weights.copy().reshape(sc.n_subfields, -1)
    o = 0
    for name, fo, fi in weight_layout(sc.hidden_width, sc.n_hidden, sc.pe_pos_levels, sc.pe_dir_levels):
        if name == "density":
            w[:, o + fo * fi] = bias
        o += fo * fi + fo
    return w.reshape(-1)


# Threshold-ambiguity band of a render mode (reading G4): the stopping sample depends on T = exp(-sum sigma delta),
# and |dT / T| <= ln(1 / tau) * max relative error of sigma = 6.9 * eps at the threshold tau = 1e-3.
#   fp32  : the kernel's binary32 field against the oracle's binary64, eps ~ 1e-6 -> the 1e-3 of reading G4
#   bf16  : eps <= 9.2e-3 / 1.3 = 7e-3 (largest raw-sigma error of tests/test_rounding_budget.py at the smallest
#           density the scenes have, softplus(1) = 1.3) -> 0.049, rounded up to 0.06
#   f16   : eps <= 1.5e-3 / 1.3 -> 0.008, rounded up to 0.02
AMB_BAND = {"fp32": 1e-3, "bf16": 0.06, "f16": 0.02}


def check_image(gpu_rgb, gpu_depth, ref, tol, amb_band=1e-3, depth_tol=None):
    """Element-by-element comparison with the oracle's outputs for the same pixels.

    Unambiguous rays: |gpu - oracle| <= tol.  Threshold-ambiguous rays (oracle's
    min_i |T_i - tau|/tau < amb_band, reading G4): any stopping point is valid, so the GPU
    value must lie between the stopped and the continued oracle results (C and D only grow).
    Returns (max_err_rgb, max_err_depth, n_ambiguous)."""
    depth_tol = tol if depth_tol is None else depth_tol
    g_rgb = np.asarray(gpu_rgb, np.float64).reshape(-1, 3)
    g_d = np.asarray(gpu_depth, np.float64).reshape(-1)
    amb = ref["ambiguity"] < amb_band
    e_rgb = np.abs(g_rgb - ref["rgb"])
    e_d = np.abs(g_d - ref["depth"])
    ok = ~amb
    max_rgb = float(e_rgb[ok].max()) if ok.any() else 0.0
    max_d = float(e_d[ok].max()) if ok.any() else 0.0
    assert max_rgb <= tol, f"rgb error {max_rgb:.3e} > {tol}"
    assert max_d <= depth_tol, f"depth error {max_d:.3e} > {depth_tol}"
    if amb.any():
        lo, hi = ref["rgb"][amb] - tol, ref["rgb_full"][amb] + tol
        assert np.all((g_rgb[amb] >= lo) & (g_rgb[amb] <= hi))
        assert np.all((g_d[amb] >= ref["depth"][amb] - depth_tol) & (g_d[amb] <= ref["depth_full"][amb] + depth_tol))
    return max_rgb, max_d, int(amb.sum())


def ray_major_index(counts, offsets):
    """Gather index that lists every ray's samples, rays in ray-major order.

    The order of the rays inside the sample buffers is free (the bit-exact
    contract covers, per ray, the count and the sequence of (t, subfield)); what must hold is that the
    per-ray ranges [offset, offset + count) are disjoint and cover [0, total).  Returns the index and
    checks exactly that."""
    counts = np.asarray(counts, np.int64).reshape(-1)
    offsets = np.asarray(offsets, np.int64).reshape(-1)
    total = int(counts.sum())
    first = np.repeat(np.cumsum(counts) - counts, counts)       # ray-major start of each sample's ray
    idx = np.repeat(offsets, counts) + (np.arange(total, dtype=np.int64) - first)
    assert np.array_equal(np.sort(idx), np.arange(total, dtype=np.int64)), "per-ray ranges overlap or leave gaps"
    return idx
