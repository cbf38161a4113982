"""ctypes binding of libr360.so: same names as include/r360.h, marshalling only."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "csrc", "libr360.so")

STATUS = {0: "R360_OK", 1: "R360_ERR_INVALID_ARG", 2: "R360_ERR_BAD_LABEL", 3: "R360_ERR_NONFINITE",
          4: "R360_ERR_CUDA", 5: "R360_ERR_OOM", 6: "R360_ERR_CAPACITY"}


class R360Error(RuntimeError):
    def __init__(self, status, where, detail=""):
        self.status = int(status)
        super().__init__(f"{where}: {STATUS.get(self.status, self.status)} {detail}".strip())


class Desc(C.Structure):
    _fields_ = [("dims", C.c_int32 * 3), ("box_min", C.c_float * 3), ("box_max", C.c_float * 3),
                ("n_subfields", C.c_int32), ("hidden_width", C.c_int32), ("n_hidden", C.c_int32),
                ("pe_pos_levels", C.c_int32), ("pe_dir_levels", C.c_int32),
                ("samples_per_voxel", C.c_int32), ("t_threshold", C.c_float),
                ("density_activation", C.c_int32), ("occ_threshold", C.c_uint8)]


class Stats(C.Structure):
    _fields_ = [("rays", C.c_uint64), ("segments", C.c_uint64), ("samples_emitted", C.c_uint64),
                ("samples_used", C.c_uint64), ("mlp_tiles", C.c_uint64), ("chunks", C.c_uint32),
                ("kernel_launches", C.c_uint32), ("ms_count", C.c_float), ("ms_scan", C.c_float),
                ("ms_emit", C.c_float), ("ms_mlp", C.c_float), ("ms_composite", C.c_float),
                ("ms_total", C.c_float), ("retries", C.c_uint32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_LIB = None


def lib_path():
    return _SO


def lib():
    """Load libr360.so (built in-tree by paper_2208_02705_b200.build / __graft_entry__.build)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    L = C.CDLL(_SO)
    vp, i32, f32p = C.c_void_p, C.c_int32, C.POINTER(C.c_float)
    L.r360_params_per_subfield.restype = C.c_int64
    L.r360_params_per_subfield.argtypes = [C.POINTER(Desc)]
    L.r360_scene_create.restype = C.c_int
    L.r360_scene_create.argtypes = [C.POINTER(Desc), vp, vp, vp, C.POINTER(vp)]
    L.r360_scene_destroy.restype = None
    L.r360_scene_destroy.argtypes = [vp]
    L.r360_render.restype = C.c_int
    L.r360_render.argtypes = [vp, f32p, i32, i32, vp, vp]
    L.r360_render_batch.restype = C.c_int
    L.r360_render_batch.argtypes = [vp, f32p, i32, i32, i32, vp, vp]
    L.r360_render_batch_host.restype = C.c_int
    L.r360_render_batch_host.argtypes = [vp, f32p, i32, i32, i32, vp, vp]
    L.r360_render_batch_host_async.restype = C.c_int
    L.r360_render_batch_host_async.argtypes = [vp, f32p, i32, i32, i32, vp, vp]
    L.r360_host_sync.restype = C.c_int
    L.r360_host_sync.argtypes = [vp]
    L.r360_render_rows.restype = C.c_int
    L.r360_render_rows.argtypes = [vp, f32p, i32, i32, i32, i32, vp, vp]
    for name in ("r360_wait", "r360_graph_status"):
        getattr(L, name).restype = C.c_int
        getattr(L, name).argtypes = [vp]
    for name in ("r360_set_output_format", "r360_set_host_bands"):
        getattr(L, name).restype = C.c_int
        getattr(L, name).argtypes = [vp, i32]
    L.r360_reserve.restype = C.c_int
    L.r360_reserve.argtypes = [vp, C.c_uint64, C.c_double]
    L.r360_set_graph_poses.restype = C.c_int
    L.r360_set_graph_poses.argtypes = [vp, f32p, i32]
    L.r360_set_precision.restype = C.c_int
    L.r360_set_precision.argtypes = [vp, i32]
    L.r360_assign_subfields.restype = C.c_int
    L.r360_assign_subfields.argtypes = [C.POINTER(C.c_int32), f32p, f32p, C.POINTER(C.c_uint8), C.c_uint8, i32,
                                        C.POINTER(C.c_int32)]
    L.r360_occupancy_fuse.restype = C.c_int
    L.r360_occupancy_fuse.argtypes = [C.POINTER(C.c_int32), f32p, f32p, f32p, f32p, i32, i32, f32p, f32p]
    L.r360_fusion_create.restype = C.c_int
    L.r360_fusion_create.argtypes = [C.POINTER(C.c_int32), f32p, f32p, f32p, C.POINTER(vp)]
    L.r360_fusion_fuse.restype = C.c_int
    L.r360_fusion_fuse.argtypes = [vp, f32p, i32, i32, f32p, f32p]
    L.r360_fusion_fuse_device.restype = C.c_int
    L.r360_fusion_fuse_device.argtypes = [vp, f32p, i32, i32, vp, vp]
    L.r360_fusion_read.restype = C.c_int
    L.r360_fusion_read.argtypes = [vp, f32p, C.POINTER(C.c_uint8)]
    L.r360_fusion_destroy.restype = None
    L.r360_fusion_destroy.argtypes = [vp]
    L.r360_floorplan.restype = C.c_int
    L.r360_floorplan.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_uint8), C.c_uint8, i32, i32, f32p, f32p,
                                 C.POINTER(C.c_uint8)]
    L.r360_set_wavefront.restype = C.c_int
    L.r360_set_wavefront.argtypes = [vp, i32]
    L.r360_set_camera.restype = C.c_int
    L.r360_set_camera.argtypes = [vp, i32, C.c_double, C.c_double, C.c_double, C.c_double]
    L.r360_set_stream.restype = C.c_int
    L.r360_set_stream.argtypes = [vp, vp]
    L.r360_set_chunk_rays.restype = C.c_int
    L.r360_set_chunk_rays.argtypes = [vp, C.c_int64]
    L.r360_get_stats.restype = C.c_int
    L.r360_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.r360_debug_samples.restype = C.c_int
    L.r360_debug_samples.argtypes = [vp, f32p, i32, i32, vp, vp, vp, vp, C.c_uint64, C.POINTER(C.c_uint64)]
    L.r360_debug_field.restype = C.c_int
    L.r360_debug_field.argtypes = [vp, f32p, i32, i32, vp, vp, vp, vp, vp, C.c_uint64, C.POINTER(C.c_uint64)]
    L.r360_status_string.restype = C.c_char_p
    L.r360_status_string.argtypes = [C.c_int]
    L.r360_last_cuda_error.restype = C.c_char_p
    L.r360_version.restype = C.c_char_p
    _LIB = L
    return L


def version():
    return lib().r360_version().decode()


def measure_fp32_fma():
    """(TFLOP/s, nominal SM MHz) of the FP32 FMA pipes of the current device: bench.py's roofline of the fp32 MLP
    path.  Lives in libr360_bench.so (csrc/microbench.cu), a measurement helper outside the product ABI."""
    so = os.path.join(_HERE, "csrc", "libr360_bench.so")
    if not os.path.exists(so):
        raise ImportError(f"{so} is missing: run `python -c 'import __graft_entry__ as g; g.build()'`")
    fn = C.CDLL(so).r360bench_fp32_fma
    fn.restype = C.c_int
    fn.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
    tf, mhz = C.c_double(0), C.c_double(0)
    rc = fn(C.byref(tf), C.byref(mhz))
    if rc != 0:
        raise RuntimeError(f"r360bench_fp32_fma failed: cudaError_t {rc}")
    return tf.value, mhz.value


def _check(st, where):
    if st != 0:
        raise R360Error(st, where, lib().r360_last_cuda_error().decode() if st in (4, 5) else "")


def make_desc(dims, box_min, box_max, n_subfields, hidden_width=32, n_hidden=2, pe_pos_levels=10,
              pe_dir_levels=4, samples_per_voxel=8, t_threshold=1e-3, density_activation=1, occ_threshold=1):
    d = Desc()
    d.dims[:] = [int(x) for x in dims]
    d.box_min[:] = [float(x) for x in box_min]
    d.box_max[:] = [float(x) for x in box_max]
    d.n_subfields, d.hidden_width, d.n_hidden = int(n_subfields), int(hidden_width), int(n_hidden)
    d.pe_pos_levels, d.pe_dir_levels = int(pe_pos_levels), int(pe_dir_levels)
    d.samples_per_voxel, d.t_threshold = int(samples_per_voxel), float(t_threshold)
    d.density_activation, d.occ_threshold = int(density_activation), int(occ_threshold)
    return d


def params_per_subfield(**kw):
    kw.setdefault("dims", (1, 1, 1)); kw.setdefault("box_min", (0, 0, 0)); kw.setdefault("box_max", (1, 1, 1))
    kw.setdefault("n_subfields", 1)
    return int(lib().r360_params_per_subfield(C.byref(make_desc(**kw))))


def assign_subfields(occupancy, dims, box_min, box_max, occ_threshold, n):
    """Algorithm 1 stage II on the GPU (r360_assign_subfields): int32 labels[N], -1 for empty voxels."""
    occ = np.ascontiguousarray(occupancy, np.uint8).reshape(-1)
    d = (C.c_int32 * 3)(*[int(v) for v in dims])
    lo = (C.c_float * 3)(*[float(v) for v in box_min])
    hi = (C.c_float * 3)(*[float(v) for v in box_max])
    assert occ.size == d[0] * d[1] * d[2]
    out = np.empty(occ.size, np.int32)
    _check(lib().r360_assign_subfields(d, lo, hi, occ.ctypes.data_as(C.POINTER(C.c_uint8)), int(occ_threshold),
                                       int(n), out.ctypes.data_as(C.POINTER(C.c_int32))), "r360_assign_subfields")
    return out


def occupancy_fuse(logodds, dims, box_min, box_max, pose, W, H, depth, uncertainty=None):
    """One observation fused into the log-odds grid on the GPU (r360_occupancy_fuse); returns the new float32 grid."""
    d = (C.c_int32 * 3)(*[int(v) for v in dims])
    lo = (C.c_float * 3)(*[float(v) for v in box_min])
    hi = (C.c_float * 3)(*[float(v) for v in box_max])
    L = np.array(logodds, np.float32).reshape(-1).copy()
    assert L.size == d[0] * d[1] * d[2]
    fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
    p = np.ascontiguousarray(pose, np.float32).reshape(12)
    dep = np.ascontiguousarray(depth, np.float32).reshape(-1)
    assert dep.size == W * H
    unc = None if uncertainty is None else np.ascontiguousarray(uncertainty, np.float32).reshape(-1)
    _check(lib().r360_occupancy_fuse(d, lo, hi, fp(L), fp(p), W, H, fp(dep), None if unc is None else fp(unc)),
           "r360_occupancy_fuse")
    return L


class Fusion:
    """r360_fusion handle: the log-odds grid of Eq. 6 resident on the device between observations."""

    def __init__(self, dims, box_min, box_max, logodds_init=None):
        self._h = C.c_void_p()
        d = (C.c_int32 * 3)(*[int(v) for v in dims])
        lo = (C.c_float * 3)(*[float(v) for v in box_min])
        hi = (C.c_float * 3)(*[float(v) for v in box_max])
        self.N = d[0] * d[1] * d[2]
        init = None
        if logodds_init is not None:
            keep = np.ascontiguousarray(logodds_init, np.float32).reshape(-1)
            assert keep.size == self.N
            init = keep.ctypes.data_as(C.POINTER(C.c_float))
        _check(lib().r360_fusion_create(d, lo, hi, init, C.byref(self._h)), "r360_fusion_create")

    def fuse(self, pose, W, H, depth, uncertainty=None):
        """One observation; depth / uncertainty are numpy arrays (host) or torch CUDA float32 tensors (device)."""
        p = np.ascontiguousarray(pose, np.float32).reshape(12)
        pp = p.ctypes.data_as(C.POINTER(C.c_float))
        if hasattr(depth, "is_cuda"):
            assert depth.is_cuda and depth.is_contiguous() and depth.numel() == W * H
            u = None if uncertainty is None else uncertainty.data_ptr()
            _check(lib().r360_fusion_fuse_device(self._h, pp, W, H, depth.data_ptr(), u), "r360_fusion_fuse_device")
            return
        dep = np.ascontiguousarray(depth, np.float32).reshape(-1)
        assert dep.size == W * H
        unc = None if uncertainty is None else np.ascontiguousarray(uncertainty, np.float32).reshape(-1)
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        _check(lib().r360_fusion_fuse(self._h, pp, W, H, fp(dep), None if unc is None else fp(unc)), "r360_fusion_fuse")

    def read(self, occupancy=False):
        """The log-odds grid (float32[N]); with occupancy=True also the thresholded uint8 grid (255 / 0)."""
        L = np.empty(self.N, np.float32)
        occ = np.empty(self.N, np.uint8) if occupancy else None
        _check(lib().r360_fusion_read(self._h, L.ctypes.data_as(C.POINTER(C.c_float)),
                                      None if occ is None else occ.ctypes.data_as(C.POINTER(C.c_uint8))), "r360_fusion_read")
        return (L, occ) if occupancy else L

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().r360_fusion_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


STATIC_MAX_VOXELS, STATIC_MAX_W, STATIC_MAX_H = 8 << 20, 4096, 2048   # R360_STATIC_MAX_* of include/r360.h


def fusion_fuse_static(logodds, dims, box_min, box_max, pose, W, H, depth, uncertainty=None, stream=None):
    """One observation of Eq. 6 fused in place into `logodds` without any device allocation
    (r360_fusion_fuse_static).  For callers that cannot call cudaMalloc: a process whose own pool already holds the
    whole GPU, a frame loop that cannot take an allocation's device-wide stall, code running while allocation is
    forbidden.  The scratch is a static array inside libr360.so, which limits the problem to STATIC_MAX_VOXELS
    voxels and a STATIC_MAX_W x STATIC_MAX_H image.

    logodds: torch CUDA float32 tensor [Nx*Ny*Nz], updated in place; depth / uncertainty: torch CUDA float32 tensors
    of W*H elements; stream: a torch.cuda.Stream, a raw cudaStream_t as int, or None for the default stream.
    Asynchronous.  All calls on one device share the scratch: keep them on one stream (overlapping calls race).
    Make the first call on a device during set-up (it resolves the scratch's device address)."""
    fn = lib().r360_fusion_fuse_static
    if fn.argtypes is None:
        f32p = C.POINTER(C.c_float)
        fn.restype = C.c_int
        fn.argtypes = [C.POINTER(C.c_int32), f32p, f32p, C.c_void_p, f32p, C.c_int32, C.c_int32, C.c_void_p,
                       C.c_void_p, C.c_void_p]
    d = (C.c_int32 * 3)(*[int(v) for v in dims])
    lo = (C.c_float * 3)(*[float(v) for v in box_min])
    hi = (C.c_float * 3)(*[float(v) for v in box_max])
    N = d[0] * d[1] * d[2]
    for t, n in ((logodds, N), (depth, W * H)) + (() if uncertainty is None else ((uncertainty, W * H),)):
        assert t.is_cuda and t.is_contiguous() and t.numel() == n and t.element_size() == 4
    p = np.ascontiguousarray(pose, np.float32).reshape(12)
    s = None if stream is None else int(getattr(stream, "cuda_stream", stream))
    st = fn(d, lo, hi, logodds.data_ptr(), p.ctypes.data_as(C.POINTER(C.c_float)), int(W), int(H), depth.data_ptr(),
            None if uncertainty is None else uncertainty.data_ptr(), s)
    if st == 6:
        raise R360Error(st, "r360_fusion_fuse_static", lib().r360_last_cuda_error().decode())
    _check(st, "r360_fusion_fuse_static")


def floorplan(occupancy, dims, occ_threshold, seed_xy, upper=None, lower=None):
    """Floorplan from the occupancy map on the GPU (r360_floorplan): uint8 [Ny][Nx], bit 0 interior, bit 1 inner
    boundary, bit 2 obstacle."""
    occ = np.ascontiguousarray(occupancy, np.uint8).reshape(-1)
    d = (C.c_int32 * 3)(*[int(v) for v in dims])
    assert occ.size == d[0] * d[1] * d[2]
    up = (C.c_float * 2)(*upper) if upper is not None else None
    lo = (C.c_float * 2)(*lower) if lower is not None else None
    out = np.empty((d[1], d[0]), np.uint8)
    _check(lib().r360_floorplan(d, occ.ctypes.data_as(C.POINTER(C.c_uint8)), int(occ_threshold), int(seed_xy[0]),
                                int(seed_xy[1]), up, lo, out.ctypes.data_as(C.POINTER(C.c_uint8))), "r360_floorplan")
    return out


def _pose_ptr(poses, B):
    p = np.ascontiguousarray(poses, dtype=np.float32).reshape(B * 12)
    return p, p.ctypes.data_as(C.POINTER(C.c_float))


class Scene:
    """r360_scene handle.  Device outputs are torch CUDA tensors (torch = device memory only)."""

    def __init__(self, occupancy, voxel_subfield, weights, **desc_kw):
        self._h = C.c_void_p()
        self.desc = make_desc(**desc_kw)
        occ = np.ascontiguousarray(occupancy, dtype=np.uint8).reshape(-1)
        lab = np.ascontiguousarray(voxel_subfield, dtype=np.int32).reshape(-1)
        w = np.ascontiguousarray(weights, dtype=np.float32).reshape(-1)
        N = int(self.desc.dims[0]) * int(self.desc.dims[1]) * int(self.desc.dims[2])
        P = int(lib().r360_params_per_subfield(C.byref(self.desc)))
        if P and (occ.size != N or lab.size != N or w.size != P * int(self.desc.n_subfields)):
            raise R360Error(1, "r360_scene_create", "array sizes do not match the description")
        st = lib().r360_scene_create(C.byref(self.desc), occ.ctypes.data, lab.ctypes.data, w.ctypes.data,
                                     C.byref(self._h))
        _check(st, "r360_scene_create")
        self.K = int(self.desc.samples_per_voxel)

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().r360_scene_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_precision(self, mode):
        """"fp32" (FP32 ALUs), "bf16" (tensor cores, bfloat16 operands) or "f16" (tensor cores, binary16 operands)."""
        _check(lib().r360_set_precision(self._h, {"fp32": 0, "bf16": 1, "f16": 2}.get(mode, mode)), "r360_set_precision")

    def set_wavefront(self, mode):
        """False / 0 = single pass, True / 1 = wavefronted passes, "auto" / 2 = passes iff the last frame was opaque."""
        _check(lib().r360_set_wavefront(self._h, 2 if mode == "auto" else int(mode)), "r360_set_wavefront")

    def set_camera(self, model="equirect", fx=0.0, fy=0.0, cx=0.0, cy=0.0):
        _check(lib().r360_set_camera(self._h, {"equirect": 0, "pinhole": 1}.get(model, model), fx, fy, cx, cy),
               "r360_set_camera")

    def set_stream(self, cuda_stream_ptr):
        _check(lib().r360_set_stream(self._h, C.c_void_p(cuda_stream_ptr)), "r360_set_stream")

    def set_chunk_rays(self, n):
        _check(lib().r360_set_chunk_rays(self._h, int(n)), "r360_set_chunk_rays")

    def use_current_torch_stream(self):
        import torch
        self.set_stream(torch.cuda.current_stream().cuda_stream)

    def set_output_format(self, fmt):
        """"f32" (rgb float32 x 3 + depth float32, default) or "rgb8_d16" (rgb uint8 x 3 + depth float16)."""
        f = {"f32": 0, "rgb8_d16": 1}.get(fmt, fmt)
        _check(lib().r360_set_output_format(self._h, f), "r360_set_output_format")
        self._fmt = int(f)

    def set_host_bands(self, n):
        _check(lib().r360_set_host_bands(self._h, int(n)), "r360_set_host_bands")

    def reserve(self, max_rays_per_chunk, segments_per_ray):
        _check(lib().r360_reserve(self._h, int(max_rays_per_chunk), float(segments_per_ray)), "r360_reserve")

    def wait(self):
        """r360_wait: the outputs of the last render call are complete in stream order once this returns."""
        _check(lib().r360_wait(self._h), "r360_wait")

    def graph_status(self):
        _check(lib().r360_graph_status(self._h), "r360_graph_status")

    def set_graph_poses(self, poses):
        poses = np.asarray(poses, np.float32)
        keep, p = _pose_ptr(poses, poses.size // 12)
        _check(lib().r360_set_graph_poses(self._h, p, poses.size // 12), "r360_set_graph_poses")

    def _out_tensors(self, shape_px, out_rgb, out_depth):
        import torch
        fmt = getattr(self, "_fmt", 0)
        t_rgb, t_d = (torch.float32, torch.float32) if fmt == 0 else (torch.uint8, torch.float16)
        n = int(np.prod(shape_px))
        if out_rgb is None:
            out_rgb = torch.empty((*shape_px, 3), dtype=t_rgb, device="cuda")
        if out_depth is None:
            out_depth = torch.empty(tuple(shape_px), dtype=t_d, device="cuda")
        assert out_rgb.is_cuda and out_depth.is_cuda and out_rgb.is_contiguous() and out_depth.is_contiguous()
        assert out_rgb.dtype == t_rgb and out_depth.dtype == t_d
        assert out_rgb.numel() == n * 3 and out_depth.numel() == n
        return out_rgb, out_depth

    def render(self, pose, W, H, out_rgb=None, out_depth=None, wait=True):
        """r360_render (+ r360_wait unless wait=False: needed before the outputs are used by other stream work)."""
        out_rgb, out_depth = self._out_tensors((1, H, W), out_rgb, out_depth)
        keep, p = _pose_ptr(pose, 1)
        _check(lib().r360_render(self._h, p, W, H, out_rgb.data_ptr(), out_depth.data_ptr()), "r360_render")
        if wait:
            self.wait()
        return out_rgb.view(H, W, 3), out_depth.view(H, W)

    def render_batch(self, poses, W, H, out_rgb=None, out_depth=None, wait=True):
        poses = np.asarray(poses, np.float32)
        B = poses.size // 12
        out_rgb, out_depth = self._out_tensors((B, H, W), out_rgb, out_depth)
        keep, p = _pose_ptr(poses, B)
        st = lib().r360_render_batch(self._h, p, B, W, H, out_rgb.data_ptr(), out_depth.data_ptr())
        _check(st, "r360_render_batch")
        if wait:
            self.wait()
        return out_rgb, out_depth

    def render_rows(self, pose, W, H, row0, row1, out_rgb=None, out_depth=None, wait=True):
        """r360_render_rows: image rows [row0, row1) of one view into band-sized outputs [(row1-row0), W(, 3)]."""
        out_rgb, out_depth = self._out_tensors((row1 - row0, W), out_rgb, out_depth)
        keep, p = _pose_ptr(pose, 1)
        st = lib().r360_render_rows(self._h, p, W, H, row0, row1, out_rgb.data_ptr(), out_depth.data_ptr())
        _check(st, "r360_render_rows")
        if wait:
            self.wait()
        return out_rgb, out_depth

    def host_sync(self):
        _check(lib().r360_host_sync(self._h), "r360_host_sync")

    def render_batch_host(self, poses, W, H, out_rgb=None, out_depth=None, sync=True):
        """HOST buffers in and out (numpy, ideally pinned): the end-to-end call.  sync=False: the streaming form
        (r360_render_batch_host_async); the buffers hold the frame after host_sync()."""
        poses = np.asarray(poses, np.float32)
        B = poses.size // 12
        fmt = getattr(self, "_fmt", 0)
        t_rgb, t_d = (np.float32, np.float32) if fmt == 0 else (np.uint8, np.float16)
        if out_rgb is None:
            out_rgb = np.empty((B, H, W, 3), t_rgb)
        if out_depth is None:
            out_depth = np.empty((B, H, W), t_d)
        assert out_rgb.dtype == t_rgb and out_depth.dtype == t_d
        assert out_rgb.size == B * H * W * 3 and out_depth.size == B * H * W
        keep, p = _pose_ptr(poses, B)
        fn = lib().r360_render_batch_host if sync else lib().r360_render_batch_host_async
        _check(fn(self._h, p, B, W, H, out_rgb.ctypes.data, out_depth.ctypes.data), "r360_render_batch_host")
        return out_rgb, out_depth

    def stats(self):
        s = Stats()
        _check(lib().r360_get_stats(self._h, C.byref(s)), "r360_get_stats")
        return s

    def debug_samples(self, pose, W, H, cap=None):
        """(counts, offsets, t, subfield) as torch CUDA tensors; steps a1-a5 only."""
        import torch
        keep, p = _pose_ptr(pose, 1)
        counts = torch.empty(W * H, dtype=torch.int32, device="cuda")
        offsets = torch.empty(W * H, dtype=torch.int32, device="cuda")
        total = C.c_uint64(0)
        if cap is None:
            st = lib().r360_debug_samples(self._h, p, W, H, counts.data_ptr(), offsets.data_ptr(), None, None, 0,
                                          C.byref(total))
            if st not in (0, 6):
                _check(st, "r360_debug_samples")
            cap = int(total.value)
        t = torch.empty(max(cap, 1), dtype=torch.float32, device="cuda")
        sid = torch.empty(max(cap, 1), dtype=torch.int32, device="cuda")
        st = lib().r360_debug_samples(self._h, p, W, H, counts.data_ptr(), offsets.data_ptr(), t.data_ptr(),
                                      sid.data_ptr(), cap, C.byref(total))
        _check(st, "r360_debug_samples")
        n = int(total.value)
        return counts, offsets, t[:n], sid[:n]


def _debug_field(self, pose, W, H):
    """(counts, offsets, t, subfield, field[S, 4]) as torch CUDA tensors; steps a1-a9 (r360_debug_field)."""
    import torch
    counts, offsets, t, sid = self.debug_samples(pose, W, H)
    n = int(t.numel())
    field = torch.empty((max(n, 1), 4), dtype=torch.float32, device="cuda")
    keep, p = _pose_ptr(pose, 1)
    total = C.c_uint64(0)
    _check(lib().r360_debug_field(self._h, p, W, H, counts.data_ptr(), offsets.data_ptr(), t.data_ptr(), sid.data_ptr(),
                                  field.data_ptr(), max(n, 1), C.byref(total)), "r360_debug_field")
    assert int(total.value) == n
    return counts, offsets, t, sid, field[:n]


Scene.debug_field = _debug_field


def scene_from(sc, **override):
    """Scene from a scenegen.Scene (data only)."""
    kw = dict(dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max, n_subfields=sc.n_subfields,
              hidden_width=sc.hidden_width, n_hidden=sc.n_hidden, pe_pos_levels=sc.pe_pos_levels,
              pe_dir_levels=sc.pe_dir_levels, samples_per_voxel=sc.samples_per_voxel, t_threshold=sc.t_threshold,
              density_activation=sc.density_activation, occ_threshold=sc.occ_threshold)
    arrays = dict(occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield, weights=sc.weights)
    for k, v in override.items():
        (arrays if k in arrays else kw)[k] = v
    return Scene(**arrays, **kw)
