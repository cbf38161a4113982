"""ctypes binding of oracle/r360_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Marshalling only; all arithmetic is in the C file.  Shares nothing with
paper_2208_02705_b200/.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libr360_oracle.so")
_SRC = os.path.join(_HERE, "r360_oracle.c")
_HDR = os.path.join(_HERE, "r360_oracle.h")

CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
          "-Wall", "-Wextra"]


def build_oracle(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, no CUDA)."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _SO
    # R360_ORACLE_CFLAGS: extra flags, e.g. "-fsanitize=address,undefined -g" for a sanitizer run of the CPU tests
    subprocess.check_call(["gcc", *CFLAGS, *os.environ.get("R360_ORACLE_CFLAGS", "").split(), "-o", _SO, _SRC, "-lm"])
    return _SO


class _Desc(C.Structure):
    _fields_ = [("dims", C.c_int32 * 3), ("box_min", C.c_float * 3), ("box_max", C.c_float * 3),
                ("n_subfields", C.c_int32), ("hidden_width", C.c_int32), ("n_hidden", C.c_int32),
                ("pe_pos_levels", C.c_int32), ("pe_dir_levels", C.c_int32),
                ("samples_per_voxel", C.c_int32), ("t_threshold", C.c_float),
                ("density_activation", C.c_int32), ("occ_threshold", C.c_int32)]


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


_F, _D, _I, _U, _B = C.c_float, C.c_double, C.c_int32, C.c_uint32, C.c_uint8
_PF, _PD, _PI, _PU = C.POINTER(_F), C.POINTER(_D), C.POINTER(_I), C.POINTER(_U)


class Oracle:
    def __init__(self, lib):
        self.lib = lib
        L = lib
        L.r360o_create.restype = C.c_void_p
        L.r360o_create.argtypes = [C.POINTER(_Desc), C.POINTER(_B), _PI, _PF]
        L.r360o_destroy.argtypes = [C.c_void_p]
        L.r360o_params_per_subfield.restype = C.c_int64
        L.r360o_params_per_subfield.argtypes = [C.POINTER(_Desc)]
        L.r360o_trig_tables.argtypes = [_I, _I, _PF, _PF, _PF, _PF]
        L.r360o_sphere_to_pixel.argtypes = [_D, _D, _I, _I, _PD, _PD]
        L.r360o_pixel_to_sphere.argtypes = [_I, _I, _I, _I, _PD, _PD]
        L.r360o_ray.argtypes = [_PF, _I, _I, _I, _I, _PF, _PF]
        L.r360o_walk.restype = C.c_int64
        L.r360o_walk.argtypes = [C.c_void_p, _PF, _PF, C.c_int, C.c_int64, _PI, _PF, _PF]
        L.r360o_clip.restype = C.c_int
        L.r360o_clip.argtypes = [C.c_void_p, _PF, _PF, _PF, _PF]
        L.r360o_ray_samples.restype = C.c_int64
        L.r360o_ray_samples.argtypes = [C.c_void_p, _PF, _I, _I, _I, _I, C.c_int64, _PF, _PF, _PI]
        L.r360o_subfield_frame.argtypes = [C.c_void_p, _I, _PF, _PF]
        L.r360o_pe.argtypes = [_PD, _I, _PD]
        L.r360o_field.argtypes = [C.c_void_p, _I, _PF, _PF, _PD]
        L.r360o_field_raw.argtypes = [C.c_void_p, _I, _PF, _PF, _PD]
        L.r360o_composite.argtypes = [C.c_int64, _PD, _PD, _PF, _PF, _D, _PD, _PD, _PD]
        L.r360o_render_pixels.restype = C.c_int
        L.r360o_render_pixels.argtypes = [C.c_void_p, _PF, _I, _I, C.c_int64, _PI, _PI,
                                          _PF, _PF, _PF, _PF, _PF, _PU, _PU]
        L.r360o_render_rows.restype = C.c_int
        L.r360o_render_rows.argtypes = [C.c_void_p, _PF, _I, _I, _I, _I, _PF, _PF, _PF, _PF, _PF, _PU, _PU]
        L.r360o_samples_rows.restype = C.c_int64
        L.r360o_samples_rows.argtypes = [C.c_void_p, _PF, _I, _I, _I, _I, _PU, C.c_int64, _PF, _PI]
        L.r360o_num_threads.restype = C.c_int
        L.r360o_ray_pinhole.argtypes = [_PF, _D, _D, _D, _D, _I, _I, _PF, _PF]
        L.r360o_pinhole_tables.argtypes = [_I, _I, _D, _D, _D, _D, _PF, _PF]
        L.r360o_set_camera.restype = C.c_int
        L.r360o_set_camera.argtypes = [C.c_void_p, _I, _D, _D, _D, _D]

    # ---- scene-independent taps
    def num_threads(self):
        return int(self.lib.r360o_num_threads())

    def trig_tables(self, W, H):
        sp, cp = np.empty(W, np.float32), np.empty(W, np.float32)
        st, ct = np.empty(H, np.float32), np.empty(H, np.float32)
        self.lib.r360o_trig_tables(W, H, _p(sp, _F), _p(cp, _F), _p(st, _F), _p(ct, _F))
        return sp, cp, st, ct

    def sphere_to_pixel(self, phi, theta, W, H):
        u, v = _D(), _D()
        self.lib.r360o_sphere_to_pixel(phi, theta, W, H, C.byref(u), C.byref(v))
        return u.value, v.value

    def pixel_to_sphere(self, i, j, W, H):
        a, b = _D(), _D()
        self.lib.r360o_pixel_to_sphere(i, j, W, H, C.byref(a), C.byref(b))
        return a.value, b.value

    def ray(self, pose, W, H, i, j):
        pose = np.ascontiguousarray(pose, np.float32).reshape(12)
        o, d = np.empty(3, np.float32), np.empty(3, np.float32)
        self.lib.r360o_ray(_p(pose, _F), W, H, i, j, _p(o, _F), _p(d, _F))
        return o, d

    def ray_pinhole(self, pose, fx, fy, cx, cy, i, j):
        pose = np.ascontiguousarray(pose, np.float32).reshape(12)
        o, d = np.empty(3, np.float32), np.empty(3, np.float32)
        self.lib.r360o_ray_pinhole(_p(pose, _F), fx, fy, cx, cy, i, j, _p(o, _F), _p(d, _F))
        return o, d

    def pe(self, x, L):
        x = np.ascontiguousarray(x, np.float64).reshape(3)
        out = np.empty(3 + 6 * L, np.float64)
        self.lib.r360o_pe(_p(x, _D), L, _p(out, _D))
        return out

    def composite(self, sigma, rgb, t, delta, tau):
        sigma = np.ascontiguousarray(sigma, np.float64)
        rgb = np.ascontiguousarray(rgb, np.float64).reshape(-1, 3)
        t = np.ascontiguousarray(t, np.float32)
        delta = np.ascontiguousarray(delta, np.float32)
        out, full, amb = np.empty(6), np.empty(6), _D()
        self.lib.r360o_composite(sigma.size, _p(sigma, _D), _p(rgb, _D), _p(t, _F), _p(delta, _F),
                                 float(tau), _p(out, _D), _p(full, _D), C.byref(amb))
        return out, full, amb.value

    def params_per_subfield(self, **kw):
        return int(self.lib.r360o_params_per_subfield(C.byref(_make_desc(**kw))))

    def scene(self, **kw):
        return OracleScene(self, **kw)

    def scene_from(self, sc):
        """From a scenegen.Scene (data only)."""
        return OracleScene(self, dims=sc.dims, box_min=sc.box_min, box_max=sc.box_max,
                           n_subfields=sc.n_subfields, hidden_width=sc.hidden_width, n_hidden=sc.n_hidden,
                           pe_pos_levels=sc.pe_pos_levels, pe_dir_levels=sc.pe_dir_levels,
                           samples_per_voxel=sc.samples_per_voxel, t_threshold=sc.t_threshold,
                           density_activation=sc.density_activation, occ_threshold=sc.occ_threshold,
                           occupancy=sc.occupancy, voxel_subfield=sc.voxel_subfield, weights=sc.weights)


def _make_desc(dims=(1, 1, 1), box_min=(0, 0, 0), box_max=(1, 1, 1), n_subfields=1, hidden_width=32,
               n_hidden=2, pe_pos_levels=10, pe_dir_levels=4, samples_per_voxel=8, t_threshold=1e-3,
               density_activation=1, occ_threshold=1, **_ignored):
    d = _Desc()
    d.dims[:] = [int(x) for x in dims]
    d.box_min[:] = [float(x) for x in box_min]
    d.box_max[:] = [float(x) for x in box_max]
    d.n_subfields, d.hidden_width, d.n_hidden = int(n_subfields), int(hidden_width), int(n_hidden)
    d.pe_pos_levels, d.pe_dir_levels = int(pe_pos_levels), int(pe_dir_levels)
    d.samples_per_voxel, d.t_threshold = int(samples_per_voxel), float(t_threshold)
    d.density_activation, d.occ_threshold = int(density_activation), int(occ_threshold)
    return d


class OracleScene:
    def __init__(self, oracle, occupancy, voxel_subfield, weights, **kw):
        self.o = oracle
        self.desc = _make_desc(**kw)
        occ = np.ascontiguousarray(occupancy, np.uint8).reshape(-1)
        lab = np.ascontiguousarray(voxel_subfield, np.int32).reshape(-1)
        w = np.ascontiguousarray(weights, np.float32).reshape(-1)
        self.K = int(self.desc.samples_per_voxel)
        self.h = oracle.lib.r360o_create(C.byref(self.desc), _p(occ, _B), _p(lab, _I), _p(w, _F))
        if not self.h:
            raise ValueError("r360o_create rejected the scene")

    def close(self):
        if self.h:
            self.o.lib.r360o_destroy(self.h)
            self.h = None

    def set_camera(self, model="equirect", fx=0.0, fy=0.0, cx=0.0, cy=0.0):
        """Camera of the following ray_samples / samples_rows / render_* calls (reading P for "pinhole")."""
        m = {"equirect": 0, "pinhole": 1}[model]
        if self.o.lib.r360o_set_camera(self.h, m, fx, fy, cx, cy) != 0:
            raise ValueError("r360o_set_camera rejected the camera")

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def clip(self, o, d):
        o = np.ascontiguousarray(o, np.float32); d = np.ascontiguousarray(d, np.float32)
        t0, t1 = _F(), _F()
        ok = self.o.lib.r360o_clip(self.h, _p(o, _F), _p(d, _F), C.byref(t0), C.byref(t1))
        return bool(ok), t0.value, t1.value

    def walk(self, o, d, only_occupied=False, cap=1 << 16):
        o = np.ascontiguousarray(o, np.float32); d = np.ascontiguousarray(d, np.float32)
        v = np.empty(cap, np.int32); ti = np.empty(cap, np.float32); to = np.empty(cap, np.float32)
        n = self.o.lib.r360o_walk(self.h, _p(o, _F), _p(d, _F), int(only_occupied), cap,
                                  _p(v, _I), _p(ti, _F), _p(to, _F))
        assert n <= cap
        return v[:n].copy(), ti[:n].copy(), to[:n].copy()

    def ray_samples(self, pose, W, H, i, j, cap=1 << 16):
        pose = np.ascontiguousarray(pose, np.float32).reshape(12)
        t = np.empty(cap, np.float32); dl = np.empty(cap, np.float32); sid = np.empty(cap, np.int32)
        n = self.o.lib.r360o_ray_samples(self.h, _p(pose, _F), W, H, i, j, cap, _p(t, _F), _p(dl, _F), _p(sid, _I))
        if n == -2:
            raise ValueError("r360o_ray_samples: inadmissible pose (reading B5)")
        assert n <= cap
        return t[:n].copy(), dl[:n].copy(), sid[:n].copy()

    def samples_rows(self, pose, W, H, row0=0, row1=None):
        """(counts uint32[rows*W], t float32[S], subfield int32[S]) ray-major."""
        pose = np.ascontiguousarray(pose, np.float32).reshape(12)
        row1 = H if row1 is None else row1
        counts = np.empty((row1 - row0) * W, np.uint32)
        total = self.o.lib.r360o_samples_rows(self.h, _p(pose, _F), W, H, row0, row1, _p(counts, _U), 0, None, None)
        if total == -2:
            raise ValueError("r360o_samples_rows: inadmissible pose (reading B5)")
        t = np.empty(max(total, 1), np.float32); sid = np.empty(max(total, 1), np.int32)
        got = self.o.lib.r360o_samples_rows(self.h, _p(pose, _F), W, H, row0, row1, _p(counts, _U), total,
                                            _p(t, _F), _p(sid, _I))
        assert got == total
        return counts, t[:total], sid[:total]

    def subfield_frame(self, k):
        c, ih = np.empty(3, np.float32), np.empty(3, np.float32)
        self.o.lib.r360o_subfield_frame(self.h, k, _p(c, _F), _p(ih, _F))
        return c, ih

    def field(self, k, p, d, raw=False):
        p = np.ascontiguousarray(p, np.float32); d = np.ascontiguousarray(d, np.float32)
        out = np.empty(4, np.float64)
        fn = self.o.lib.r360o_field_raw if raw else self.o.lib.r360o_field
        fn(self.h, k, _p(p, _F), _p(d, _F), _p(out, _D))
        return out

    def _outs(self, n, full):
        r = dict(rgb=np.empty((n, 3), np.float32), depth=np.empty(n, np.float32),
                 n_emitted=np.empty(n, np.uint32), n_used=np.empty(n, np.uint32))
        if full:
            r.update(rgb_full=np.empty((n, 3), np.float32), depth_full=np.empty(n, np.float32),
                     ambiguity=np.empty(n, np.float32))
        return r

    def render_pixels(self, pose, W, H, px, py, full=True):
        pose = np.ascontiguousarray(pose, np.float32).reshape(12)
        px = np.ascontiguousarray(px, np.int32); py = np.ascontiguousarray(py, np.int32)
        r = self._outs(px.size, full)
        rc = self.o.lib.r360o_render_pixels(self.h, _p(pose, _F), W, H, px.size, _p(px, _I), _p(py, _I),
                                            _p(r["rgb"], _F), _p(r["depth"], _F), _p(r.get("rgb_full"), _F),
                                            _p(r.get("depth_full"), _F), _p(r.get("ambiguity"), _F),
                                            _p(r["n_emitted"], _U), _p(r["n_used"], _U))
        if rc:
            raise ValueError("r360o_render_pixels failed")
        return r

    def render_rows(self, pose, W, H, row0=0, row1=None, full=True):
        pose = np.ascontiguousarray(pose, np.float32).reshape(12)
        row1 = H if row1 is None else row1
        r = self._outs((row1 - row0) * W, full)
        rc = self.o.lib.r360o_render_rows(self.h, _p(pose, _F), W, H, row0, row1,
                                          _p(r["rgb"], _F), _p(r["depth"], _F), _p(r.get("rgb_full"), _F),
                                          _p(r.get("depth_full"), _F), _p(r.get("ambiguity"), _F),
                                          _p(r["n_emitted"], _U), _p(r["n_used"], _U))
        if rc:
            raise ValueError("r360o_render_rows failed")
        return r


_ORACLE = None


def load_oracle() -> Oracle:
    global _ORACLE
    if _ORACLE is None:
        _ORACLE = Oracle(C.CDLL(build_oracle()))
    return _ORACLE
