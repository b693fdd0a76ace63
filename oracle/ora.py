"""ctypes binding of oracle/libora.so (built from oracle/ora.cpp).  TEST INFRASTRUCTURE ONLY."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libora.so")
_SRC = os.path.join(_HERE, "ora.cpp")
_HDR = os.path.join(_HERE, "ora.h")

FULL, PSEUDO_REF, TEMPORAL, AUTO = 0, 1, 2, 3
FRAME_R, FRAME_P, FRAME_S = 0, 1, 2
DEPTH_INVALID = np.float32(3.0e38)
CULL_NEAR, CULL_AFC, CULL_TOC, CULL_DEGENERATE, CULL_EMPTY, VISIBLE, NEWLY_VISIBLE = 1, 2, 4, 8, 16, 32, 64

RECORD_DTYPE = np.dtype([
    ("u", "<f4"), ("v", "<f4"), ("d", "<f4"), ("o", "<f4"),
    ("A", "<f4"), ("B", "<f4"), ("C", "<f4"), ("tau", "<f4"),
    ("ca", "<f4"), ("cb", "<f4"), ("cc", "<f4"), ("pad0", "<f4"),
    ("r", "<f4"), ("g", "<f4"), ("b", "<f4"), ("radius", "<f4"),
    ("x_lo", "<u2"), ("x_hi", "<u2"), ("y_lo", "<u2"), ("y_hi", "<u2"),
    ("flags", "<u4"), ("tiles_touched", "<u4"),
])
assert RECORD_DTYPE.itemsize == 80


class OraParams(C.Structure):
    _fields_ = [("lambda1", C.c_float), ("lambda2", C.c_float), ("lambda_tdc", C.c_int), ("lambda_sr", C.c_int),
                ("eta", C.c_float), ("bg", C.c_float * 3),
                ("enable_afc", C.c_int), ("enable_toc", C.c_int), ("enable_sr", C.c_int), ("exact_tiles", C.c_int),
                ("prior_policy", C.c_int), ("tgb_downscale", C.c_int)]


class OraStats(C.Structure):
    _fields_ = [("frame_type", C.c_int),
                ("n_total", C.c_uint32), ("n_near", C.c_uint32), ("n_afc", C.c_uint32), ("n_toc", C.c_uint32),
                ("n_degenerate", C.c_uint32), ("n_empty", C.c_uint32), ("n_visible", C.c_uint32),
                ("n_newly_visible", C.c_uint32),
                ("n_pairs", C.c_uint64),
                ("n_tiles", C.c_uint32), ("n_sel_oc", C.c_uint32), ("n_sel_um", C.c_uint32), ("n_sel", C.c_uint32),
                ("n_rendered", C.c_uint32),
                ("n_interactions", C.c_uint64),
                ("ms_preprocess", C.c_double), ("ms_sort", C.c_double), ("ms_blend", C.c_double),
                ("ms_temporal", C.c_double), ("ms_total", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class OraSched(C.Structure):
    _fields_ = [("since_R", C.c_int), ("since_ref", C.c_int), ("force_P", C.c_int), ("valid", C.c_int)]


def build(force: bool = False) -> str:
    """Compile oracle/ora.cpp -> oracle/libora.so (g++ -O2, no contraction, no fast-math).
    ORA_SANITIZE=1 builds oracle/libora_san.so with -fsanitize=address,undefined instead (run the pins under
    LD_PRELOAD=$(gcc -print-file-name=libasan.so); profiles/r2_sanitizers.md has the command and its result)."""
    san = os.environ.get("ORA_SANITIZE") == "1"
    so = os.path.join(_HERE, "libora_san.so") if san else _SO
    if (not force and os.path.exists(so)
            and os.path.getmtime(so) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return so
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-shared", "-fPIC"]
    if san:
        cmd += ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    subprocess.run(cmd + ["-o", so, _SRC], check=True)
    return so


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        fp = C.POINTER(C.c_float)
        L.ora_create.restype = C.c_void_p
        L.ora_destroy.argtypes = [C.c_void_p]
        L.ora_load_gaussians.argtypes = [C.c_void_p, C.c_uint32, C.c_int, fp, fp, fp, fp, fp]
        L.ora_set_camera.argtypes = [C.c_void_p, fp, C.c_float, C.c_float, C.c_float, C.c_float, C.c_int, C.c_int,
                                     C.c_float, C.c_float]
        L.ora_set_params.argtypes = [C.c_void_p, C.POINTER(OraParams)]
        L.ora_default_params.argtypes = [C.POINTER(OraParams)]
        L.ora_render.argtypes = [C.c_void_p, C.c_int]
        L.ora_read_image.argtypes = [C.c_void_p, fp]
        L.ora_read_depth.argtypes = [C.c_void_p, fp, fp]
        L.ora_read_tile_mask.argtypes = [C.c_void_p, C.POINTER(C.c_uint8)]
        L.ora_get_stats.argtypes = [C.c_void_p, C.POINTER(OraStats)]
        L.ora_reset_priors.argtypes = [C.c_void_p]
        L.ora_force_all_tiles.argtypes = [C.c_void_p, C.c_int]
        L.ora_get.argtypes = [C.c_void_p, C.c_char_p, C.c_void_p, C.c_size_t]
        L.ora_get.restype = C.c_longlong
        L.ora_put.argtypes = [C.c_void_p, C.c_char_p, C.c_void_p, C.c_size_t]
        L.ora_stage.argtypes = [C.c_void_p, C.c_char_p]
        L.ora_sh_basis.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.ora_box_qmin.argtypes = [C.c_float] * 9
        L.ora_box_qmin.restype = C.c_float
        L.ora_schedule_next.argtypes = [C.POINTER(OraSched), C.c_int, C.c_int]
        L.ora_schedule_feedback.argtypes = [C.POINTER(OraSched), C.c_int, C.c_uint32, C.c_uint32, C.c_float]
        _lib = L
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


_GET_DTYPES = {
    "records": RECORD_DTYPE, "keys": np.uint64, "vals": np.uint32, "ranges": np.uint32,
    "warp_depth": np.float32, "warp_sigma": np.float32, "fill_depth": np.float32, "corr_xy": np.float32,
    "matched": np.uint8, "rendered": np.uint8, "rendered_now": np.uint8, "rendered_sure": np.uint8, "rendered_maybe": np.uint8,
    "borderline": np.uint8, "F": np.float32, "prior_depth": np.float32, "prior_sigma": np.float32,
    "prior_image": np.float32, "prior_view": np.float32, "M": np.float32, "Minv": np.float32,
    "cov3d": np.float32, "tau": np.float32,
}


class Oracle:
    """Thin object wrapper; method names mirror the C functions."""

    def __init__(self):
        self.L = lib()
        self.h = C.c_void_p(self.L.ora_create())
        self.W = self.H = 0
        self.n = 0

    def close(self):
        if self.h:
            self.L.ora_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _chk(rc, what):
        if rc < 0:
            raise RuntimeError(f"oracle {what} failed: {rc}")
        return rc

    def load_gaussians(self, means, scales, quats, opacity, sh, sh_degree):
        means, scales, quats, opacity, sh = map(_f32, (means, scales, quats, opacity, sh))
        self.n = means.shape[0]
        return self._chk(self.L.ora_load_gaussians(self.h, self.n, sh_degree, _fp(means), _fp(scales), _fp(quats),
                                                   _fp(opacity), _fp(sh)), "load_gaussians")

    def load_scene(self, sc):
        return self.load_gaussians(sc.means, sc.scales, sc.quats, sc.opacity, sc.sh, sc.sh_degree)

    def set_camera(self, view, cam):
        v = _f32(view).reshape(16)
        self.W, self.H = cam.W, cam.H
        return self._chk(self.L.ora_set_camera(self.h, _fp(v), cam.fx, cam.fy, cam.cx, cam.cy, cam.W, cam.H,
                                               cam.znear, cam.zfar), "set_camera")

    def default_params(self) -> OraParams:
        p = OraParams()
        self.L.ora_default_params(C.byref(p))
        return p

    def set_params(self, p: OraParams):
        return self._chk(self.L.ora_set_params(self.h, C.byref(p)), "set_params")

    def render(self, mode) -> int:
        return self._chk(self.L.ora_render(self.h, mode), "render")

    def render_rc(self, mode) -> int:
        return self.L.ora_render(self.h, mode)

    def read_image(self):
        out = np.empty((self.H, self.W, 3), dtype=np.float32)
        self._chk(self.L.ora_read_image(self.h, _fp(out)), "read_image")
        return out

    def read_depth(self):
        d = np.empty((self.H, self.W), dtype=np.float32)
        s = np.empty((self.H, self.W), dtype=np.float32)
        self._chk(self.L.ora_read_depth(self.h, _fp(d), _fp(s)), "read_depth")
        return d, s

    def read_tile_mask(self):
        TX, TY = (self.W + 15) // 16, (self.H + 15) // 16
        m = np.empty((TY, TX), dtype=np.uint8)
        self._chk(self.L.ora_read_tile_mask(self.h, m.ctypes.data_as(C.POINTER(C.c_uint8))), "read_tile_mask")
        return m

    def stats(self) -> dict:
        s = OraStats()
        self._chk(self.L.ora_get_stats(self.h, C.byref(s)), "get_stats")
        return s.as_dict()

    def reset_priors(self):
        self.L.ora_reset_priors(self.h)

    def force_all_tiles(self, on=True):
        self.L.ora_force_all_tiles(self.h, int(on))

    def get(self, name):
        nb = self._chk(self.L.ora_get(self.h, name.encode(), None, 0), f"get({name})")
        dt = np.dtype(_GET_DTYPES[name])
        out = np.empty(nb // dt.itemsize, dtype=dt)
        if nb:
            self.L.ora_get(self.h, name.encode(), out.ctypes.data_as(C.c_void_p), nb)
        return out

    def put(self, name, arr):
        a = np.ascontiguousarray(arr)
        return self._chk(self.L.ora_put(self.h, name.encode(), a.ctypes.data_as(C.c_void_p), a.nbytes), f"put({name})")

    def stage(self, name):
        return self._chk(self.L.ora_stage(self.h, name.encode()), f"stage({name})")


def sh_basis(degree, d):
    d = np.ascontiguousarray(d, dtype=np.float64)
    K = (degree + 1) ** 2
    Y = np.zeros(K, dtype=np.float64)
    lib().ora_sh_basis(degree, d.ctypes.data_as(C.POINTER(C.c_double)), Y.ctypes.data_as(C.POINTER(C.c_double)))
    return Y


def box_qmin(u, v, A, B, Cc, x0, x1, y0, y1):
    return float(lib().ora_box_qmin(u, v, A, B, Cc, x0, x1, y0, y1))
