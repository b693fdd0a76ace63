"""ctypes binding of include/tgs.h -- same names as the C entry points, argument marshalling only.

Host buffers are numpy arrays, device buffers are torch CUDA tensors (their `data_ptr()` is passed as is).
There is no fallback: if libtgs.so is missing or CUDA is unusable the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libtgs.so")

HOST, DEVICE = 0, 1
FULL, PSEUDO_REF, TEMPORAL, AUTO = 0, 1, 2, 3
FRAME_R, FRAME_P, FRAME_S = 0, 1, 2
OK, E_INVALID_ARG, E_NO_SCENE, E_NO_CAMERA, E_NO_PRIORS, E_CAPACITY, E_CUDA = 0, -1, -2, -3, -4, -5, -6
CULL_NEAR, CULL_AFC, CULL_TOC, CULL_DEGENERATE, CULL_EMPTY, VISIBLE, NEWLY_VISIBLE = 1, 2, 4, 8, 16, 32, 64
DEPTH_INVALID = np.float32(3.0e38)

EXPORTS = ["tgs_create", "tgs_destroy", "tgs_load_gaussians", "tgs_load_ply", "tgs_set_camera", "tgs_default_params", "tgs_set_params",
           "tgs_render", "tgs_read_image", "tgs_read_image_async", "tgs_wait_reads", "tgs_read_depth", "tgs_read_tile_mask", "tgs_get_stats", "tgs_reset_priors",
           "tgs_strerror", "tgs_last_error", "tgs_debug_get", "tgs_debug_put", "tgs_debug_run_stage",
           "tgs_sort_pairs_static", "tgs_static_last_error"]
SORT_STATIC_MAX_ITEMS = 1 << 20


class TgsParams(C.Structure):
    _fields_ = [("lambda1", C.c_float), ("lambda2", C.c_float), ("lambda_tdc", C.c_int), ("lambda_sr", C.c_int),
                ("eta", C.c_float), ("bg", C.c_float * 3),
                ("enable_afc", C.c_int), ("enable_toc", C.c_int), ("enable_sr", C.c_int), ("max_pairs", C.c_uint32),
                ("exact_tiles", C.c_int), ("prior_policy", C.c_int), ("tgb_downscale", C.c_int),
                ("depth_slabs", C.c_int), ("slab_split", C.c_uint32 * 3)]


class TgsStats(C.Structure):
    _fields_ = [("frame_type", C.c_int),
                ("n_total", C.c_uint32), ("n_near", C.c_uint32), ("n_afc", C.c_uint32), ("n_toc", C.c_uint32),
                ("n_degenerate", C.c_uint32), ("n_empty", C.c_uint32), ("n_visible", C.c_uint32),
                ("n_newly_visible", C.c_uint32),
                ("n_pairs", C.c_uint64),
                ("n_tiles", C.c_uint32), ("n_sel_oc", C.c_uint32), ("n_sel_um", C.c_uint32), ("n_sel", C.c_uint32),
                ("n_rendered", C.c_uint32), ("overflow", C.c_uint32), ("n_interactions", C.c_uint64), ("n_blended", C.c_uint64), ("n_pixel_slots", C.c_uint64),
                ("ms_stage", C.c_float * 8), ("ms_total", C.c_float),
                ("device_bytes", C.c_uint64), ("n_tests", C.c_uint64), ("n_tests_evaluated", C.c_uint64), ("n_half_tile_visits", C.c_uint64), ("n_half_tile_visits_dead", C.c_uint64), ("n_pairs_consumed", C.c_uint64), ("n_slabs", C.c_uint32), ("n_pairs_slab", C.c_uint32 * 4), ("n_finished_slab", C.c_uint32 * 4),
                ("launches_total", C.c_uint64)]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_}
        d["ms_stage"] = list(self.ms_stage)
        d["n_pairs_slab"] = list(self.n_pairs_slab)
        d["n_finished_slab"] = list(self.n_finished_slab)
        return d


class TgsError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        super().__init__(f"{what}: {code} ({detail})")


_lib = None


def lib():
    """Load libtgs.so; raises if it has not been built (python -m paper_2607_03390_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO):
            raise FileNotFoundError(f"{SO} is missing: build it with `python -m paper_2607_03390_b200.build`")
        L = C.CDLL(SO)
        vp, fp = C.c_void_p, C.c_void_p
        L.tgs_create.argtypes = [C.POINTER(vp), C.c_int, vp]
        L.tgs_destroy.argtypes = [vp]
        L.tgs_destroy.restype = None
        L.tgs_load_gaussians.argtypes = [vp, C.c_uint32, C.c_int, fp, fp, fp, fp, fp, C.c_int]
        L.tgs_set_camera.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_float, C.c_float, C.c_float, C.c_int, C.c_int,
                                     C.c_float, C.c_float]
        L.tgs_default_params.argtypes = [C.POINTER(TgsParams)]
        L.tgs_default_params.restype = None
        L.tgs_set_params.argtypes = [vp, C.POINTER(TgsParams)]
        L.tgs_load_ply.argtypes = [vp, C.c_char_p]
        L.tgs_render.argtypes = [vp, C.c_int]
        L.tgs_read_image.argtypes = [vp, vp, C.c_int]
        L.tgs_read_image_async.argtypes = [vp, vp]
        L.tgs_wait_reads.argtypes = [vp]
        L.tgs_read_depth.argtypes = [vp, vp, vp, C.c_int]
        L.tgs_read_tile_mask.argtypes = [vp, vp, C.c_int]
        L.tgs_get_stats.argtypes = [vp, C.POINTER(TgsStats)]
        L.tgs_reset_priors.argtypes = [vp]
        L.tgs_strerror.argtypes = [C.c_int]
        L.tgs_strerror.restype = C.c_char_p
        L.tgs_last_error.argtypes = [vp]
        L.tgs_last_error.restype = C.c_char_p
        L.tgs_debug_get.argtypes = [vp, C.c_char_p, vp, C.c_size_t, C.c_int]
        L.tgs_debug_get.restype = C.c_longlong
        L.tgs_debug_put.argtypes = [vp, C.c_char_p, vp, C.c_size_t, C.c_int]
        L.tgs_debug_run_stage.argtypes = [vp, C.c_char_p]
        L.tgs_sort_pairs_static.argtypes = [C.c_int, vp, vp, vp, vp, vp, C.c_uint32, C.c_int, vp]
        L.tgs_static_last_error.argtypes = []
        L.tgs_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _ptr_mem(a):
    """(pointer, mem) of a numpy array (host) or a torch CUDA tensor (device)."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data, HOST
    # torch tensor
    assert a.is_contiguous()
    return a.data_ptr(), (DEVICE if a.is_cuda else HOST)


_DEBUG_DTYPES = {
    "rec_uvdo": np.float32, "rec_conic": np.float32, "rec_rect": np.uint16, "rec_flags": np.uint32, "rec_rgb": np.float32,
    "tiles_touched": np.uint32, "offsets": np.uint32, "keys": np.uint64, "vals": np.uint32, "ranges": np.uint32,
    "tile_order": np.uint32, "warp_depth": np.float32, "warp_sigma": np.float32, "fill_depth": np.float32,
    "rendered": np.uint8, "F": np.float32, "prior_depth": np.float32, "prior_sigma": np.float32, "prior_image": np.float32,
    "cov3d": np.float32, "tau": np.float32,
}


def sort_pairs_static(keys_in, vals_in, keys_out, vals_out, n, key_bytes, device=0, stream=None, status=None):
    """tgs_sort_pairs_static: the entry point that allocates nothing (include/tgs.h).  The buffers are CUDA tensors of 4-byte
    elements (anything with data_ptr()) or raw device addresses; only enqueues work on `stream` (default stream if None)."""
    def ptr(a):
        return C.c_void_p(a if isinstance(a, int) else (a.data_ptr() if a is not None else 0))
    L = lib()
    rc = L.tgs_sort_pairs_static(device, C.c_void_p(stream or 0), ptr(keys_in), ptr(vals_in), ptr(keys_out), ptr(vals_out), n, key_bytes,
                                 ptr(status))
    if rc != OK:
        raise TgsError(rc, "tgs_sort_pairs_static", L.tgs_strerror(rc).decode() + "; " + L.tgs_static_last_error().decode())
    return rc


class Context:
    """One tgs_ctx.  Methods are the C calls without the `tgs_` prefix."""

    def __init__(self, device: int = 0, stream: int | None = None):
        self.L = lib()
        self.h = C.c_void_p()
        rc = self.L.tgs_create(C.byref(self.h), device, C.c_void_p(stream or 0))
        if rc != OK:
            raise TgsError(rc, "tgs_create", self.L.tgs_strerror(rc).decode())
        self.W = self.H = self.n = 0

    def destroy(self):
        if getattr(self, "h", None):
            self.L.tgs_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc < 0:
            raise TgsError(rc, what, self.L.tgs_strerror(rc).decode() + "; " + self.L.tgs_last_error(self.h).decode())
        return rc

    # -- scene / camera / params
    def load_gaussians(self, means, scales, quats, opacity, sh, sh_degree):
        arrs = []
        mems = set()
        for a in (means, scales, quats, opacity, sh):
            if isinstance(a, np.ndarray) or not hasattr(a, "data_ptr"):
                a = np.ascontiguousarray(a, dtype=np.float32)
            p, m = _ptr_mem(a)
            arrs.append((a, p))
            mems.add(m)
        assert len(mems) == 1, "all arrays must live in the same memory space"
        self.n = int(arrs[0][0].shape[0])
        rc = self.L.tgs_load_gaussians(self.h, self.n, sh_degree, *[C.c_void_p(p) for _, p in arrs], mems.pop())
        return self._chk(rc, "tgs_load_gaussians")

    def load_ply(self, path):
        """Trained 3DGS checkpoint (`point_cloud.ply`); returns (n, sh_degree) is not needed: stats carry n_total."""
        return self._chk(self.L.tgs_load_ply(self.h, str(path).encode()), "tgs_load_ply")

    def load_scene(self, sc):
        return self.load_gaussians(sc.means, sc.scales, sc.quats, sc.opacity, sc.sh, sc.sh_degree)

    def set_camera(self, view, cam):
        v = np.ascontiguousarray(view, dtype=np.float32).reshape(16)
        self.W, self.H = cam.W, cam.H
        rc = self.L.tgs_set_camera(self.h, v.ctypes.data_as(C.POINTER(C.c_float)), cam.fx, cam.fy, cam.cx, cam.cy, cam.W, cam.H,
                                   cam.znear, cam.zfar)
        return self._chk(rc, "tgs_set_camera")

    def default_params(self) -> TgsParams:
        p = TgsParams()
        self.L.tgs_default_params(C.byref(p))
        return p

    def set_params(self, p: TgsParams):
        return self._chk(self.L.tgs_set_params(self.h, C.byref(p)), "tgs_set_params")

    def render(self, mode=AUTO):
        return self._chk(self.L.tgs_render(self.h, mode), "tgs_render")

    def render_rc(self, mode):
        return self.L.tgs_render(self.h, mode)

    def reset_priors(self):
        return self._chk(self.L.tgs_reset_priors(self.h), "tgs_reset_priors")

    # -- read back
    def read_image(self, out=None):
        if out is None:
            out = np.empty((self.H, self.W, 3), dtype=np.float32)
        p, m = _ptr_mem(out)
        self._chk(self.L.tgs_read_image(self.h, C.c_void_p(p), m), "tgs_read_image")
        return out

    def read_image_async(self, out):
        """`out`: page-locked host array [H][W][3] float32; valid after wait_reads()."""
        assert out.dtype == np.float32 and out.flags["C_CONTIGUOUS"] and out.size == self.H * self.W * 3
        self._chk(self.L.tgs_read_image_async(self.h, C.c_void_p(out.ctypes.data)), "tgs_read_image_async")

    def wait_reads(self):
        self._chk(self.L.tgs_wait_reads(self.h), "tgs_wait_reads")

    def read_depth(self, depth=None, sigma=None):
        if depth is None:
            depth = np.empty((self.H, self.W), dtype=np.float32)
            sigma = np.empty((self.H, self.W), dtype=np.float32)
        p, m = _ptr_mem(depth)
        ps = _ptr_mem(sigma)[0] if sigma is not None else None
        self._chk(self.L.tgs_read_depth(self.h, C.c_void_p(p), C.c_void_p(ps), m), "tgs_read_depth")
        return depth, sigma

    def read_tile_mask(self):
        out = np.empty(((self.H + 15) // 16, (self.W + 15) // 16), dtype=np.uint8)
        self._chk(self.L.tgs_read_tile_mask(self.h, C.c_void_p(out.ctypes.data), HOST), "tgs_read_tile_mask")
        return out

    def get_stats(self, check=True) -> dict:
        s = TgsStats()
        rc = self.L.tgs_get_stats(self.h, C.byref(s))
        if check:
            self._chk(rc, "tgs_get_stats")
        return s.as_dict()

    # -- test-only
    def debug_get(self, name):
        nb = self._chk(self.L.tgs_debug_get(self.h, name.encode(), None, 0, HOST), f"tgs_debug_get({name})")
        dt = np.dtype(_DEBUG_DTYPES[name])
        out = np.empty(nb // dt.itemsize, dtype=dt)
        if nb:
            self._chk(self.L.tgs_debug_get(self.h, name.encode(), C.c_void_p(out.ctypes.data), nb, HOST), f"tgs_debug_get({name})")
        return out

    def debug_put(self, name, arr):
        if isinstance(arr, np.ndarray):
            arr = np.ascontiguousarray(arr)
            nbytes = arr.nbytes
        else:
            nbytes = arr.numel() * arr.element_size()
        p, m = _ptr_mem(arr)
        return self._chk(self.L.tgs_debug_put(self.h, name.encode(), C.c_void_p(p), nbytes, m), f"tgs_debug_put({name})")

    def debug_run_stage(self, stage):
        return self._chk(self.L.tgs_debug_run_stage(self.h, stage.encode()), f"tgs_debug_run_stage({stage})")
