"""Seeded scene / trajectory generators for the five configs of BASELINE.json.

These synthetic inputs STAND IN for the paper's datasets (Mip-NeRF-360, MatrixCity, Mega-NeRF
Residence/Building/Rubble, Hierarchical-GS SmallCity) and their trained 3DGS /
CityGS checkpoints, none of which are available.  Everything is drawn from
`numpy.random.default_rng(seed)` (PCG64), seed = config index (0-based).

Conventions: world->camera matrix `view` is row-major 4x4 and rigid; the camera
looks along +z, x is right, y is DOWN; pixel (i, j) is sampled at (u, v) = (i, j);
cx = (W-1)/2, cy = (H-1)/2.

No arithmetic of the method lives here (no projection, no blending, no warping).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import math
import numpy as np

CONFIG_NAMES = {
    1: "tiny_16k_256x256",
    2: "object_500k_720p",
    3: "unbounded_3M_1080p",
    4: "aerial_8M_1080p",
    5: "layers_3M_1080p",
}


@dataclass
class Camera:
    W: int
    H: int
    fx: float
    fy: float
    cx: float
    cy: float
    znear: float = 0.01
    zfar: float = 1000.0


@dataclass
class Scene:
    name: str
    means: np.ndarray      # [N,3] f32
    scales: np.ndarray     # [N,3] f32, linear (post-exp)
    quats: np.ndarray      # [N,4] f32, (w,x,y,z), not necessarily normalised
    opacity: np.ndarray    # [N]   f32, post-sigmoid
    sh: np.ndarray         # [N,K,3] f32
    sh_degree: int
    camera: Camera
    poses: np.ndarray      # [F,4,4] f32 world->camera
    modes: list = field(default_factory=list)   # per-frame render mode names ("auto" | "full" | "temporal")

    @property
    def n(self) -> int:
        return int(self.means.shape[0])


def _normalize(v):
    v = np.asarray(v, dtype=np.float64)
    return v / np.linalg.norm(v)


def look_at(eye, target, up) -> np.ndarray:
    """World->camera (row-major 4x4 float64): z forward, x right, y down."""
    eye = np.asarray(eye, dtype=np.float64)
    f = _normalize(np.asarray(target, dtype=np.float64) - eye)
    return view_from_forward(eye, f, up)


def view_from_forward(eye, f, up) -> np.ndarray:
    eye = np.asarray(eye, dtype=np.float64)
    f = _normalize(f)
    r = _normalize(np.cross(f, np.asarray(up, dtype=np.float64)))
    d = np.cross(f, r)
    R = np.stack([r, d, f], axis=0)
    V = np.eye(4)
    V[:3, :3] = R
    V[:3, 3] = -R @ eye
    return V


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def _sh(rng, n, degree, dc_std=0.5, rest_std=0.05):
    K = (degree + 1) ** 2
    sh = np.empty((n, K, 3), dtype=np.float32)
    sh[:, 0, :] = rng.normal(0.0, dc_std, size=(n, 3)).astype(np.float32)
    if K > 1:
        sh[:, 1:, :] = rng.normal(0.0, rest_std, size=(n, K - 1, 3)).astype(np.float32)
    return sh


def _quats(rng, n):
    return rng.normal(0.0, 1.0, size=(n, 4)).astype(np.float32)


def _hfov_fx(W, deg):
    return 0.5 * W / math.tan(math.radians(deg) * 0.5)


def _std_camera(W, H, fx):
    return Camera(W=W, H=H, fx=float(fx), fy=float(fx), cx=(W - 1) / 2.0, cy=(H - 1) / 2.0)


# ----------------------------------------------------------------------------- config 1
def _config1(n, frames, rng):
    means = np.empty((0, 3))
    while means.shape[0] < n:
        m = rng.normal(0.0, 1.0, size=(n, 3))
        m = m[np.all(np.abs(m) < 3.0, axis=1)]
        means = np.concatenate([means, m], axis=0)
    means = means[:n].astype(np.float32)
    scales = np.exp(rng.normal(-3.5, 0.5, size=(n, 3))).astype(np.float32)
    quats = _quats(rng, n)
    opacity = _sigmoid(rng.normal(0.0, 1.5, size=n)).astype(np.float32)
    sh = _sh(rng, n, 0)
    cam = _std_camera(256, 256, 256.0)
    poses = []
    for f in range(frames):
        a = math.radians(1.0 * f)
        eye = (6.0 * math.sin(a), 0.0, -6.0 * math.cos(a))
        poses.append(look_at(eye, (0, 0, 0), (0, 1, 0)))
    modes = ["full"] + ["temporal"] * (frames - 1)
    return Scene(CONFIG_NAMES[1], means, scales, quats, opacity, sh, 0, cam,
                 np.asarray(poses, dtype=np.float32), modes)


# ----------------------------------------------------------------------------- config 2
def _random_rotation(rng):
    q = _normalize(rng.normal(size=4))
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def _config2(n, frames, rng):
    ncl = 20
    centres = rng.uniform(-2.0, 2.0, size=(ncl, 3))
    per = np.full(ncl, n // ncl)
    per[: n - per.sum()] += 1
    chunks = []
    for c in range(ncl):
        R = _random_rotation(rng)
        s = np.exp(rng.normal(-1.0, 0.5, size=3))
        pts = rng.normal(size=(per[c], 3)) * s
        chunks.append(centres[c] + pts @ R.T)
    means = np.clip(np.concatenate(chunks, axis=0), -2.0, 2.0).astype(np.float32)
    scales = np.exp(rng.normal(-4.0, 0.7, size=(n, 3))).astype(np.float32)
    quats = _quats(rng, n)
    opacity = _sigmoid(rng.normal(0.5, 2.0, size=n)).astype(np.float32)
    sh = _sh(rng, n, 3)
    cam = _std_camera(1280, 720, _hfov_fx(1280, 60.0))
    poses = []
    for f in range(frames):
        a = math.radians(0.5 * f)
        eye = (5.0 * math.sin(a), 0.2 * math.sin(2 * math.pi * f / 120.0), -5.0 * math.cos(a))
        poses.append(look_at(eye, (0, 0, 0), (0, 1, 0)))
    return Scene(CONFIG_NAMES[2], means, scales, quats, opacity, sh, 3, cam,
                 np.asarray(poses, dtype=np.float32), ["auto"] * frames)


# ----------------------------------------------------------------------------- config 3
def _catmull_rom_centripetal(P, samples_per_seg=2000):
    """Dense samples of the centripetal Catmull-Rom spline through P[1..-2]."""
    out = []
    for i in range(1, len(P) - 2):
        p0, p1, p2, p3 = P[i - 1], P[i], P[i + 1], P[i + 2]
        t0 = 0.0
        t1 = t0 + math.sqrt(np.linalg.norm(p1 - p0))
        t2 = t1 + math.sqrt(np.linalg.norm(p2 - p1))
        t3 = t2 + math.sqrt(np.linalg.norm(p3 - p2))
        t = np.linspace(t1, t2, samples_per_seg, endpoint=False)[:, None]
        A1 = (t1 - t) / (t1 - t0) * p0 + (t - t0) / (t1 - t0) * p1
        A2 = (t2 - t) / (t2 - t1) * p1 + (t - t1) / (t2 - t1) * p2
        A3 = (t3 - t) / (t3 - t2) * p2 + (t - t2) / (t3 - t2) * p3
        B1 = (t2 - t) / (t2 - t0) * A1 + (t - t0) / (t2 - t0) * A2
        B2 = (t3 - t) / (t3 - t1) * A2 + (t - t1) / (t3 - t1) * A3
        out.append((t2 - t) / (t2 - t1) * B1 + (t - t1) / (t2 - t1) * B2)
    return np.concatenate(out, axis=0)


def _spline_trajectory(waypoints, frames, step, max_deg, up):
    dense = _catmull_rom_centripetal(waypoints)
    seg = np.linalg.norm(np.diff(dense, axis=0), axis=1)
    s = np.concatenate([[0.0], np.cumsum(seg)])
    need = step * (frames + 1)
    if s[-1] < need:
        raise ValueError("spline too short for the trajectory")
    targets = step * np.arange(frames + 1)
    pos = np.stack([np.interp(targets, s, dense[:, k]) for k in range(3)], axis=1)
    poses = []
    fwd = _normalize(pos[1] - pos[0])
    max_rad = math.radians(max_deg)
    for f in range(frames):
        want = _normalize(pos[f + 1] - pos[f])
        ang = math.acos(float(np.clip(np.dot(fwd, want), -1.0, 1.0)))
        if ang > max_rad:
            # rotate fwd towards want by max_rad (slerp)
            k = max_rad / ang
            sa = math.sin(ang)
            fwd = _normalize(math.sin((1 - k) * ang) / sa * fwd + math.sin(k * ang) / sa * want)
        else:
            fwd = want
        poses.append(view_from_forward(pos[f], fwd, up))
    return np.asarray(poses, dtype=np.float32)


def _config3(n, frames, rng):
    n_c = int(round(0.7 * n))
    n_s = n - n_c
    means_c = rng.normal(0.0, math.sqrt(1.5), size=(n_c, 3))
    scales_c = np.exp(rng.normal(-4.5, 0.8, size=(n_c, 3)))
    radius = rng.uniform(20.0, 60.0, size=n_s)
    d = rng.normal(size=(n_s, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    means_s = d * radius[:, None]
    scales_s = np.exp(rng.normal(-1.5, 0.8, size=(n_s, 3)))
    means = np.concatenate([means_c, means_s]).astype(np.float32)
    scales = np.concatenate([scales_c, scales_s]).astype(np.float32)
    # interleave centre / shell so that memory order carries no depth structure
    perm = rng.permutation(n)
    means, scales = means[perm], scales[perm]
    quats = _quats(rng, n)
    opacity = _sigmoid(rng.normal(0.0, 2.0, size=n)).astype(np.float32)
    sh = _sh(rng, n, 3)
    cam = _std_camera(1920, 1080, _hfov_fx(1920, 60.0))
    # 8 waypoints uniform in the ball r<4
    wp = []
    while len(wp) < 8:
        p = rng.uniform(-4.0, 4.0, size=3)
        if np.linalg.norm(p) < 4.0:
            wp.append(p)
    poses = _spline_trajectory(np.asarray(wp), frames, 0.02, 0.6, (0, 1, 0))
    return Scene(CONFIG_NAMES[3], means, scales, quats, opacity, sh, 3, cam, poses, ["auto"] * frames)


# ----------------------------------------------------------------------------- config 4
def _value_noise(rng, x, y, wavelength, size=512):
    grid = rng.uniform(-1.0, 1.0, size=(size, size))
    gx = x / wavelength
    gy = y / wavelength
    ix = np.floor(gx).astype(np.int64)
    iy = np.floor(gy).astype(np.int64)
    fx = gx - ix
    fy = gy - iy
    fx = fx * fx * (3 - 2 * fx)
    fy = fy * fy * (3 - 2 * fy)
    ix0, iy0 = ix % size, iy % size
    ix1, iy1 = (ix + 1) % size, (iy + 1) % size
    v00, v10 = grid[iy0, ix0], grid[iy0, ix1]
    v01, v11 = grid[iy1, ix0], grid[iy1, ix1]
    return (v00 * (1 - fx) + v10 * fx) * (1 - fy) + (v01 * (1 - fx) + v11 * fx) * fy


def _fbm(rng, x, y, octaves=5, base_wavelength=100.0, amplitude=15.0, gain=0.5):
    h = np.zeros_like(x)
    amp, wl = amplitude, base_wavelength
    for _ in range(octaves):
        h += amp * _value_noise(rng, x, y, wl)
        amp *= gain
        wl *= 0.5
    return h


def _config4(n, frames, rng):
    n_b = int(round(0.15 * n))
    n_g = n - n_b
    xy = rng.uniform(-200.0, 200.0, size=(n_g, 2))
    z = _fbm(rng, xy[:, 0] + 200.0, xy[:, 1] + 200.0) + rng.normal(0.0, 2.0, size=n_g)
    ground = np.concatenate([xy, z[:, None]], axis=1)
    # 200 boxes: points on walls / roofs
    nb = 200
    bc = rng.uniform(-190.0, 190.0, size=(nb, 2))
    bw = rng.uniform(10.0, 30.0, size=(nb, 2))
    bh = rng.uniform(10.0, 50.0, size=nb)
    which = rng.integers(0, nb, size=n_b)
    face = rng.integers(0, 5, size=n_b)          # 0..3 walls, 4 roof
    a = rng.uniform(-0.5, 0.5, size=n_b)
    b = rng.uniform(0.0, 1.0, size=n_b)
    c = rng.uniform(-0.5, 0.5, size=n_b)
    px = np.where(face == 0, -0.5, np.where(face == 1, 0.5, a))
    py = np.where(face == 2, -0.5, np.where(face == 3, 0.5, np.where(face == 4, c, a)))
    pz = np.where(face == 4, 1.0, b)
    bx = bc[which, 0] + px * bw[which, 0]
    by = bc[which, 1] + py * bw[which, 1]
    bz = pz * bh[which]
    boxes = np.stack([bx, by, bz], axis=1)
    means = np.concatenate([ground, boxes]).astype(np.float32)
    perm = rng.permutation(n)
    means = means[perm]
    scales = np.exp(rng.normal(-2.5, 0.9, size=(n, 3))).astype(np.float32)
    quats = _quats(rng, n)
    opacity = _sigmoid(rng.normal(0.5, 2.0, size=n)).astype(np.float32)
    sh = _sh(rng, n, 3)
    cam = _std_camera(1920, 1080, _hfov_fx(1920, 70.0))
    pitch = math.radians(30.0)
    fwd = (math.cos(pitch), 0.0, -math.sin(pitch))
    poses = [view_from_forward((-75.0 + 0.5 * f, 0.0, 80.0), fwd, (0, 0, 1)) for f in range(frames)]
    return Scene(CONFIG_NAMES[4], means, scales, quats, opacity, sh, 3, cam,
                 np.asarray(poses, dtype=np.float32), ["auto"] * frames)


# ----------------------------------------------------------------------------- config 5
def _config5(n, frames, rng):
    layers = 10
    per = n // layers
    n = per * layers
    means = np.empty((n, 3), dtype=np.float32)
    quats = np.empty((n, 4), dtype=np.float32)
    for l in range(layers):
        sl = slice(l * per, (l + 1) * per)
        means[sl, 0:2] = rng.uniform(-5.0, 5.0, size=(per, 2))
        means[sl, 2] = 0.5 * l
        th = rng.uniform(0.0, 2 * math.pi, size=per)       # spin about the sheet normal (z)
        quats[sl] = np.stack([np.cos(th / 2), np.zeros(per), np.zeros(per), np.sin(th / 2)], axis=1)
    scales = np.empty((n, 3), dtype=np.float32)
    scales[:, 0:2] = np.exp(rng.normal(-3.0, 0.3, size=(n, 2)))
    scales[:, 2] = math.exp(-6.0)
    perm = rng.permutation(n)
    means, quats, scales = means[perm], quats[perm], scales[perm]
    opacity = _sigmoid(rng.normal(1.0, 1.0, size=n)).astype(np.float32)
    sh = _sh(rng, n, 1)
    cam = _std_camera(1920, 1080, _hfov_fx(1920, 60.0))
    poses = []
    yaw, zpos = 0.0, -8.0
    f = 0
    cycle = 0
    while f < frames:
        sign = 1.0 if cycle % 2 == 0 else -1.0
        for k in range(40):
            if f >= frames:
                break
            if k < 10:
                yaw += sign * 4.0
                zpos += 0.1
            else:
                yaw += sign * 0.2
            a = math.radians(yaw)
            fwd = (math.sin(a), 0.0, math.cos(a))
            poses.append(view_from_forward((0.0, 0.0, zpos), fwd, (0, -1, 0)))
            f += 1
        cycle += 1
    return Scene(CONFIG_NAMES[5], means, scales, quats, opacity, sh, 1, cam,
                 np.asarray(poses, dtype=np.float32), ["auto"] * frames)


_DEFAULTS = {1: (16384, 8), 2: (500_000, 120), 3: (3_000_000, 300), 4: (8_000_000, 300), 5: (3_000_000, 200)}
_BUILDERS = {1: _config1, 2: _config2, 3: _config3, 4: _config4, 5: _config5}


def make_config(idx: int, n: int | None = None, frames: int | None = None,
                width: int | None = None, height: int | None = None) -> Scene:
    """Config `idx` (1-based, BASELINE.json:configs).  `n`/`frames`/`width`/`height` may be
    reduced for tests; the distributions and the trajectory recipe stay the same (focal length is
    rescaled with the width so the field of view is kept)."""
    if idx not in _BUILDERS:
        raise ValueError(f"unknown config {idx}")
    dn, df = _DEFAULTS[idx]
    rng = np.random.default_rng(idx - 1)
    sc = _BUILDERS[idx](n or dn, frames or df, rng)
    if width is not None or height is not None:
        W = width or sc.camera.W
        H = height or sc.camera.H
        k = W / sc.camera.W
        sc.camera = Camera(W=W, H=H, fx=sc.camera.fx * k, fy=sc.camera.fy * k,
                           cx=(W - 1) / 2.0, cy=(H - 1) / 2.0, znear=sc.camera.znear, zfar=sc.camera.zfar)
    return sc
