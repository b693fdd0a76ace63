"""oracle/ply.py -- CPU oracle of the checkpoint loader.  TEST INFRASTRUCTURE ONLY.

Reads a trained-3DGS `point_cloud.ply` (the storage format of the scenes the paper renders; per-Gaussian
mean, scale + rotation -> covariance, opacity, SH: L55) and applies the activations of that format, in float64:

    scale = exp(scale_raw)                opacity = 1 / (1 + exp(-opacity_raw))
    sh[n][k][ch]: k = 0 from f_dc_<ch>;   k >= 1 from f_rest_<ch (K-1) + (k-1)>     (channel-major)
    quaternion (rot_0..3) = (w, x, y, z), left un-normalised (the loader of the scene normalises)

Plain numpy, no shared code with the CUDA path (paper_2607_03390_b200/csrc/tgs_ply.cu).  Pinned in
tests/test_oracle_pins.py by a hand-written file with closed-form values (exp(0) = 1, sigmoid(0) = 1/2,
exp(ln 3) = 3, sigmoid(ln 3) = 3/4) and distinct f_rest values that fix the channel-major order.
"""
from __future__ import annotations

import numpy as np


def read_ply(path):
    """-> dict(means [n,3], scales [n,3], quats [n,4], opacity [n], sh [n,K,3], sh_degree), float32 arrays."""
    with open(path, "rb") as f:
        if f.readline().strip() != b"ply":
            raise ValueError("not a ply file")
        fmt, n, props, in_vertex = None, None, [], False
        while True:
            line = f.readline()
            if not line:
                raise ValueError("header without end_header")
            tok = line.decode("ascii").split()
            if not tok:
                continue
            if tok[0] == "end_header":
                break
            if tok[0] == "format":
                fmt = tok[1]
            elif tok[0] == "element":
                in_vertex = tok[1] == "vertex"
                if in_vertex:
                    n = int(tok[2])
            elif tok[0] == "property" and in_vertex:
                if tok[1] not in ("float", "float32"):
                    raise ValueError("vertex properties must be float32")
                props.append(tok[2])
        if fmt != "binary_little_endian" or not n:
            raise ValueError("unsupported ply")
        rows = np.frombuffer(f.read(4 * n * len(props)), dtype="<f4").reshape(n, len(props)).astype(np.float64)
    col = {name: rows[:, i] for i, name in enumerate(props)}
    n_rest = sum(1 for p in props if p.startswith("f_rest_"))
    K = n_rest // 3 + 1
    deg = int(round(np.sqrt(K))) - 1
    if (deg + 1) ** 2 != K or 3 * (K - 1) != n_rest or not 0 <= deg <= 3:
        raise ValueError("f_rest count fits no SH degree")
    sh = np.zeros((n, K, 3))
    for ch in range(3):
        sh[:, 0, ch] = col[f"f_dc_{ch}"]
        for k in range(1, K):
            sh[:, k, ch] = col[f"f_rest_{ch * (K - 1) + (k - 1)}"]
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return {
        "means": f32(np.stack([col["x"], col["y"], col["z"]], axis=1)),
        "scales": f32(np.exp(np.stack([col["scale_0"], col["scale_1"], col["scale_2"]], axis=1))),
        "quats": f32(np.stack([col["rot_0"], col["rot_1"], col["rot_2"], col["rot_3"]], axis=1)),
        "opacity": f32(1.0 / (1.0 + np.exp(-col["opacity"]))),
        "sh": f32(sh),
        "sh_degree": deg,
    }
