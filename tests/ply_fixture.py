"""Test fixture: writes a synthetic scene in the trained-3DGS `point_cloud.ply` layout (inverse activations applied:
log scale, logit opacity; SH rest coefficients channel-major).  Only tests use it; no checkpoint ships with the repo."""
import numpy as np


def property_names(K):
    return (["x", "y", "z", "nx", "ny", "nz", "f_dc_0", "f_dc_1", "f_dc_2"] + [f"f_rest_{i}" for i in range(3 * (K - 1))]
            + ["opacity", "scale_0", "scale_1", "scale_2", "rot_0", "rot_1", "rot_2", "rot_3"])


def write_ply(path, means, scales, quats, opacity, sh):
    n, K = sh.shape[0], sh.shape[1]
    names = property_names(K)
    cols = {"x": means[:, 0], "y": means[:, 1], "z": means[:, 2], "nx": np.zeros(n), "ny": np.zeros(n), "nz": np.zeros(n),
            "opacity": np.log(opacity.astype(np.float64) / (1.0 - opacity.astype(np.float64)))}
    for i in range(3):
        cols[f"scale_{i}"] = np.log(scales[:, i].astype(np.float64))
        cols[f"f_dc_{i}"] = sh[:, 0, i]
        for k in range(1, K):
            cols[f"f_rest_{i * (K - 1) + (k - 1)}"] = sh[:, k, i]
    for i in range(4):
        cols[f"rot_{i}"] = quats[:, i]
    rows = np.stack([np.asarray(cols[nm], dtype=np.float64) for nm in names], axis=1).astype("<f4")
    with open(path, "wb") as f:
        f.write(b"ply\nformat binary_little_endian 1.0\n")
        f.write(f"element vertex {n}\n".encode())
        for nm in names:
            f.write(f"property float {nm}\n".encode())
        f.write(b"end_header\n")
        f.write(rows.tobytes())
    return names
