"""Helpers of the GPU parity tests: drive the CUDA path (through the C-ABI binding) and the oracle on the
same seeded inputs and compare them element by element.

Tolerances (BASELINE.json north_star; derivation in DESIGN.md §5):
  integers (flags, rects, pair counts, sorted keys and values, ranges, tile masks, warped-pixel hits): bit-exact;
  decision floats (u, v, d, conic, warped depth/sigma, repaired depth): bit-exact (same fp32 operation order);
  RGB: max abs error <= 2e-3; depth: <= 1e-4 relative; sigma: <= 2e-3 * depth (sqrt of an fp32 cancellation);
  pixels the oracle marks `borderline` (an alpha or transmittance test within its rounding margin) may take
  the other branch: there RGB <= 6e-3 (measured <= 3.8e-3) and their share is bounded per test (measured <= 1.42 %).
"""
import json
import os

import numpy as np

from oracle import ora
from oracle.ora import Oracle
from paper_2607_03390_b200 import tgs

RGB_TOL = 2e-3                 # north_star: max abs error per RGB channel
RGB_GUARD_OFF_BORDER = 1e-3    # regression guard below north_star's bound: worst measured 5.2e-4 (one pixel under needle-like splats, whose
                               # exponent is ill-conditioned in fp32, R36); 1.9e-5 on every other test frame
DEPTH_RTOL = 1e-4              # north_star: relative depth
SIGMA_TOL_REL_DEPTH = 2e-3     # the builder's own (north_star states none): sigma is the square root of an fp32 cancellation
BORDERLINE_RGB_TOL = 6e-3      # pixels whose skip / stop decision is within its rounding margin (worst measured: 3.8e-3)
BORDER_MAX_DEFAULT = 2.5e-2    # share of such pixels (worst measured on any test frame: 1.42 %)

MODE_G = {"full": tgs.FULL, "pseudo": tgs.PSEUDO_REF, "temporal": tgs.TEMPORAL, "auto": tgs.AUTO}
MODE_O = {"full": ora.FULL, "pseudo": ora.PSEUDO_REF, "temporal": ora.TEMPORAL, "auto": ora.AUTO}


GPU_ONLY_PARAMS = ("max_pairs", "depth_slabs", "slab_split")     # how the CUDA path organises its work, not what it computes


def make_pair(sc, params=None):
    """A CUDA context and an oracle on the same scene and parameters.  depth_slabs defaults to 1 here (one piece: the pair
    lists are the complete lists of L61 and are compared bit for bit); the slab tests set it explicitly."""
    g = tgs.Context(0)
    o = Oracle()
    g.load_scene(sc)
    o.load_scene(sc)
    params = dict(params or {})
    params.setdefault("depth_slabs", 1)
    pg, po = g.default_params(), o.default_params()
    for k, v in params.items():
        if k == "bg":
            for i in range(3):
                pg.bg[i] = v[i]
                po.bg[i] = v[i]
        elif k == "slab_split":
            for i, x in enumerate(v):
                pg.slab_split[i] = x
        else:
            setattr(pg, k, v)
            if k not in GPU_ONLY_PARAMS:
                setattr(po, k, v)
    g.set_params(pg)
    o.set_params(po)
    return g, o


def inject_priors(g, o):
    """Feed the oracle's priors to the CUDA context so that an S / P frame starts from identical inputs."""
    g.debug_put("prior_depth", o.get("prior_depth"))
    g.debug_put("prior_sigma", o.get("prior_sigma"))
    g.debug_put("prior_image", o.get("prior_image"))
    g.debug_put("rendered", o.get("rendered"))
    g.debug_put("F", o.get("F"))
    g.debug_put("prior_view", o.get("prior_view"))


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


def compare_records(g, o, n, pairs=True):
    rec = o.get("records")
    fl_g = g.debug_get("rec_flags")
    assert np.array_equal(fl_g, rec["flags"]), f"flags differ at {np.nonzero(fl_g != rec['flags'])[0][:10]}"
    vis = (rec["flags"] & ora.VISIBLE) != 0
    uvdo = g.debug_get("rec_uvdo").reshape(n, 4)
    conic = g.debug_get("rec_conic").reshape(n, 4)
    rect = g.debug_get("rec_rect").reshape(n, 4)
    for j, name in enumerate(("u", "v", "d", "o")):
        assert np.array_equal(bits(uvdo[vis, j]), bits(rec[name][vis])), name
    for j, name in enumerate(("A", "B", "C", "tau")):
        assert np.array_equal(bits(conic[vis, j]), bits(rec[name][vis])), name
    for j, name in enumerate(("x_lo", "x_hi", "y_lo", "y_hi")):
        assert np.array_equal(rect[vis, j], rec[name][vis]), name
    if pairs:
        tt = g.debug_get("tiles_touched")
        assert np.array_equal(tt, rec["tiles_touched"])
    col = rec["tiles_touched"] > 0
    rgb = g.debug_get("rec_rgb").reshape(n, 4)[:, :3]
    ref = np.stack([rec["r"], rec["g"], rec["b"]], 1)
    np.testing.assert_allclose(rgb[col], ref[col], atol=2e-5)
    return rec


def compare_binning(g, o):
    keys_o, vals_o, ranges_o = o.get("keys"), o.get("vals"), o.get("ranges")
    keys_g, vals_g, ranges_g = g.debug_get("keys"), g.debug_get("vals"), g.debug_get("ranges")
    assert len(keys_g) == len(keys_o)
    assert np.array_equal(keys_g, keys_o)
    assert np.array_equal(vals_g, vals_o)
    assert np.array_equal(ranges_g, ranges_o)


def compare_temporal_buffers(g, o):
    wd_o, ws_o, fd_o = o.get("warp_depth"), o.get("warp_sigma"), o.get("fill_depth")
    assert np.array_equal(bits(g.debug_get("warp_depth")), bits(wd_o))
    assert np.array_equal(bits(g.debug_get("warp_sigma")), bits(ws_o))
    assert np.array_equal(bits(g.debug_get("fill_depth")), bits(fd_o))


def compare_outputs(g, o, ftype, border_max=BORDER_MAX_DEFAULT, border_rgb_tol=BORDERLINE_RGB_TOL):
    """Float outputs.  north_star's tolerance (RGB <= 2e-3, depth <= 1e-4 relative) holds on every pixel the oracle does
    not flag `borderline`; flagged pixels (a skip / stop decision within its rounding margin, R38) may take the
    other branch: there RGB <= `border_rgb_tol`, and their share must stay below `border_max`.  Returns what was
    measured, so that the tests can print it and assert per-config bounds (DESIGN.md §5 has the table)."""
    img_g, img_o = g.read_image(), o.read_image()
    d_g, s_g = g.read_depth()
    d_o, s_o = o.read_depth()
    border = o.get("borderline").reshape(d_o.shape).astype(bool)
    err = np.abs(img_g - img_o).max(-1)
    m = {"border_share": float(border.mean()), "rgb_max_off_border": float(err[~border].max()) if (~border).any() else 0.0,
         "rgb_max_on_border": float(err[border].max()) if border.any() else 0.0,
         "border_over_2e-3_share": float((err[border] > RGB_TOL).mean()) if border.any() else 0.0,
         "depth_rel_max": 0.0, "sigma_err_max_rel_depth": 0.0}
    assert m["border_share"] <= border_max, m   # T parks just above 1e-4 behind two near-opaque Gaussians
    assert m["rgb_max_off_border"] <= RGB_TOL, m
    assert m["rgb_max_off_border"] <= RGB_GUARD_OFF_BORDER, m
    assert m["rgb_max_on_border"] <= border_rgb_tol, m
    ok = ~border
    vg, vo = d_g < 1e38, d_o < 1e38
    assert np.array_equal(vg[ok], vo[ok])
    both = vg & vo & ok
    if both.any():
        rel = np.abs(d_g[both] - d_o[both]) / d_o[both]
        m["depth_rel_max"] = float(rel.max())
        assert rel.max() <= DEPTH_RTOL, m
        serr = np.abs(s_g[both] - s_o[both]) / d_o[both]
        m["sigma_err_max_rel_depth"] = float(serr.max())
        assert serr.max() <= SIGMA_TOL_REL_DEPTH, m
    return m


def compare_rendered(g, o):
    """G_rendered: must contain every Gaussian the oracle surely blended and none it surely did not."""
    r_g = g.debug_get("rendered").astype(bool)
    sure, maybe = o.get("rendered_sure").astype(bool), o.get("rendered_maybe").astype(bool)
    assert not np.any(sure & ~r_g), np.nonzero(sure & ~r_g)[0][:10]
    assert not np.any(r_g & ~maybe), np.nonzero(r_g & ~maybe)[0][:10]
    return int((r_g != o.get("rendered").astype(bool)).sum())


STAT_KEYS = ("frame_type", "n_total", "n_near", "n_afc", "n_toc", "n_degenerate", "n_empty", "n_visible", "n_newly_visible",
             "n_pairs", "n_tiles", "n_sel_oc", "n_sel_um", "n_sel")


def compare_stats(g, o, pairs=True):
    sg, so = g.get_stats(), o.stats()
    for k in STAT_KEYS:
        if k == "n_pairs" and not pairs:
            continue
        assert sg[k] == so[k], (k, sg[k], so[k])
    return sg, so


REPORT = []          # one dict per compared frame (printed by the tests; `pytest -rP` or -s shows it)


def compare_frame(g, o, n, ftype, check_rendered=True, label=None, **tol):
    """Everything of one frame, both sides already rendered."""
    sg, so = compare_stats(g, o)
    if ftype == ora.FRAME_S:
        compare_temporal_buffers(g, o)
    assert np.array_equal(g.read_tile_mask(), o.read_tile_mask())
    compare_records(g, o, n)
    compare_binning(g, o)
    out = compare_outputs(g, o, ftype, **tol)
    if ftype != ora.FRAME_S and check_rendered:
        out["rendered_diff"] = compare_rendered(g, o)
        out["rendered"] = int(so["n_rendered"])
    out.update(frame="RPS"[ftype], label=label, n_pairs=int(sg["n_pairs"]), n_sel=int(sg["n_sel"]), n_tiles=int(sg["n_tiles"]))
    REPORT.append(out)
    print("[parity] " + " ".join(f"{k}={v:.3g}" if isinstance(v, float) else f"{k}={v}" for k, v in out.items()))
    path = os.environ.get("TGS_PARITY_REPORT")
    if path:
        with open(path, "a") as f:
            f.write(json.dumps(out) + "\n")
    return sg, so, out


def compare_frame_slabs(g, o, n, ftype, label=None, **tol):
    """A frame rendered in several front-to-back slabs (tgs_params.depth_slabs > 1): everything of compare_frame except the
    pair lists, which lack the pairs of tiles that had finished in an earlier slab.  That no NEEDED pair is missing is
    what the image, depth, sigma and G_rendered comparisons check; the counts must add up."""
    sg, so = compare_stats(g, o, pairs=False)
    assert sg["n_slabs"] > 1 and sum(sg["n_pairs_slab"][: sg["n_slabs"]]) == sg["n_pairs"] <= so["n_pairs"]
    if ftype == ora.FRAME_S:
        compare_temporal_buffers(g, o)
    assert np.array_equal(g.read_tile_mask(), o.read_tile_mask())
    compare_records(g, o, n, pairs=False)
    out = compare_outputs(g, o, ftype, **tol)
    if ftype != ora.FRAME_S:
        out["rendered_diff"] = compare_rendered(g, o)
    out.update(frame="RPS"[ftype], label=label, n_pairs=int(sg["n_pairs"]), n_pairs_oracle=int(so["n_pairs"]), n_slabs=int(sg["n_slabs"]),
               n_sel=int(sg["n_sel"]), n_tiles=int(sg["n_tiles"]))
    REPORT.append(out)
    print("[parity] " + " ".join(f"{k}={v:.3g}" if isinstance(v, float) else f"{k}={v}" for k, v in out.items()))
    path = os.environ.get("TGS_PARITY_REPORT")
    if path:
        with open(path, "a") as f:
            f.write(json.dumps(out) + "\n")
    return sg, so, out
