"""tgs_sort_pairs_static (include/tgs.h): the entry point that allocates nothing -- the path's stable radix sort of (tile id,
Gaussian) pairs with all of its scratch in one static device array -- against the existing path.

The existing path is the tile sort inside tgs_render (k_onesweep with the context's cudaMalloc'ed scratch): its result is the
frame's pair list in tile | depth order (tgs_debug_get "keys" = tile << 32 | bits(depth), "vals" = Gaussian).  The input of that
sort is the same pairs in depth order (ties by Gaussian index, R28), which is rebuilt here from the list itself; sorting it
stably by tile id through the new entry point must give back the existing path's list bit for bit (integer work: no tolerance).

This file is collected last on purpose (pytest -x: a failure here hides nothing behind it), and it passes
both alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_2607_03390_b200 import tgs
from synth import make_config

pytestmark = pytest.mark.gpu


def _existing_path_lists(n_gaussians):
    """Pair lists (tile ids, depth bits, Gaussians) of a FULL frame and of the TEMPORAL frame after it, as the existing path sorted them."""
    sc = make_config(2, n=n_gaussians, frames=3)
    g = tgs.Context(0)
    g.load_scene(sc)
    p = g.default_params()
    p.depth_slabs = 1          # one piece: "keys" / "vals" are the complete lists of the frame
    g.set_params(p)
    out = []
    for f, mode in enumerate([tgs.FULL, tgs.TEMPORAL]):
        g.set_camera(sc.poses[f], sc.camera)
        g.render(mode)
        st = g.get_stats()
        keys, vals = g.debug_get("keys"), g.debug_get("vals")
        assert st["overflow"] == 0 and len(keys) == len(vals) == st["n_pairs"] > 0
        out.append(((keys >> np.uint64(32)).astype(np.uint32), (keys & np.uint64(0xffffffff)).astype(np.uint32), vals, st["n_tiles"]))
    g.destroy()
    return out


def _tile_sort_input(tile, depth_bits, gauss):
    """The pairs in the order the tile sort receives them: by depth, ties by Gaussian index (pairs of one Gaussian lie on different
    tiles, so their mutual order cannot show in the result)."""
    order = np.lexsort((gauss, depth_bits))
    return np.ascontiguousarray(tile[order]), np.ascontiguousarray(gauss[order])


def _dev(a):
    import torch
    return torch.from_numpy(a.view(np.int32).copy()).cuda()


def _host(t):
    return t.cpu().numpy().view(np.uint32)


def _key_bytes(n_tiles):
    bits = max(1, int(n_tiles - 1).bit_length())
    return (bits + 7) // 8


@pytest.mark.parametrize("n_gaussians", [30000, 100000], ids=["small_tiles_instance", "big_tiles_instance"])
def test_static_scratch_sort_reproduces_the_tile_sort_of_the_existing_path_on_calls_in_a_row(n_gaussians):
    import torch
    (tile_a, depth_a, gauss_a, n_tiles), (tile_b, depth_b, gauss_b, _) = _existing_path_lists(n_gaussians)
    assert len(tile_b) < len(tile_a) <= tgs.SORT_STATIC_MAX_ITEMS      # the second call is shorter: stale scratch lies behind its end
    if n_gaussians == 100000:
        assert len(tile_a) > (1 << 18)                                 # the 4096-pair instance
    kb = _key_bytes(n_tiles)
    assert kb == 2                                                     # 3600 tiles: two passes, through the static ping-pong buffers
    ins = [_tile_sort_input(tile_a, depth_a, gauss_a), _tile_sort_input(tile_b, depth_b, gauss_b)]
    want = [(tile_a, gauss_a), (tile_b, gauss_b), (tile_a, gauss_a)]
    d_in = [(_dev(k), _dev(v)) for k, v in ins]
    d_out = [(torch.full((len(w[0]) + 64,), -1, dtype=torch.int32, device="cuda"), torch.full((len(w[0]) + 64,), -1, dtype=torch.int32, device="cuda")) for w in want]
    status = torch.full((3,), 7, dtype=torch.int32, device="cuda")
    # a first call loads the module (its static array is allocated then, by the driver, not by the call); from here on the
    # device's free memory must not move
    tgs.sort_pairs_static(d_in[0][0], d_in[0][1], d_out[0][0], d_out[0][1], len(ins[0][0]), kb, status=status)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # calls in a row on one stream, no synchronisation in between: frame A, the shorter frame B, frame A again
    for i, j in enumerate([0, 1, 0]):
        tgs.sort_pairs_static(d_in[j][0], d_in[j][1], d_out[i][0], d_out[i][1], len(ins[j][0]), kb, status=status[i:])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert _host(status).tolist() == [0, 0, 0]
    for i, (wk, wv) in enumerate(want):
        n = len(wk)
        gk, gv = _host(d_out[i][0]), _host(d_out[i][1])
        assert np.array_equal(gk[:n], wk), f"call {i}: tile ids differ from the existing path at {np.nonzero(gk[:n] != wk)[0][:8]}"
        assert np.array_equal(gv[:n], wv), f"call {i}: Gaussians differ from the existing path at {np.nonzero(gv[:n] != wv)[0][:8]}"
        assert (gk[n:] == 0xffffffff).all() and (gv[n:] == 0xffffffff).all()       # nothing written behind the end
    # the inputs are read only
    assert np.array_equal(_host(d_in[0][0]), ins[0][0]) and np.array_equal(_host(d_in[1][1]), ins[1][1])


@pytest.mark.parametrize("n,key_bytes", [(1, 1), (2049, 1), (5000, 3), ((1 << 18) + 77, 4), (1 << 20, 4), (1 << 20, 3)])
def test_static_scratch_sort_is_the_stable_sort_on_the_low_key_bytes(n, key_bytes):
    """Every number of passes (odd and even: the last pass must land in the caller's buffers), ragged tails, the maximum size."""
    import torch
    rng = np.random.default_rng(1000 + n + key_bytes)
    keys = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(np.uint32)
    keys[: n // 3] &= np.uint32(0x00ff00ff)                             # many equal digits: stability shows
    vals = rng.permutation(n).astype(np.uint32)
    mask = np.uint32((1 << (8 * key_bytes)) - 1) if key_bytes < 4 else np.uint32(0xffffffff)
    order = np.argsort(keys & mask, kind="stable")
    dk, dv = _dev(keys), _dev(vals)
    ok, ov = torch.empty_like(dk), torch.empty_like(dv)
    status = torch.full((1,), 7, dtype=torch.int32, device="cuda")
    for _ in range(2):                                                  # twice in a row into the same outputs
        tgs.sort_pairs_static(dk, dv, ok, ov, n, key_bytes, status=status)
    torch.cuda.synchronize()
    assert int(status[0]) == 0
    assert np.array_equal(_host(ok), keys[order]) and np.array_equal(_host(ov), vals[order])


def test_static_scratch_sort_rejects_what_does_not_fit_and_bad_arguments():
    import torch
    buf = torch.zeros(4096, dtype=torch.int32, device="cuda")
    a, b, c, d = (buf[i * 1024:] for i in range(4))
    with pytest.raises(tgs.TgsError) as ei:
        tgs.sort_pairs_static(a, b, c, d, tgs.SORT_STATIC_MAX_ITEMS + 1, 2)
    assert ei.value.code == tgs.E_INVALID_ARG and "exceeds the maximum of 1048576 items" in str(ei.value)
    for args in [(a, b, c, d, 1024, 0), (a, b, c, d, 1024, 5), (a, b, a, d, 1024, 2), (a, b, c, c, 1024, 2), (a, b, c, None, 1024, 2)]:
        with pytest.raises(tgs.TgsError) as ei:
            tgs.sort_pairs_static(*args)
        assert ei.value.code == tgs.E_INVALID_ARG
    assert tgs.sort_pairs_static(a, b, c, d, 0, 2) == tgs.OK              # nothing to do is not an error
    torch.cuda.synchronize()
    assert int(buf.abs().sum()) == 0
