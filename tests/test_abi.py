"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/tgs.h
declares; struct layouts of the Python binding match the header; the product path fails loudly without a
GPU (no CPU fallback); the product package never imports the oracle."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_03390_b200 import build, tgs
    build.build()
    return tgs.lib()


def _declared_functions():
    hdr = open(os.path.join(ROOT, "include", "tgs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(tgs_[a-z_]+)\s*\(", hdr)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2607_03390_b200 import tgs
    names = _declared_functions()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(tgs.EXPORTS) == names


def test_struct_layouts_match_header(lib, tmp_path):
    from paper_2607_03390_b200 import tgs
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "tgs.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu\\n",'
                   "sizeof(tgs_params),sizeof(tgs_stats),offsetof(tgs_stats,n_pairs),offsetof(tgs_stats,ms_stage),"
                   "offsetof(tgs_stats,device_bytes),offsetof(tgs_stats,n_pairs_slab),offsetof(tgs_stats,launches_total),"
                   "offsetof(tgs_params,depth_slabs),offsetof(tgs_params,slab_split));return 0;}\n")
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    assert [int(x) for x in out] == [C.sizeof(tgs.TgsParams), C.sizeof(tgs.TgsStats), tgs.TgsStats.n_pairs.offset,
                                     tgs.TgsStats.ms_stage.offset, tgs.TgsStats.device_bytes.offset, tgs.TgsStats.n_pairs_slab.offset,
                                     tgs.TgsStats.launches_total.offset, tgs.TgsParams.depth_slabs.offset, tgs.TgsParams.slab_split.offset]


def test_defaults_are_the_papers(lib):
    from paper_2607_03390_b200 import tgs
    p = tgs.TgsParams()
    lib.tgs_default_params(C.byref(p))
    # PAPER.md:L99 lambda1 = 3, lambda2 = 0; L142 lambda_TDC = 50, lambda_SR = 5; L128 eta = 40 %
    assert (p.lambda1, p.lambda2, p.lambda_tdc, p.lambda_sr) == (3.0, 0.0, 50, 5) and abs(p.eta - 0.4) < 1e-7
    assert (p.enable_afc, p.enable_toc, p.enable_sr) == (1, 1, 1)
    # R39 exact tile intersection on; R42 ANCHORED priors (the paper, L86); R43 / L142 TGB at full resolution unless asked
    assert (p.exact_tiles, p.prior_policy, p.tgb_downscale) == (1, 0, 1)
    # the number of front-to-back slabs is chosen by the library unless asked
    assert p.depth_slabs == 0 and list(p.slab_split) == [0, 0, 0]
    assert lib.tgs_strerror(tgs.E_NO_PRIORS).decode().startswith("no valid temporal priors")


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2607_03390_b200 import tgs
    with pytest.raises(tgs.TgsError) as ei:
        tgs.Context(0)
    assert ei.value.code == tgs.E_CUDA


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_03390_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "libora" not in txt and "ora.h" not in txt, f
    code = "import sys; import paper_2607_03390_b200; assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)"
    subprocess.run([sys.executable, "-c", code], cwd=ROOT, check=True)


def test_oracle_does_not_import_product():
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2607_03390_b200" not in txt and "from paper_2607_03390_b200" not in txt, f
            assert '"tgs.h"' not in txt and "tgs_internal" not in txt and "libtgs" not in txt, f


def test_synth_is_free_of_both():
    for f in os.listdir(os.path.join(ROOT, "synth")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "synth", f)).read()
            code = "\n".join(l for l in txt.splitlines() if l.lstrip().startswith(("import ", "from ")))
            assert "oracle" not in code and "paper_2607_03390_b200" not in code, f


def test_scene_generators_are_seeded_and_shaped():
    from synth import make_config
    a, b = make_config(1), make_config(1)
    assert a.n == 16384 and a.poses.shape == (8, 4, 4) and a.camera.W == 256 and a.sh.shape == (16384, 1, 3)
    assert np.array_equal(a.means, b.means) and np.array_equal(a.sh, b.sh)
    assert np.abs(a.means).max() < 3.0 and a.modes == ["full"] + ["temporal"] * 7
    c = make_config(2, n=2000, frames=5)
    assert c.sh.shape == (2000, 16, 3) and c.camera.W == 1280 and abs(c.camera.fx - 640 / np.tan(np.radians(30))) < 1e-3
    d = make_config(3, n=5000, frames=300)
    pos = np.stack([-(p[:3, :3].T @ p[:3, 3]) for p in d.poses.astype(np.float64)])
    step = np.linalg.norm(np.diff(pos, axis=0), axis=1)
    assert np.allclose(step, 0.02, atol=2e-4) and np.linalg.norm(pos, axis=1).max() < 6.0
    fw = d.poses[:, 2, :3].astype(np.float64)
    ang = np.degrees(np.arccos(np.clip((fw[1:] * fw[:-1]).sum(1), -1, 1)))
    assert ang.max() <= 0.6 + 1e-3
    e = make_config(5, n=1000, frames=50)
    assert e.sh_degree == 1 and e.sh.shape == (1000, 4, 3) and len(np.unique(e.means[:, 2])) == 10
