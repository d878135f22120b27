"""-m gpu test of the launch split (csrc/microlens.cu: a shoot is a 2-D grid of tiles; regions wider than 2^31 - 1 tile
columns or taller than 65535 tile rows are cut into several launches that continue the same tile raster through
ShootParams::tile_i0 / tile_j0).  No BASELINE config comes near those limits (C5: 2147 x 5725 tiles), so a TEST build of
the same sources with -DML_MAX_GRID_X=7 -DML_MAX_GRID_Y=50 is made here; C1's 20 x 160 tiles then take twelve
launches, and map and statistics must equal the normal build's bit for bit.  The same test build takes
-DML_UNIFORM_LIST_BYTES=4194304: the bucket lists of ML_RAYS_UNIFORM then hold 4 MB, so C1 is shot in many passes over
stripes of bucket rows (the path C4 and C5 take at full size on a 180 GB device)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from paper_1005_5198_b200 import build as mlbuild
from workloads import CONFIGS, lens_disk

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import json, sys
import numpy as np
import paper_1005_5198_b200 as ml
from workloads import CONFIGS, lens_disk
out = sys.argv[1]
p = CONFIGS[0]
res = {"library": ml.library_path()}
for prec in (ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64):
    with ml.MagnificationMap(p.sigma, p.stellar_fraction, p.gamma, p.n_pix, p.n_rays, p.L, precision=prec) as m:
        info = m.info
        m.set_lenses(lens_disk(info["n_star_expected"], info["r_star"], p.seed))
        m.shoot()
        st = m.stats
        np.save("%s/map_%d.npy" % (out, prec), m.counts())
        res[str(prec)] = {k: int(st[k]) for k in ("rays_shot", "rays_in_map", "rays_dropped", "kernel_launches")}
        m.shoot_region(100, 2001, 37, 1999)      # a ragged region: tile_i0 / tile_j0 != 0 with a split
        np.save("%s/reg_%d.npy" % (out, prec), m.counts())
        res[str(prec)]["region_launches"] = int(m.stats["kernel_launches"])
# uniform rays (reading R20): the bucket lists of a call are built in passes over stripes of bucket rows
for prec in (ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP64):
    with ml.MagnificationMap(p.sigma, p.stellar_fraction, p.gamma, p.n_pix, p.n_rays, p.L, precision=prec) as m:
        info = m.info
        m.set_lenses(lens_disk(info["n_star_expected"], info["r_star"], p.seed))
        m.set_ray_mode(ml.ML_RAYS_UNIFORM, 31)
        m.shoot()
        st = m.stats
        np.save("%s/umap_%d.npy" % (out, prec), m.counts())
        res["u%d" % prec] = {k: int(st[k]) for k in ("rays_shot", "rays_in_map", "rays_dropped", "kernel_launches")}
        np.save("%s/ucap_%d.npy" % (out, prec), m.capture_region(5, 700, 11, 400))
json.dump(res, open(out + "/stats.json", "w"))
"""


def _run_child(tmp, lib=None):
    os.makedirs(tmp, exist_ok=True)
    env = dict(os.environ, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
    if lib:
        env["MICROLENS_B200_LIBRARY"] = lib
    else:
        env.pop("MICROLENS_B200_LIBRARY", None)
    r = subprocess.run([sys.executable, "-c", CHILD, tmp], env=env, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    return json.load(open(os.path.join(tmp, "stats.json")))


def test_a_build_with_tiny_grid_limits_reproduces_the_map_bit_for_bit(tmp_path):
    # ML_UNIFORM_FAIL_ALLOCS=2: the first two allocations of the uniform mode's bucket lists "fail", so the run also goes
    # through the retry with half (then a quarter) of the bucket rows per stripe instead of returning ML_ERR_OOM
    lib = mlbuild.build_library(defines=["ML_MAX_GRID_X=7", "ML_MAX_GRID_Y=50", "ML_UNIFORM_LIST_BYTES=4194304",
                                         "ML_UNIFORM_FAIL_ALLOCS=2"],
                                out=str(tmp_path / "libmicrolens_split.so"))
    normal = _run_child(str(tmp_path / "normal"))
    split = _run_child(str(tmp_path / "split"), lib)
    assert split["library"] == lib and normal["library"] != lib
    for prec in ("0", "1", "2"):
        a, b = normal[prec], split[prec]
        assert a["kernel_launches"] == 1 and b["kernel_launches"] == 12      # 20 x 160 tiles in blocks of <= 7 x 50
        assert b["region_launches"] >= 6
        for k in ("rays_shot", "rays_in_map", "rays_dropped"):
            assert a[k] == b[k]
        for name in ("map", "reg"):
            x = np.load(tmp_path / "normal" / ("%s_%s.npy" % (name, prec)))
            y = np.load(tmp_path / "split" / ("%s_%s.npy" % (name, prec)))
            assert np.array_equal(x, y)
    # uniform rays with 4 MB of list memory: C1's 6.5e6 rays (56 MB of lists) go through in stripes of bucket rows, each
    # pass = scatter + maximum + shoot; the map and the captured positions do not change by a bit
    for prec in ("u0", "u2"):
        a, b = normal[prec], split[prec]
        assert a["kernel_launches"] == 3 and b["kernel_launches"] >= 3 * 10
        for k in ("rays_shot", "rays_in_map", "rays_dropped"):
            assert a[k] == b[k]
        for name in ("umap", "ucap"):
            x = np.load(tmp_path / "normal" / ("%s_%s.npy" % (name, prec[1:])))
            y = np.load(tmp_path / "split" / ("%s_%s.npy" % (name, prec[1:])))
            assert np.array_equal(x, y, equal_nan=True)
