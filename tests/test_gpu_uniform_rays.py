"""-m gpu parity tests of the uniform-ray mode (ml_set_ray_mode(ML_RAYS_UNIFORM, seed): every ray an independent
uniform point of the whole shooting rectangle, the literal GPU-D ray generation of PAPER.md:131, :167; reading R20)
against the oracle's ray_mode "uniform" on the same seed: both sides draw the same Philox-4x32-10 numbers from the ray
id, so the four north_star criteria apply ray by ray although the device shoots the rays in another order (sorted into
buckets of the image plane)."""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, lens_disk, lens_masses

from parity_common import (PREC_NAME, check_maps, check_rays, problem_args, report, run_subregions,
                           subregion_tiles)

pytestmark = pytest.mark.gpu

PRECISIONS = [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64]
PREC_IDS = ["fp32_tiled", "fp32_compensated", "fp64"]


@pytest.mark.parametrize("precision", PRECISIONS, ids=PREC_IDS)
def test_c1_uniform_rays_all_four_criteria(precision):
    p = CONFIGS[0]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    seed = 2 ** 41 + 5
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy)
        m.set_ray_mode(ml.ML_RAYS_UNIFORM, seed)
        info = m.info
        assert info["ray_mode"] == ml.ML_RAYS_UNIFORM and info["ray_seed"] == seed and (info["tile_w"], info["tile_h"]) == (128, 63)
        m.shoot()
        gmap, gst = m.counts(), m.stats
        omap, ost = oracle.shoot(*problem_args(p), xy, ray_seed=seed, ray_mode="uniform")
        r = check_maps(p, gmap, gst, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2), ray_seed=seed, ray_mode="uniform")
        ii, jj = np.meshgrid(np.arange(g.n1, dtype=np.int64), np.arange(g.n2, dtype=np.int64))
        r.update(check_rays(p, g, y_g, y_o, precision, rays_ij=(ii, jj), lenses=xy, ray_seed=seed, tile_w=info["tile_w"],
                            ray_mode="uniform", representative=True))
        # the list order inside a bucket follows the atomics, the arithmetic of a ray does not: same bits every time
        m.shoot()
        assert np.array_equal(m.counts(), gmap)
        assert np.array_equal(m.capture_region(0, g.n1, 0, g.n2), y_g, equal_nan=True)
        # another seed is another map; the one-ray-per-cell sampler and the regular grid are other maps too
        m.set_ray_mode(ml.ML_RAYS_UNIFORM, seed + 1)
        m.shoot()
        assert (m.counts() != gmap).mean() > 0.5
        m.set_ray_mode(ml.ML_RAYS_RANDOM, seed)
        m.shoot()
        assert (m.counts() != gmap).mean() > 0.5
        m.set_ray_mode(ml.ML_RAYS_REGULAR)
        m.shoot()
        if precision == ml.ML_PREC_FP64:
            assert np.array_equal(m.counts(), oracle.shoot(*problem_args(p), xy)[0])
        report("C1 whole map, uniform rays, %s" % PREC_NAME[precision], r)


# Sub-regions of C2-C5: 16 rectangles of 512 x 512 ray IDS = 4.19e6 rays each, scattered over the whole rectangle (a few
# rays per bucket: every bucket of the image plane is visited), every ray compared.
@pytest.mark.parametrize("cfg,masses,precision",
                         [(1, False, ml.ML_PREC_FP32_TILED), (2, False, ml.ML_PREC_FP32_TILED), (3, False, ml.ML_PREC_FP32_TILED),
                          (4, True, ml.ML_PREC_FP32_TILED), (3, False, ml.ML_PREC_FP32_COMPENSATED), (1, True, ml.ML_PREC_FP64)],
                         ids=["C2", "C3", "C4", "C5-masses", "C4-compensated", "C2-masses-fp64"])
def test_subregions_uniform_rays(cfg, masses, precision):
    p = CONFIGS[cfg]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    mass = lens_masses(g.n_star, p.seed) if masses else None
    tiles = subregion_tiles(p, g, xy.shape[0])
    seed = 2000 + cfg
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy, mass)
        m.set_ray_mode(ml.ML_RAYS_UNIFORM, seed)
        r = run_subregions(p, m, g, xy, tiles, precision, mass=mass, ray_seed=seed, ray_mode="uniform")
        report("%s sub-regions, uniform rays%s, %s" % (p.name, ", masses" if masses else "", PREC_NAME[precision]), r)


def test_uniform_rays_partition_by_id_and_probe():
    p = CONFIGS[0]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    with ml.MagnificationMap(*problem_args(p)) as m:
        m.set_lenses(xy)
        m.set_ray_mode(ml.ML_RAYS_UNIFORM, 5)
        m.shoot()
        full, st = m.counts(), m.stats
        assert st["rays_shot"] == g.n1 * g.n2 and st["rays_in_map"] == int(full.sum(dtype=np.uint64))
        for t, reg in enumerate([(0, 1000, 0, g.n2), (1000, g.n1, 0, 777), (1000, g.n1, 777, g.n2)]):
            m.shoot_region(*reg, accumulate=(t > 0))
        assert np.array_equal(m.counts(), full)          # regions partition the ray ids; a ray's draw depends on its id only
        assert m.stats["rays_shot"] == g.n1 * g.n2
        ri = np.array([0, 1, g.n1 - 1, 1234, 77, 1234], dtype=np.int64)
        rj = np.array([0, 5, g.n2 - 1, 999, 2000, 999], dtype=np.int64)
        y = m.probe(ri, rj)
        cap = m.capture_region(0, g.n1, 0, g.n2)
        assert np.array_equal(y, cap[rj, ri])
        y_o = oracle.capture_region(*problem_args(p), xy, (1234, 1235, 999, 1000), ray_seed=5, ray_mode="uniform")
        assert np.abs(y[3] - y_o.reshape(2)).max() <= 1e-3 * g.pixel
        m.shoot_region(5, 5, 0, g.n2)                     # empty region: nothing shot, map zeroed
        assert m.stats["rays_shot"] == 0 and not m.counts().any()


def test_no_stars_uniform_rays_are_exact_and_poisson():
    """Without stars both sides evaluate y = c x in fp64: equal maps; and the counts carry Poisson noise:
    index of dispersion 1, where ML_RAYS_RANDOM's one ray per cell stays below 0.5."""
    args = (0.4, 0.0, 0.0, 64, 100.0, 10.0)
    with ml.MagnificationMap(*args) as m:
        m.set_lenses(np.zeros((0, 2)))
        m.set_ray_mode(ml.ML_RAYS_UNIFORM, 5)
        m.shoot()
        a = m.counts()
        m.set_ray_mode(ml.ML_RAYS_RANDOM, 5)
        m.shoot()
        b = m.counts()
    o, _ = oracle.shoot(*args, np.zeros((0, 2)), ray_seed=5, ray_mode="uniform")
    assert np.array_equal(a, o)
    assert abs(a.mean() / 100.0 * 0.36 - 1) < 4 / np.sqrt(a.sum())
    assert abs(a.var(ddof=1) / a.mean() - 1) < 0.09 and b.var(ddof=1) < 0.5 * b.mean()
