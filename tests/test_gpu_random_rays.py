"""-m gpu parity tests of the random-ray mode (ml_set_ray_mode(ML_RAYS_RANDOM, seed): GPU-D's random ray
positions; reading R17) against the oracle's ray_mode 1 on the same seed: both sides draw
the same Philox-4x32-10 numbers from the ray id, so the four north_star criteria apply ray by ray."""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, lens_disk, lens_masses, parity_tiles

from parity_common import PREC_NAME, check_maps, check_rays, problem_args, report, run_subregions, subregion_tiles

pytestmark = pytest.mark.gpu

PRECISIONS = [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64]
PREC_IDS = ["fp32_tiled", "fp32_compensated", "fp64"]


@pytest.mark.parametrize("precision", PRECISIONS, ids=PREC_IDS)
def test_c1_random_rays_all_four_criteria(precision):
    p = CONFIGS[0]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    seed = 2 ** 40 + 17
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy)
        m.set_ray_mode(ml.ML_RAYS_RANDOM, seed)
        assert m.info["ray_mode"] == ml.ML_RAYS_RANDOM and m.info["ray_seed"] == seed
        m.shoot()
        gmap, gst = m.counts(), m.stats
        omap, ost = oracle.shoot(*problem_args(p), xy, ray_seed=seed)
        r = check_maps(p, gmap, gst, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2), ray_seed=seed)
        r.update(check_rays(p, g, y_g, y_o, precision))
        # another seed is another map; the regular grid is back after ML_RAYS_REGULAR
        m.set_ray_mode(ml.ML_RAYS_RANDOM, seed + 1)
        m.shoot()
        assert (m.counts() != gmap).mean() > 0.5
        m.set_ray_mode(ml.ML_RAYS_REGULAR)
        m.shoot()
        if precision == ml.ML_PREC_FP64:
            assert np.array_equal(m.counts(), oracle.shoot(*problem_args(p), xy)[0])
        report("C1 whole map, random rays, %s" % PREC_NAME[precision], r)


# Sub-regions of C2-C5 with random rays, 4.19e6 rays each (16 rectangles of 512 x 512), every ray compared.  Masses AND
# random rays together are the hardest combination for the FP32 arithmetic (every ray carries its own offsets and the
# terms are scaled by m_i); on C4 DESIGN.md recommends ML_PREC_FP32_COMPENSATED for it, and that is the mode tested there.
@pytest.mark.parametrize("cfg,masses,precision",
                         [(1, False, ml.ML_PREC_FP32_TILED), (2, True, ml.ML_PREC_FP32_TILED), (3, False, ml.ML_PREC_FP32_TILED),
                          (4, False, ml.ML_PREC_FP32_TILED), (3, True, ml.ML_PREC_FP32_COMPENSATED), (3, False, ml.ML_PREC_FP32_COMPENSATED)],
                         ids=["C2", "C3-masses", "C4", "C5", "C4-masses-compensated", "C4-compensated"])
def test_subregions_random_rays(cfg, masses, precision):
    p = CONFIGS[cfg]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    mass = lens_masses(g.n_star, p.seed) if masses else None
    tiles = subregion_tiles(p, g, xy.shape[0])
    seed = 1000 + cfg
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy, mass)
        m.set_ray_mode(ml.ML_RAYS_RANDOM, seed)
        r = run_subregions(p, m, g, xy, tiles, precision, mass=mass, ray_seed=seed)
        report("%s sub-regions, random rays%s, %s" % (p.name, ", masses" if masses else "", PREC_NAME[precision]), r)


def test_random_rays_partition_invariance_and_probe():
    p = CONFIGS[0]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    with ml.MagnificationMap(*problem_args(p)) as m:
        m.set_lenses(xy)
        m.set_ray_mode(ml.ML_RAYS_RANDOM, 5)
        m.shoot()
        full = m.counts()
        for t, reg in enumerate([(0, 1000, 0, g.n2), (1000, g.n1, 0, 777), (1000, g.n1, 777, g.n2)]):
            m.shoot_region(*reg, accumulate=(t > 0))
        assert np.array_equal(m.counts(), full)          # a ray's draw depends on its id only
        ri = np.array([0, 1, g.n1 - 1, 1234, 77], dtype=np.int64)
        rj = np.array([0, 5, g.n2 - 1, 999, 2000], dtype=np.int64)
        y = m.probe(ri, rj)
        cap = m.capture_region(0, g.n1, 0, g.n2)
        assert np.array_equal(y, cap[rj, ri])
        with pytest.raises(ml.MicrolensError) as e:
            m.set_ray_mode(7, 0)
        assert e.value.code == ml.ML_ERR_INVALID_ARG


def test_no_stars_random_rays_reproduce_eq12_in_the_mean():
    args = (0.4, 0.0, 0.0, 64, 100.0, 10.0)
    with ml.MagnificationMap(*args) as m:
        m.set_lenses(np.zeros((0, 2)))
        m.set_ray_mode(ml.ML_RAYS_RANDOM, 5)
        m.shoot()
        a = m.counts()
    o, _ = oracle.shoot(*args, np.zeros((0, 2)), ray_seed=5)
    assert np.array_equal(a, o)                           # no deflection sum: fp64 on both sides, exact
    assert abs(a.mean() / 100.0 * 0.36 - 1) < 2e-3
