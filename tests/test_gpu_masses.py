"""-m gpu parity tests of unequal lens masses (ml_set_lens_masses; eq. 4 with its m_i) against the
fp64 oracle's *_m variants on the same seeded lenses and masses: the four north_star criteria."""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, lens_disk, lens_masses, parity_tiles

from parity_common import PREC_NAME, check_maps, check_rays, problem_args, report, run_subregions, subregion_tiles

pytestmark = pytest.mark.gpu

PRECISIONS = [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64]
PREC_IDS = ["fp32_tiled", "fp32_compensated", "fp64"]


def field(p, g):
    """Seeded lens field with a mass spectrum: N* = sigma_* R*^2 / <M> lenses (eq. 5)."""
    mean = lens_masses(1000, p.seed).mean()           # the recipe's <M> (about 1)
    n = oracle.n_star(g.kappa_star, g.r_star, mean)
    return lens_disk(n, g.r_star, p.seed), lens_masses(n, p.seed)


@pytest.mark.parametrize("precision", PRECISIONS, ids=PREC_IDS)
def test_c1_with_a_mass_spectrum_all_four_criteria(precision):
    p = CONFIGS[0]
    g = oracle.geometry(*problem_args(p))
    xy, mass = field(p, g)
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy, mass)
        m.shoot()
        gmap, gst = m.counts(), m.stats
        omap, ost = oracle.shoot(*problem_args(p), xy, mass=mass)
        r = check_maps(p, gmap, gst, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2), mass=mass)
        r.update(check_rays(p, g, y_g, y_o, precision))
        # the masses matter: the unit-mass map of the same positions is a different map
        m.set_lenses(xy)
        m.shoot()
        assert (m.counts() != gmap).mean() > 0.5
        report("C1 whole map, masses, %s" % PREC_NAME[precision], r)


@pytest.mark.parametrize("cfg,precision", [(2, ml.ML_PREC_FP32_TILED), (4, ml.ML_PREC_FP32_TILED), (3, ml.ML_PREC_FP32_COMPENSATED)],
                         ids=["C3-fp32_tiled", "C5-fp32_tiled", "C4-fp32_compensated"])
def test_subregions_with_masses(cfg, precision):
    """16 seeded rectangles of 512 x 512 rays, every ray compared (same sample as the unit-mass sub-region test)."""
    p = CONFIGS[cfg]
    g = oracle.geometry(*problem_args(p))
    xy, mass = field(p, g)
    tiles = subregion_tiles(p, g, xy.shape[0])
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy, mass)
        r = run_subregions(p, m, g, xy, tiles, precision, mass=mass)
        report("%s sub-regions, masses, %s" % (p.name, PREC_NAME[precision]), r)


@pytest.mark.parametrize("precision", PRECISIONS, ids=PREC_IDS)
def test_unit_masses_equal_the_unit_mass_kernels_exactly(precision):
    p = CONFIGS[0]
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy)
        m.shoot_region(0, g.n1, 0, 640)
        a = m.counts()
        m.set_lenses(xy, np.ones(xy.shape[0]))          # x * 1.0f is exact: the MASS instantiation must agree bit for bit
        m.shoot_region(0, g.n1, 0, 640)
        assert np.array_equal(a, m.counts())


def test_mass_scaling_law_on_the_device():
    """Lenses of mass 4 at 2 xi with L doubled = unit lenses at xi: every quantity scales by a power of two."""
    rng = np.random.default_rng(5)
    xy = rng.uniform(-4, 4, size=(6, 2))
    with ml.MagnificationMap(0.0, 1.0, 0.0, 64, 16.0, 8.0, precision=ml.ML_PREC_FP64) as m1, \
            ml.MagnificationMap(0.0, 1.0, 0.0, 64, 16.0, 16.0, precision=ml.ML_PREC_FP64) as m4:
        m1.set_lenses(xy)
        m4.set_lenses(2.0 * xy, np.full(6, 4.0))
        m1.shoot()
        m4.shoot()
        assert np.array_equal(m1.counts(), m4.counts()) and m1.stats["rays_in_map"] > 0


def test_bad_masses_are_rejected_and_leave_the_lenses_in_place():
    with ml.MagnificationMap(0.4, 1.0, 0.0, 32, 16.0, 4.0) as m:
        xy = np.array([[0.5, 0.5], [-1.0, 2.0]])
        m.set_lenses(xy, [1.0, 2.0])
        m.shoot()
        a = m.counts()
        for bad in ([1.0, 0.0], [1.0, -2.0], [float("nan"), 1.0], [float("inf"), 1.0]):
            with pytest.raises(ml.MicrolensError) as e:
                m.set_lenses(xy, bad)
            assert e.value.code == ml.ML_ERR_INVALID_ARG
        with pytest.raises(ValueError):
            m.set_lenses(xy, [1.0])
        m.shoot()
        assert np.array_equal(a, m.counts()) and m.info["n_lenses"] == 2
