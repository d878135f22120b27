"""-m gpu parity at large lens counts (the paper's cross-over with the tree code sits at
N* ~ 5e4 and its record run used far more).  The kernel streams the fp64 lens array through
shared memory in 512-lens chunks, so nothing limits N* but device memory; the oracle can only afford a few
thousand rays at these counts, shot by both sides into partial maps (reading R16)."""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, lens_disk, lens_masses

from parity_common import check_maps, check_rays, problem_args, report

pytestmark = pytest.mark.gpu


# The FP32 rounding of 1e6 terms random-walks to ~1e-3 pixel at C4's pixel size (measured: default mode 1.04e-3 px max,
# compensated mode 5.2e-4, fp64 4e-10): from N* ~ 5e5 up the compensated or fp64 mode is the one that meets the
# 1e-3-pixel criterion, and that is what the 1e6 case asserts.
@pytest.mark.parametrize("n_lenses,masses,precision",
                         [(100_003, False, ml.ML_PREC_FP32_TILED), (1_000_001, False, ml.ML_PREC_FP32_COMPENSATED),
                          (1_000_001, False, ml.ML_PREC_FP64), (250_007, True, ml.ML_PREC_FP32_TILED)],
                         ids=["1e5", "1e6-compensated", "1e6-fp64", "2.5e5-masses"])
def test_large_lens_counts_match_the_oracle(n_lenses, masses, precision):
    p = CONFIGS[3]                                     # C4 geometry (a1 = 120 R_E), lens count overridden
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(n_lenses, g.r_star, 11)
    mass = lens_masses(n_lenses, 11) if masses else None
    rays = 64 if n_lenses > 500_000 else 160           # oracle budget: <= 4e9 interactions
    i0, j0 = g.n1 // 2 - 777, g.n2 // 2 + 1234         # not aligned to the 128 x 16 kernel tiles
    reg = (i0, i0 + rays, j0, j0 + rays)
    with ml.MagnificationMap(*problem_args(p), precision=precision) as m:
        m.set_lenses(xy, mass)
        m.shoot_region(*reg)
        omap, ost = oracle.shoot_region(*problem_args(p), xy, region=reg, mass=mass)
        assert m.stats["interactions"] == rays * rays * n_lenses
        r = check_maps(p, m.counts(), m.stats, omap, ost)
        y_g = m.capture_region(*reg)
        y_o = oracle.capture_region(*problem_args(p), xy, reg, mass=mass)
        r.update(check_rays(p, g, y_g, y_o, precision))
        report("C4 geometry, N* = %d%s, mode %d, %d x %d rays" % (n_lenses, " with masses" if masses else "", precision, rays, rays), r)


def test_few_rays_many_lenses_split_the_lens_loop_over_ctas():
    """SURVEY.md 8(f) item 4, second clause: ml_probe / ml_capture_region / a small ml_shoot_region
    at N* = 1e6 must not leave the GPU idle -- with fewer tiles than SMs the lens loop is split over CTAs (lens ranges
    of whole 512-lens chunks, fp64 partial sums added in range order).  Checked: the split launches have >= 100 CTAs
    (ml_stats.capture_ctas), positions match the oracle, and they equal the unsplit path's up to the regrouping of the
    fp64 additions."""
    p = CONFIGS[3]
    g = oracle.geometry(*problem_args(p))
    n_lenses = 1_000_003
    xy = lens_disk(n_lenses, g.r_star, 12)
    rng = np.random.default_rng(77)
    with ml.MagnificationMap(*problem_args(p), precision=ml.ML_PREC_FP32_COMPENSATED) as m:
        m.set_lenses(xy)
        # 40 rays in 40 different tiles: split
        ri = rng.integers(0, g.n1, 40).astype(np.int64)
        rj = rng.integers(0, g.n2, 40).astype(np.int64)
        y_split = m.probe(ri, rj)
        assert m.stats["capture_ctas"] >= 100
        y_o = oracle.probe(*problem_args(p), xy, ri, rj)
        r = check_rays(p, g, y_split, y_o, ml.ML_PREC_FP32_COMPENSATED)
        # the same 40 rays inside a list of 1000 rays (1000 tiles: one CTA per tile walks every lens, no split)
        ri2 = np.concatenate([ri, rng.integers(0, g.n1, 960)]).astype(np.int64)
        rj2 = np.concatenate([rj, rng.integers(0, g.n2, 960)]).astype(np.int64)
        y_whole = m.probe(ri2, rj2)
        assert m.stats["capture_ctas"] == 0
        assert np.abs(y_split - y_whole[:40]).max() <= 1e-11 * np.abs(y_whole[:40]).max()
        r2 = check_rays(p, g, y_whole, oracle.probe(*problem_args(p), xy, ri2, rj2), ml.ML_PREC_FP32_COMPENSATED)
        # a small region binned through the same split path equals the oracle's partial map
        i0, j0 = g.n1 // 3 + 5, g.n2 // 3 + 7
        reg = (i0, i0 + 48, j0, j0 + 48)
        m.shoot_region(*reg)
        assert m.stats["capture_ctas"] >= 100 and m.stats["interactions"] == 48 * 48 * n_lenses
        omap, ost = oracle.shoot_region(*problem_args(p), xy, region=reg)
        r3 = check_maps(p, m.counts(), m.stats, omap, ost)
        report("C4 geometry, N* = 1000003, compensated: 40-ray probe (split)", r)
        report("C4 geometry, N* = 1000003, compensated: 1000-ray probe (one CTA per tile)", r2)
        report("C4 geometry, N* = 1000003, compensated: 48 x 48-ray region binned through the split path", r3)
