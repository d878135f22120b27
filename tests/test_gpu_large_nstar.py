"""-m gpu parity at large lens counts (the paper's cross-over with the tree code sits at
N* ~ 5e4 and its record run used far more).  The kernel streams the fp64 lens array through
shared memory in 512-lens chunks, so nothing limits N* but device memory; the oracle can only afford a few
thousand rays at these counts, shot by both sides into partial maps (reading R16)."""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, lens_disk, lens_masses

from parity_common import check_maps, check_rays, problem_args

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
        r.update(check_rays(p, g, y_g, y_o))
        print("N* = %d%s:" % (n_lenses, " with masses" if masses else ""), r)
