"""-m gpu parity tests: the CUDA library, called through its C ABI, against the fp64 CPU
oracle on the same seeded inputs (BASELINE.json:north_star criteria):

  1. source-plane positions of sampled rays within 1e-3 pixel widths,
  2. >= 99.99 % of rays in the oracle's pixel,
  3. total in-map counts within 1e-5 relative,
  4. |mu_gpu - mu_oracle| <= 1e-3 on 8x8-block averages,

on C1 whole, on seeded sub-regions of C2-C5 (the oracle would need hours for their full
maps: SURVEY.md section 8(c) "parity ladder"), and at C2's full size
in the launch configuration bench.py times (sampled rays + invariants).
"""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, lens_disk, parity_tiles, probe_rays

from parity_common import (PREC_NAME, check_maps, check_rays, make_pair, oracle_subregions, problem_args, report,
                           run_subregions, subregion_tiles)

pytestmark = pytest.mark.gpu

PRECISIONS = [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64]
PREC_IDS = ["fp32_tiled", "fp32_compensated", "fp64"]


@pytest.mark.parametrize("precision", PRECISIONS, ids=PREC_IDS)
def test_c1_whole_map_all_four_criteria(precision):
    p = CONFIGS[0]
    m, g, xy = make_pair(p, precision)
    with m:
        m.shoot()
        gmap, gst = m.counts(), m.stats
        omap, ost = oracle.shoot(*problem_args(p), xy)
        # golden integers of the C1 worked example (oracle side; SURVEY.md 8(c) pin (e))
        assert ost["rays_shot"] == 6553600 and ost["rays_in_map"] == 4012112
        r = check_maps(p, gmap, gst, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2))
        r.update(check_rays(p, g, y_g, y_o, precision))
        # the shoot and capture instantiations run the same arithmetic: binning the captured positions (oracle's floor
        # rule) reproduces the device map -- up to exact ties.  FP32 partial sums make y lattice-valued (spacing ~2^-26
        # R_E), pixel edges are lattice points, so about one ray in 1e7 sits EXACTLY on an edge; the device floors the
        # pixel coordinate u = fma(-S, n_pix/L, fma(x, c n_pix/L, n_pix/2)) and the oracle rule floors (y + L/2)/pixel,
        # which may resolve such a tie to either side (the reason the criterion is 99.99 %, not 100 %).
        pix = oracle.pixels_of(*problem_args(p), y_g).ravel()
        rebinned = np.bincount(pix[pix >= 0], minlength=p.n_pix * p.n_pix).reshape(p.n_pix, p.n_pix)
        assert int(rebinned.sum()) == int(gmap.sum(dtype=np.uint64))
        assert int(np.abs(rebinned.astype(np.int64) - gmap.astype(np.int64)).sum()) <= 8   # <= 4 tied rays of 6.5e6
        if precision == ml.ML_PREC_FP64:
            assert r["same_pixel"] >= 0.999999
        report("C1 whole map %s" % PREC_NAME[precision], r)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4], ids=["C2", "C3", "C4", "C5"])
@pytest.mark.parametrize("precision", PRECISIONS, ids=PREC_IDS)
def test_subregions_all_four_criteria(cfg, precision):
    """C2-C5: 16 seeded rectangles of 512 x 512 rays (4.19e6 rays per config), every ray compared."""
    p = CONFIGS[cfg]
    m, g, xy = make_pair(p, precision)
    with m:
        tiles = subregion_tiles(p, g, xy.shape[0])
        r = run_subregions(p, m, g, xy, tiles, precision)
        assert r["rays"] >= 4000000 or len(tiles) < 16
        report("%s sub-regions %s" % (p.name, PREC_NAME[precision]), r)


@pytest.mark.parametrize("cfg", [2, 3], ids=["C3", "C4"])
@pytest.mark.parametrize("precision", [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED], ids=["fp32_tiled", "fp32_compensated"])
def test_unsplit_launch_at_large_nstar(cfg, precision):
    """The launch bench.py times on C3 / C4: at N* >= 8192 a region of fewer than 2 x 148 tiles has its lens loop split
    over CTAs (capture instantiation + combine kernel), so the 512 x 512-ray rectangles above (<= 165 tiles) never run
    the unsplit shoot instantiation with its fused binning epilogue there.  One seeded rectangle of 1024 x 1024 rays
    (>= 8 x 64 = 512 tiles) does: all four criteria, every ray compared."""
    p = CONFIGS[cfg]
    m, g, xy = make_pair(p, precision)
    assert xy.shape[0] >= 8192
    with m:
        reg = parity_tiles(g.n1, g.n2, 6, 1024, p.seed + 7)[5]   # an interior rectangle, not aligned to the tile grid
        m.shoot_region(*reg)
        st = m.stats
        assert st["capture_ctas"] == 0 and st["kernel_launches"] == 1, st   # one launch of the shoot kernel, no lens split
        r = run_subregions(p, m, g, xy, [reg], precision)
        assert m.stats["capture_ctas"] == 0                                 # the capture of the same rectangle: unsplit too
        assert r["rays"] == 1024 * 1024
        report("%s one 1024 x 1024-ray rectangle, unsplit launch, %s" % (p.name, PREC_NAME[precision]), r)


@pytest.mark.parametrize("cfg", [2, 3, 4], ids=["C3", "C4", "C5"])
@pytest.mark.parametrize("precision", [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED], ids=["fp32_tiled", "fp32_compensated"])
def test_representative_ray_sample(cfg, precision):
    """The sub-rectangles above are sixteen patches of the image plane: they hold a lens or they do not.  Here 250 000
    rays are drawn uniformly over the WHOLE grid and probed one by one, so close passages of lenses occur at their true
    rate (reading R21: the rays judged by the close-passage bound are capped at a fixed 1e-4 of the sample)."""
    p = CONFIGS[cfg]
    m, g, xy = make_pair(p, precision)
    with m:
        ri, rj = probe_rays(g.n1, g.n2, 250000, p.seed + 50)
        y_g = m.probe(ri, rj)
        y_o = oracle.probe(*problem_args(p), xy, ri, rj)
        r = check_rays(p, g, y_g, y_o, precision, rays_ij=(ri, rj), lenses=xy, tile_w=m.info["tile_w"], representative=True)
        report("%s representative sample (250 000 probed rays) %s" % (p.name, PREC_NAME[precision]), r)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4], ids=["C2", "C3", "C4", "C5"])
def test_full_size_bench_configuration(cfg):
    """Every BASELINE config at full size (C2 8.4e9, C3 3.0e9, C4 1.2e10, C5 rays), exactly what bench.py launches:
    invariants that hold at any size, 200 000 rays probed over the whole grid that the oracle computes one by one, and
    one rectangle re-shot alone and compared with the oracle's partial map (north_star: "on all 5 configs")."""
    p = CONFIGS[cfg]
    m, g, xy = make_pair(p)
    with m:
        m.shoot()
        st, gmap = m.stats, m.counts()
        assert st["rays_shot"] == g.n1 * g.n2
        assert st["interactions"] == g.n1 * g.n2 * xy.shape[0]
        assert int(gmap.sum(dtype=np.uint64)) == st["rays_in_map"]
        assert st["rays_dropped"] == 0 and st["capture_ctas"] == 0
        # mean magnification within the sanity band of SURVEY.md 8(c) pin (d)
        ratio = gmap.mean() / p.n_rays / abs(g.mu_th)
        assert 0.88 <= ratio <= 1.12, ratio
        ri, rj = probe_rays(g.n1, g.n2, 200000, p.seed)
        y_g = m.probe(ri, rj)
        y_o = oracle.probe(*problem_args(p), xy, ri, rj)
        r = check_rays(p, g, y_g, y_o, rays_ij=(ri, rj), lenses=xy, tile_w=m.info["tile_w"], representative=True)
        # a sub-rectangle shot alone equals its share of the full run bit for bit: compare
        # the oracle's partial map with the device's on the same region
        if cfg == 1:
            reg = (40000, 40700, 50000, 50900)
            omap, ost = oracle.shoot_region(*problem_args(p), xy, region=reg)
        else:   # 1024 x 1024 rays: enough tiles that the lens loop is not split (the oracle's side is shared with
            reg = parity_tiles(g.n1, g.n2, 6, 1024, p.seed + 7)[5]   # test_unsplit_launch_at_large_nstar through the cache)
            _, omap, ost = oracle_subregions(p, g, xy, [reg])
        m.shoot_region(*reg)
        r.update(check_maps(p, m.counts(), m.stats, omap, ost))
        r.update(mean_mu_over_theory=float(ratio))
        report("%s full size (bench launch), 200000 probed rays + one re-shot rectangle" % p.name, r)
