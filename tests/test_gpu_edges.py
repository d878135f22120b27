"""-m gpu edge cases of the C-ABI hot path, each against the fp64 oracle or an invariant:
no lenses, one lens, lens counts around the staging chunk, empty / single-ray / ragged
regions, partition invariance, a ray sitting on a lens, caller-owned map + stream."""
import ctypes as C

import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import CONFIGS, Problem, lens_disk, lens_masses

from parity_common import check_maps, check_rays, make_pair, problem_args

pytestmark = pytest.mark.gpu

ALL = [ml.ML_PREC_FP32_TILED, ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64]
SMALL = Problem("S", 0.45, 0.1, 1.0, 8.0, 64, 36.0, 11)


@pytest.mark.parametrize("precision", ALL)
@pytest.mark.parametrize("sg", [(0.4, 0.0), (0.6, 0.2), (0.8, 0.3)])
def test_no_lenses_uniform_map_equals_oracle_exactly(precision, sg):
    """n = 0: y = (1 -/+ gamma - sigma) x in fp64 on both sides (eq.12 case)."""
    p = Problem("U", sg[0], sg[1], 0.0, 10.0, 64, 100.0, 0)
    m, g, _ = make_pair(p, precision, lenses=np.zeros((0, 2)))
    with m:
        m.shoot()
        omap, ost = oracle.shoot(*problem_args(p), np.zeros((0, 2)))
        gmap = m.counts()
        check_maps(p, gmap, m.stats, omap, ost)
        # identical up to rays that sit on a pixel edge to within 1 ulp
        assert (gmap != omap).sum() <= 2 * p.n_pix
        mean = gmap.mean() / p.n_rays
        assert abs(mean / abs(g.mu_th) - 1.0) < 0.02


@pytest.mark.parametrize("precision", ALL)
def test_single_lens_at_origin(precision):
    p = Problem("P", 0.0, 0.0, 1.0, 10.0, 128, 100.0, 0)
    lens = np.array([[0.0, 0.0]])
    m, g, xy = make_pair(p, precision, lenses=lens)
    with m:
        m.shoot()
        omap, ost = oracle.shoot(*problem_args(p), xy)
        assert ost["rays_shot"] == 2359296 and ost["rays_in_map"] == 1738304  # SURVEY.md 8(c) pin (b)
        check_maps(p, m.counts(), m.stats, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2))
        check_rays(p, g, y_g, y_o, precision)


@pytest.mark.parametrize("n", [1, 2, 7, 8, 9, 63, 64, 65, 511, 512, 513, 1025, 1536])
def test_lens_counts_around_tile_and_flush_boundaries(n):
    p = SMALL
    # n lenses at the problem's own surface density: disk radius sqrt(n / kappa_*) (eq.5)
    xy = lens_disk(n, (n / (p.sigma * p.stellar_fraction)) ** 0.5, 100 + n)
    m, g, xy = make_pair(p, lenses=xy)
    with m:
        m.shoot()
        omap, ost = oracle.shoot(*problem_args(p), xy)
        check_maps(p, m.counts(), m.stats, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2))
        check_rays(p, g, y_g, y_o)


@pytest.mark.parametrize("precision", [ml.ML_PREC_FP32_COMPENSATED, ml.ML_PREC_FP64])
@pytest.mark.parametrize("masses,random_rays", [(False, False), (True, False), (False, True), (True, True)],
                         ids=["plain", "masses", "random", "masses+random"])
@pytest.mark.parametrize("n", [1, 9, 15, 16, 17, 65, 512, 513, 1025])
def test_lens_count_boundaries_in_the_other_kernel_instantiations(n, masses, random_rays, precision):
    """The same boundaries (flush groups of 8 / 16 / 64 lenses, 512-lens chunks, odd counts with a padding lens) in the
    Newton-refined pipe kernel, the fp64 kernel and their MASS / RANDOM instantiations; the default mode with masses and
    random rays is covered by test_gpu_masses.py / test_gpu_random_rays.py."""
    p = SMALL
    xy = lens_disk(n, (n / (p.sigma * p.stellar_fraction)) ** 0.5, 100 + n)
    mass = lens_masses(n, 200 + n) if masses else None
    seed = 31 + n if random_rays else None
    m, g, xy = make_pair(p, precision, lenses=xy)
    with m:
        m.set_lenses(xy, mass)
        if random_rays:
            m.set_ray_mode(ml.ML_RAYS_RANDOM, seed)
        m.shoot()
        omap, ost = oracle.shoot(*problem_args(p), xy, mass=mass, ray_seed=seed)
        check_maps(p, m.counts(), m.stats, omap, ost)
        y_g = m.capture_region(0, g.n1, 0, g.n2)
        y_o = oracle.capture_region(*problem_args(p), xy, (0, g.n1, 0, g.n2), mass=mass, ray_seed=seed)
        info = m.info
    # This problem has coarse rays (delta = 0.021 R_E, tile half-width T = 64 delta = 1.3 R_E), so in the FP32 modes a
    # handful of rays that pass close to a lens exceed 1e-3 pixel by the rounding of their tile-local coordinates: reading
    # R15, parity_common.close_passage_bound.  check_rays excuses those rays, and only those, from the position criterion
    # (each must stay inside the bound of its nearest lens; ML_PREC_FP64 excuses nothing); the same-pixel criterion
    # applies to every ray.
    jj, ii = np.meshgrid(np.arange(g.n2, dtype=np.int64), np.arange(g.n1, dtype=np.int64), indexing="ij")
    r = check_rays(p, g, y_g, y_o, precision, rays_ij=(ii, jj), lenses=xy, mass=mass, ray_seed=seed, tile_w=info["tile_w"])
    assert r["rays_excused_close_passage"] <= 3


@pytest.mark.parametrize("precision", ALL)
def test_regions_empty_single_ray_ragged_and_partition_invariance(precision):
    p = SMALL
    m, g, xy = make_pair(p, precision)
    with m:
        m.shoot()
        full, full_stats = m.counts().copy(), m.stats
        assert full_stats["rays_shot"] == g.n1 * g.n2
        # empty regions
        m.shoot_region(5, 5, 0, g.n2)
        assert m.stats["rays_shot"] == 0 and m.counts().sum() == 0
        m.shoot_region(0, g.n1, 7, 7)
        assert m.stats["rays_shot"] == 0
        # a single ray: lands where the oracle says
        i, j = g.n1 // 3, g.n2 // 5
        m.shoot_region(i, i + 1, j, j + 1)
        omap, ost = oracle.shoot_region(*problem_args(p), xy, region=(i, i + 1, j, j + 1))
        assert m.stats["rays_shot"] == 1 and np.array_equal(m.counts(), omap)
        # a ragged partition (cuts not aligned to any tile) reproduces the full map bit for bit
        ci = [0, 1, 130, 131, 389, g.n1 - 1, g.n1]
        cj = [0, 33, 34, 250, g.n2 - 3, g.n2]
        first = True
        for a in range(len(ci) - 1):
            for b in range(len(cj) - 1):
                m.shoot_region(ci[a], ci[a + 1], cj[b], cj[b + 1], accumulate=not first)
                first = False
        assert np.array_equal(m.counts(), full)
        st = m.stats
        assert st["rays_shot"] == full_stats["rays_shot"] and st["rays_in_map"] == full_stats["rays_in_map"]
        # bad regions are rejected
        lib = ml.load()
        for bad in ((-1, 4, 0, 4), (0, g.n1 + 1, 0, 4), (5, 4, 0, 4), (0, 4, 9, 8), (0, 4, 0, g.n2 + 1)):
            assert lib.ml_shoot_region(m.ctx, *bad, 0) == ml.ML_ERR_INVALID_ARG


def test_state_and_argument_errors_on_a_live_context():
    lib = ml.load()
    ctx = ml.ml_create(0.4, 1.0, 0.0, 32, 16.0, 5.0)
    try:
        assert lib.ml_shoot(ctx) == ml.ML_ERR_STATE  # before ml_set_lenses
        assert lib.ml_shoot_region(ctx, 0, 1, 0, 1, 0) == ml.ML_ERR_STATE
        bad = np.array([[0.0, np.nan]])
        assert lib.ml_set_lenses(ctx, bad.ctypes.data_as(C.POINTER(C.c_double)), 1) == ml.ML_ERR_INVALID_ARG
        assert lib.ml_set_lenses(ctx, None, -1) == ml.ML_ERR_INVALID_ARG
        assert lib.ml_set_precision(ctx, 7) == ml.ML_ERR_INVALID_ARG
        ml.ml_set_lenses(ctx, np.zeros((0, 2)))
        ml.ml_shoot(ctx)
        small = np.zeros(10, dtype=np.uint32)
        assert lib.ml_get_map(ctx, small.ctypes.data_as(C.POINTER(C.c_uint32)), small.size) == ml.ML_ERR_INVALID_ARG
        info = ml.ml_get_info(ctx)
        assert info["n_lenses"] == 0 and info["sm_count"] > 0
    finally:
        ml.ml_destroy(ctx)


@pytest.mark.parametrize("precision", ALL)
def test_ray_on_a_lens_does_not_poison_the_map(precision):
    """Reading R12: the deflection of a ray that sits exactly on a point mass is undefined.  The oracle and the fp64
    kernel find r^2 = 0, get a non-finite position and DROP the ray (counted in rays_dropped, not binned).  The FP32
    kernels hold ray and lens in tile-local FP32 coordinates, where the two coincide as well: r^2 = 0 + 2^-80, the term
    d/r^2 = 0 * 2^80 = 0, i.e. the ray does not see that one lens and is binned from the other N* - 1 (its partner in
    the shared reciprocal is untouched).  Either way nothing is NaN-poisoned and every ray is accounted for."""
    p = SMALL
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(40, g.r_star, 5)
    i, j = g.n1 // 2 + 3, g.n2 // 2 - 2
    xy[0] = ((i - (g.n1 - 1) / 2.0) * g.delta, (j - (g.n2 - 1) / 2.0) * g.delta)
    m, g, xy = make_pair(p, precision, lenses=xy)
    with m:
        m.shoot()
        omap, ost = oracle.shoot(*problem_args(p), xy)
        assert ost["rays_dropped"] == 1
        st = m.stats
        assert st["rays_shot"] == g.n1 * g.n2
        assert st["rays_in_map"] + st["rays_dropped"] <= st["rays_shot"]
        check_maps(p, m.counts(), st, omap, ost)
        y = m.probe([i], [j])[0]
        y_rest = oracle.deflect_points(p.gamma, g.kappa_c, xy[1:], np.array([xy[0]]))[0]   # the same ray without lens 0
        if precision == ml.ML_PREC_FP64:
            assert st["rays_dropped"] == 1 and np.isnan(y).all()
        else:
            assert st["rays_dropped"] == 0 and np.abs(y - y_rest).max() < 1e-3 * g.pixel


def test_caller_owned_torch_map_and_stream():
    """PyTorch supplies device memory and the stream; the library computes into them."""
    import torch
    p = SMALL
    m, g, xy = make_pair(p)
    with m:
        m.shoot()
        ref = m.counts().copy()
        t = torch.full((p.n_pix, p.n_pix), 7, dtype=torch.int32, device="cuda:0")
        s = torch.cuda.Stream()
        m.use_device_map(t.data_ptr())
        m.attach_stream(s.cuda_stream)
        m.shoot()
        s.synchronize()
        assert np.array_equal(t.cpu().numpy().astype(np.uint32), ref)
        assert ml.ml_get_map_device(m.ctx) == t.data_ptr()
        # host memory, or a misaligned device pointer, is refused and leaves the map in place
        host = np.zeros(p.n_pix * p.n_pix, dtype=np.uint32)
        for bad in (host.ctypes.data, t.data_ptr() + 2):
            with pytest.raises(ml.MicrolensError) as e:
                m.use_device_map(bad)
            assert e.value.code == ml.ML_ERR_INVALID_ARG
        assert ml.ml_get_map_device(m.ctx) == t.data_ptr()
        m.use_device_map(0)
        # NULL = the legacy default stream: a shoot there is ordered after earlier work of every blocking stream, so a
        # map zeroed / filled by torch on its own (blocking) stream right before is seen as written, while unrelated
        # work keeps a second torch stream busy
        m.use_device_map(t.data_ptr())
        m.attach_stream(0)
        busy = torch.cuda.Stream()
        with torch.cuda.stream(busy):
            junk = torch.randn(4096, 4096, device="cuda:0")
            for _ in range(4):
                junk = junk @ junk
                junk = junk / junk.abs().max()
        t.fill_(123)                       # torch's current stream = legacy default stream here
        m.shoot()                          # zeroes the map itself, then shoots, on the legacy stream
        assert np.array_equal(t.cpu().numpy().astype(np.uint32), ref)
        m.shoot_region(0, g.n1, 0, g.n2 // 2)
        t2 = t.clone()                     # ordered after the shoot on the same legacy stream
        m.shoot_region(0, g.n1, g.n2 // 2, g.n2, accumulate=True)
        torch.cuda.synchronize()
        assert np.array_equal(t.cpu().numpy().astype(np.uint32), ref) and int(t2.sum()) < int(t.sum())
        m.use_device_map(0)


def test_set_lenses_is_stream_ordered_and_keeps_nothing_of_the_callers_buffer():
    """ml_set_lenses returns without waiting for the device and reuses its buffers (a map-per-lens-field loop allocates
    nothing after the first pass).  It must still have copied the caller's arrays by the time it returns -- also when
    they are PINNED, where an asynchronous copy would read them later -- and a sequence of larger and smaller fields, with
    and without masses, on changing streams, must give the maps a fresh context gives for each field."""
    import torch
    p = SMALL
    g = oracle.geometry(*problem_args(p))

    def fresh(xy, mass=None):
        with ml.MagnificationMap(*problem_args(p)) as f:
            f.set_lenses(xy, mass)
            f.shoot()
            return f.counts().copy()

    fields = [(lens_disk(g.n_star, g.r_star, 3), None),
              (lens_disk(4 * g.n_star + 3, g.r_star, 4), lens_masses(4 * g.n_star + 3, 4)),   # grows, masses appear
              (lens_disk(7, g.r_star, 5), None),                                              # shrinks, unit masses again
              (lens_disk(2 * g.n_star, g.r_star, 6), lens_masses(2 * g.n_star, 6)),           # masses buffer reused
              (np.zeros((0, 2)), None)]                                                        # no stars
    want = [fresh(xy, mass) for xy, mass in fields]
    assert not np.array_equal(want[0], want[1]) and not np.array_equal(want[2], want[3])
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    with ml.MagnificationMap(*problem_args(p)) as m:
        for k, (xy, mass) in enumerate(fields):
            t_xy = torch.from_numpy(xy.copy()).pin_memory()
            t_m = torch.from_numpy(mass.copy()).pin_memory() if mass is not None else None
            m.set_lenses(t_xy.numpy(), t_m.numpy() if t_m is not None else None)
            t_xy.fill_(123.0)                      # the caller's (pinned) arrays are the caller's again
            if t_m is not None:
                t_m.fill_(50.0)
            if k % 2 == 1:                         # lenses set on one stream, shot on another
                m.attach_stream(streams[(k // 2) % 2].cuda_stream)
            m.shoot()
            assert m.info["n_lenses"] == xy.shape[0]
            assert np.array_equal(m.counts(), want[k]), k
        # a rejected field leaves the last one (no stars) in place
        bad = fields[0][0].copy()
        bad[1, 0] = np.inf
        with pytest.raises(ml.MicrolensError):
            m.set_lenses(bad)
        m.shoot()
        assert np.array_equal(m.counts(), want[-1])
