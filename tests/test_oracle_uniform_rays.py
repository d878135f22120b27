"""Pins of the oracle's uniform-ray mode (ray_mode "uniform", reading R20): every ray an independent uniform point of
the whole shooting rectangle -- "a batch of 2^17 random ray positions" "shot from random positions in the
shooting grid ... This will introduce Poisson noise".  The generator itself (Philox-4x32-10, counter =
ray id) is pinned in test_oracle_random_rays.py; here: where the rays are, that their counts are Poisson (what the paper
says of its own maps, and what reading R17's one-ray-per-cell sampler is not), eq. 12 in the mean, a brute force."""
import math

import numpy as np

from oracle import oracle
from test_oracle_random_rays import _uniforms_py

TINY = (0.3, 0.5, 0.1, 16, 9.0, 6.0)


def test_uniform_rays_cover_the_shooting_rectangle_and_nothing_else():
    args = (0.3, 0.5, 0.1, 16, 64.0, 6.0)           # TINY with more rays: 256 x 192 of them, every one taken once
    g = oracle.geometry(*args)
    ri, rj = [v.ravel() for v in np.meshgrid(np.arange(g.n1), np.arange(g.n2))]
    x = oracle.ray_positions(*args, ri, rj, ray_seed=3, ray_mode="uniform")
    w1, w2 = g.n1 * g.delta, g.n2 * g.delta          # the rectangle the regular grid's cells tile
    assert x[:, 0].min() >= -w1 / 2 and x[:, 0].max() < w1 / 2 and x[:, 1].min() >= -w2 / 2 and x[:, 1].max() < w2 / 2
    # uniform: mean 0, variance w^2/12 per axis, axes uncorrelated, and NOT tied to the cell (i, j) that numbers the ray
    for k, w in ((0, w1), (1, w2)):
        assert abs(x[:, k].mean()) < 4 * w / math.sqrt(12 * x.shape[0])
        assert abs(x[:, k].var() / (w * w / 12) - 1) < 0.03
    assert abs(np.corrcoef(x[:, 0], x[:, 1])[0, 1]) < 0.03
    x0 = oracle.ray_positions(*args, ri, rj)
    assert abs(np.corrcoef(x[:, 0], x0[:, 0])[0, 1]) < 0.03 and abs(np.corrcoef(x[:, 1], x0[:, 1])[0, 1]) < 0.03
    h, _, _ = np.histogram2d(x[:, 0], x[:, 1], bins=(8, 8), range=((-w1 / 2, w1 / 2), (-w2 / 2, w2 / 2)))
    assert ((h - x.shape[0] / 64) ** 2 / (x.shape[0] / 64)).sum() < 110           # chi^2, 63 dof
    # exactly where a second implementation of the generator puts them
    for k in range(50):
        u1, u2 = _uniforms_py(int(rj[k]) * g.n1 + int(ri[k]), 3)
        assert x[k, 0] == (u1 * g.n1 - g.n1 / 2.0) * g.delta and x[k, 1] == (u2 * g.n2 - g.n2 / 2.0) * g.delta


def test_uniform_rays_without_stars_give_eq12_in_the_mean_with_poisson_noise():
    """without stars the map is uniform with magnification 1/|(1 - sigma)^2 - gamma^2| (eq. 12) and random
    ray positions "introduce Poisson noise": index of dispersion 1 (reading R17's sampler has < 0.5, pinned there)."""
    args = (0.4, 0.0, 0.0, 64, 100.0, 10.0)       # no stars: mu = 1/0.36, <N> = 277.8 rays per pixel, 4096 pixels
    a, st = oracle.shoot(*args, np.zeros((0, 2)), ray_seed=5, ray_mode="uniform")
    mean = a.mean()
    assert abs(mean / (100.0 / 0.36) - 1) < 4 / math.sqrt(a.sum())               # Poisson error of the total
    # sample variance of 4096 Poisson counts: relative standard error sqrt(2/4095) = 2.2 %
    assert abs(a.var(ddof=1) / mean - 1) < 0.09
    assert st["rays_in_map"] == int(a.sum()) and st["rays_shot"] == st["rays_in_map"] + st["rays_out_of_map"]
    # the one-ray-per-cell sampler on the same problem is far below Poisson
    b, _ = oracle.shoot(*args, np.zeros((0, 2)), ray_seed=5)
    assert b.var(ddof=1) < 0.5 * b.mean() < 0.6 * a.var(ddof=1)


def test_uniform_ray_map_equals_an_independent_brute_force():
    g = oracle.geometry(*TINY)
    xy = np.random.default_rng(2).uniform(-7, 7, size=(5, 2))
    mass = np.array([0.5, 2.0, 1.0, 1.5, 0.7])
    seed = 78
    sigma, f, gamma, n_pix, n_rays, L = TINY
    kc = sigma - sigma * f
    for m in (None, mass):
        a, st = oracle.shoot(*TINY, xy, mass=m, ray_seed=seed, ray_mode="uniform")
        mm = np.ones(5) if m is None else m
        counts = np.zeros((n_pix, n_pix), dtype=np.int64)
        for k in range(g.n1 * g.n2):
            u1, u2 = _uniforms_py(k, seed)
            x1, x2 = (u1 * g.n1 - g.n1 / 2.0) * g.delta, (u2 * g.n2 - g.n2 / 2.0) * g.delta
            d1, d2 = x1 - xy[:, 0], x2 - xy[:, 1]
            r2 = d1 * d1 + d2 * d2
            t1, t2 = (d1 / r2, d2 / r2) if m is None else (mm * d1 / r2, mm * d2 / r2)
            y1 = (1 - gamma) * x1 - kc * x1 - float(np.cumsum(t1)[-1])
            y2 = (1 + gamma) * x2 - kc * x2 - float(np.cumsum(t2)[-1])
            ii, jj = math.floor((y1 + L / 2) / g.pixel), math.floor((y2 + L / 2) / g.pixel)
            if 0 <= ii < n_pix and 0 <= jj < n_pix:
                counts[jj, ii] += 1
        assert st["rays_shot"] == g.n1 * g.n2 and counts.sum() == st["rays_in_map"]
        assert np.abs(counts - a).sum() <= 2          # sequential cumsum = the oracle's order; allow a stray edge ray
        assert not np.array_equal(a, oracle.shoot(*TINY, xy, mass=m, ray_seed=seed)[0])


def test_uniform_ray_regions_partition_the_rays_by_id():
    """A region (i0, i1, j0, j1) selects ray ids j n1 + i, not a patch of the image plane: regions that tile the index
    grid add up to the full map, and capture_region returns the rays in id order."""
    g = oracle.geometry(*TINY)
    xy = np.random.default_rng(3).uniform(-7, 7, size=(4, 2))
    full, _ = oracle.shoot(*TINY, xy, ray_seed=4, ray_mode="uniform")
    acc = np.zeros_like(full)
    for reg in [(0, 17, 0, g.n2), (17, g.n1, 0, 5), (17, g.n1, 5, g.n2)]:
        oracle.shoot_region(*TINY, xy, region=reg, map_out=acc, ray_seed=4, ray_mode="uniform")
    assert np.array_equal(acc, full)
    reg = (3, 9, 2, 6)
    y = oracle.capture_region(*TINY, xy, reg, ray_seed=4, ray_mode="uniform")
    ii, jj = np.meshgrid(np.arange(3, 9), np.arange(2, 6))
    x = oracle.ray_positions(*TINY, ii.ravel(), jj.ravel(), ray_seed=4, ray_mode="uniform")
    y2 = oracle.deflect_points(TINY[2], TINY[0] - TINY[0] * TINY[1], xy, x)
    assert np.array_equal(y.reshape(-1, 2), y2)


def test_single_lens_magnification_pattern_with_uniform_rays():
    """Point-lens A(u) = (u^2 + 2)/(u sqrt(u^2 + 4)) on rings around an isolated lens, within the Poisson error of the
    counts: the uniform rays sample the same lens equation as the regular grid."""
    args = (1e-9, 1.0, 0.0, 64, 400.0, 4.0)       # sigma ~ 0: the lens is isolated, N* is set by hand
    a, _ = oracle.shoot(*args, np.array([[0.0, 0.0]]), ray_seed=21, ray_mode="uniform")
    n_pix, n_rays, L = 64, 400.0, 4.0
    c = (np.arange(n_pix) + 0.5) * L / n_pix - L / 2
    r = np.hypot(*np.meshgrid(c, c))
    for lo, hi in ((0.5, 0.8), (0.8, 1.2), (1.2, 1.8)):
        ring = (r >= lo) & (r < hi)
        u = r[ring]
        expect = ((u * u + 2) / (u * np.sqrt(u * u + 4))).mean()
        got = a[ring].mean() / n_rays
        assert abs(got / expect - 1) < 5 / math.sqrt(a[ring].sum()) + 2e-3, (lo, hi, got, expect)
