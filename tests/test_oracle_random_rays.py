"""Pins of the oracle's random-ray mode (GPU-D shoots rays "from random positions in the shooting grid",
PAPER.md:131, :167; reading R17: one uniformly random ray per grid cell, Philox-4x32-10 keyed by the seed)."""
import math
import os

import numpy as np

from oracle import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
TINY = (0.3, 0.5, 0.1, 16, 9.0, 6.0)


def _philox_py(ctr, key):
    """Second, independent restatement of Philox-4x32-10 (Python integers)."""
    c, k = [int(v) for v in ctr], [int(v) for v in key]
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def _uniforms_py(ray_id, seed):
    r = _philox_py([ray_id & 0xFFFFFFFF, ray_id >> 32, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])
    return (((r[0] >> 5) * 2 ** 26 + (r[1] >> 6)) / 2 ** 53, ((r[2] >> 5) * 2 ** 26 + (r[3] >> 6)) / 2 ** 53)


def test_philox_reproduces_the_published_known_answer_vectors():
    rows = [ln.split() for ln in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if ln.strip() and ln[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        w = [int(v, 16) for v in r]
        assert oracle.philox4x32_10(w[0:4], w[4:6]) == w[6:10]
        assert _philox_py(w[0:4], w[4:6]) == w[6:10]


def test_uniforms_are_53_bit_uniform_and_keyed():
    ids = np.arange(0, 40000, dtype=np.uint64) * np.uint64(2654435761) + np.uint64(1 << 33)   # ids beyond 32 bits too
    u = np.array([oracle.ray_uniforms(int(k), 12345) for k in ids])
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size) and abs(u.var() - 1 / 12) < 2e-3
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.02
    assert abs(np.corrcoef(u[:-1, 0], u[1:, 0])[0, 1]) < 0.02
    h, _ = np.histogram(u[:, 0], bins=20, range=(0, 1))
    assert ((h - u.shape[0] / 20) ** 2 / (u.shape[0] / 20)).sum() < 60          # chi^2, 19 dof
    for k, seed in [(0, 0), (7, 3), (2 ** 40 + 5, 2 ** 63 + 11)]:
        assert oracle.ray_uniforms(k, seed) == _uniforms_py(k, seed)
    assert oracle.ray_uniforms(7, 3) != oracle.ray_uniforms(7, 4) and oracle.ray_uniforms(7, 3) != oracle.ray_uniforms(8, 3)


def test_every_random_ray_lies_in_its_own_grid_cell():
    g = oracle.geometry(*TINY)
    rng = np.random.default_rng(1)
    ri, rj = rng.integers(0, g.n1, 5000), rng.integers(0, g.n2, 5000)
    ri[:4], rj[:4] = [0, g.n1 - 1, 0, g.n1 - 1], [0, 0, g.n2 - 1, g.n2 - 1]
    xr = oracle.ray_positions(*TINY, ri, rj, ray_seed=9)
    x0 = oracle.ray_positions(*TINY, ri, rj)
    # the regular ray is the cell centre: the random one is within half a spacing of it, per axis
    d = (xr - x0) / g.delta
    assert d.min() >= -0.5 and d.max() < 0.5 and abs(d.mean()) < 0.02 and abs(d.var() - 1 / 12) < 0.01
    # and exactly where the second implementation of the generator puts it
    for k in range(50):
        u1, u2 = _uniforms_py(int(rj[k]) * g.n1 + int(ri[k]), 9)
        assert xr[k, 0] == (ri[k] + u1 - g.n1 / 2.0) * g.delta and xr[k, 1] == (rj[k] + u2 - g.n2 / 2.0) * g.delta


def test_random_ray_map_equals_an_independent_brute_force():
    g = oracle.geometry(*TINY)
    xy = np.random.default_rng(2).uniform(-7, 7, size=(5, 2))
    seed = 77
    a, st = oracle.shoot(*TINY, xy, ray_seed=seed)
    sigma, f, gamma, n_pix, n_rays, L = TINY
    kc = sigma - sigma * f
    counts = np.zeros((n_pix, n_pix), dtype=np.int64)
    for j in range(g.n2):
        for i in range(g.n1):
            u1, u2 = _uniforms_py(j * g.n1 + i, seed)
            x1, x2 = (i + u1 - g.n1 / 2.0) * g.delta, (j + u2 - g.n2 / 2.0) * g.delta
            d1, d2 = x1 - xy[:, 0], x2 - xy[:, 1]
            r2 = d1 * d1 + d2 * d2
            y1 = (1 - gamma) * x1 - kc * x1 - float(np.cumsum(d1 / r2)[-1])
            y2 = (1 + gamma) * x2 - kc * x2 - float(np.cumsum(d2 / r2)[-1])
            ii, jj = math.floor((y1 + L / 2) / g.pixel), math.floor((y2 + L / 2) / g.pixel)
            if 0 <= ii < n_pix and 0 <= jj < n_pix:
                counts[jj, ii] += 1
    assert st["rays_shot"] == g.n1 * g.n2 and counts.sum() == st["rays_in_map"]
    assert np.abs(counts - a).sum() <= 2          # sequential cumsum = the oracle's order; allow a stray edge ray
    assert not np.array_equal(a, oracle.shoot(*TINY, xy)[0]) and not np.array_equal(a, oracle.shoot(*TINY, xy, ray_seed=78)[0])


def test_random_rays_without_stars_give_eq12_in_the_mean_with_sub_poisson_noise():
    args = (0.4, 0.0, 0.0, 64, 100.0, 10.0)       # no stars: mu = 1/0.36
    a, st = oracle.shoot(*args, np.zeros((0, 2)), ray_seed=5)
    mean = a.mean() / 100.0
    assert abs(mean / (1 / 0.36) - 1) < 2e-3
    # one ray per cell: the count in a pixel fluctuates only through the cells cut by its border
    assert 0.0 < a.var() < 0.5 * a.mean()
    assert st["rays_in_map"] == int(a.sum()) and st["rays_shot"] == st["rays_in_map"] + st["rays_out_of_map"]


def test_random_ray_regions_tile_the_full_map():
    g = oracle.geometry(*TINY)
    xy = np.random.default_rng(3).uniform(-7, 7, size=(4, 2))
    full, _ = oracle.shoot(*TINY, xy, ray_seed=4)
    acc = np.zeros_like(full)
    for reg in [(0, 17, 0, g.n2), (17, g.n1, 0, 5), (17, g.n1, 5, g.n2)]:
        oracle.shoot_region(*TINY, xy, region=reg, map_out=acc, ray_seed=4)
    assert np.array_equal(acc, full)
