"""Pins of the oracle's unequal-mass variants (eq. 4 with its m_i; eq. 5 with <M>):
closed forms, exact scaling laws and an independent numpy brute force -- none of them the oracle itself."""
import math

import numpy as np

from oracle import oracle
from bruteforce import shoot_numpy

TINY = (0.0, 1.0, 0.0, 32, 16.0, 8.0)   # sigma = 0: lenses are passed explicitly


def test_mass_weighted_lens_equation_by_hand():
    # lens of mass 3 at (1,2), ray at (4,6): d = (3,4), |d|^2 = 25, deflection 3*(0.12, 0.16)
    y = oracle.deflect_points(0.3, 0.2, [[1.0, 2.0]], [[4.0, 6.0]], mass=[3.0])
    assert np.allclose(y, [[0.5 * 4 - 0.36, 1.1 * 6 - 0.48]], rtol=0, atol=1e-14)
    # a ray on the Einstein ring of a mass-m lens (radius sqrt(m)) comes from the point behind the lens
    for m in (0.25, 1.0, 4.0, 9.0):
        y = oracle.deflect_points(0.0, 0.0, [[0.0, 0.0]], [[math.sqrt(m), 0.0], [0.0, -math.sqrt(m)]], mass=[m])
        assert np.abs(y).max() < 1e-15
    # masses add linearly
    y = oracle.deflect_points(0.0, 0.0, [[1.0, 2.0], [4.0, 3.0]], [[4.0, 6.0]], mass=[2.0, 0.5])
    assert np.allclose(y, [[4 - 0.24, 6 - 0.32 - 0.5 / 3]], rtol=0, atol=1e-14)


def test_unit_masses_reproduce_the_unit_mass_path_bit_for_bit():
    rng = np.random.default_rng(3)
    xy = rng.uniform(-6, 6, size=(7, 2))
    a, sa = oracle.shoot(*TINY, xy)
    b, sb = oracle.shoot(*TINY, xy, mass=np.ones(7))
    assert np.array_equal(a, b) and sa == sb
    g = oracle.geometry(*TINY)
    ya = oracle.capture_region(*TINY, xy, (0, g.n1, 3, 9))
    yb = oracle.capture_region(*TINY, xy, (0, g.n1, 3, 9), mass=np.ones(7))
    assert np.array_equal(ya, yb)


def test_two_coincident_unit_lenses_are_one_lens_of_mass_two():
    rng = np.random.default_rng(4)
    xy = rng.uniform(-5, 5, size=(5, 2))
    doubled = np.concatenate([xy, xy[1:2]])          # lens 1 twice, unit masses
    a, _ = oracle.shoot(*TINY, doubled)
    m = np.ones(5)
    m[1] = 2.0
    b, _ = oracle.shoot(*TINY, xy, mass=m)
    # x/r2 + x/r2 = 2x/r2 exactly, but the summation order differs (the copy is added last): allow stray rays
    assert int(a.sum()) > 0 and np.abs(a.astype(np.int64) - b.astype(np.int64)).sum() <= 4
    # same order -> exact: the copy right after the original
    doubled = np.concatenate([xy[:2], xy[1:2], xy[2:]])
    g = oracle.geometry(*TINY)
    ya = oracle.capture_region(*TINY, doubled, (0, g.n1, 0, 4))
    yb = oracle.capture_region(*TINY, xy, (0, g.n1, 0, 4), mass=m)
    assert np.abs(ya - yb).max() < 1e-12


def test_mass_scaling_law_is_exact_for_a_factor_of_four():
    """x -> x/sqrt(m), y -> y/sqrt(m) maps a field of mass-m lenses onto unit lenses.  With m = 4 the factor is 2,
    exact in binary floating point, and the ray grid scales with L: the maps must be identical integers."""
    rng = np.random.default_rng(5)
    xy = rng.uniform(-4, 4, size=(6, 2))
    a, sa = oracle.shoot(0.0, 1.0, 0.0, 32, 16.0, 8.0, xy)
    b, sb = oracle.shoot(0.0, 1.0, 0.0, 32, 16.0, 16.0, 2.0 * xy, mass=np.full(6, 4.0))
    assert np.array_equal(a, b) and sa == sb and sa["rays_in_map"] > 0


def test_ring_of_unequal_masses_obeys_the_gauss_theorem():
    n, R = 64, 10.0
    th = 2 * np.pi * (np.arange(n) + 0.25) / n
    ring = np.stack([R * np.cos(th), R * np.sin(th)], axis=1)
    mass = np.where(np.arange(n) % 2 == 0, 1.0, 3.0)   # period-2 pattern: corrections of order (r/R)^(n/2)
    inside = np.array([[3.0, -2.0], [-1.5, 4.0], [0.0, 0.0]])
    y = oracle.deflect_points(0.0, 0.0, ring, inside, mass=mass)
    assert np.abs(y - inside).max() < 1e-9
    outside = np.array([[35.0, 7.0], [-3.0, -40.0]])
    y = oracle.deflect_points(0.0, 0.0, ring, outside, mass=mass)
    alpha = mass.sum() * outside / (outside ** 2).sum(axis=1, keepdims=True)
    assert np.abs((outside - y) - alpha).max() < 1e-9


def test_mass_weighted_map_equals_numpy_brute_force():
    rng = np.random.default_rng(6)
    args = (0.5, 0.4, 0.1, 16, 9.0, 6.0)
    xy = rng.uniform(-8, 8, size=(9, 2))
    mass = rng.uniform(0.2, 3.0, size=9)
    a, st = oracle.shoot(*args, xy, mass=mass)
    b, shot, n_in = shoot_numpy(*args, xy, mass=mass)
    assert shot == st["rays_shot"] and n_in == st["rays_in_map"] and np.array_equal(a, b)
    assert not np.array_equal(a, oracle.shoot(*args, xy)[0])   # the masses matter


def test_n_star_with_a_mean_mass():
    # eq. 5: N* = sigma_* A / (pi <M>): halving the mean mass doubles the number of lenses
    assert oracle.n_star(0.4, 36.7696, 1.0) == oracle.n_star(0.4, 36.7696) == 541
    assert oracle.n_star(0.4, 36.7696, 0.5) == 1082 and oracle.n_star(0.4, 36.7696, 2.0) == 270
