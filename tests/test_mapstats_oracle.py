"""Pins of oracle/mapstats_oracle.py (CPU): the paper's map-comparison measures (eq. 10)
against things that are not the oracle itself -- library routines (scipy.stats.ks_2samp, scipy.special.kolmogorov,
numpy.histogram), tabulated critical values of the Kolmogorov distribution, hand-worked samples and closed forms.
"""
import math

import numpy as np
import pytest
from scipy import special, stats

from oracle import mapstats_oracle as mo


def _maps(seed, n=64, mean=200.0):
    rng = np.random.default_rng(seed)
    lam = mean * rng.lognormal(0.0, 0.6, size=(n, n))
    return rng.poisson(lam).astype(np.uint32)


def test_delta_m_is_eq10_on_hand_values():
    # mu = 1 -> 0 mag; mu = 10 -> -2.5 mag; mu = 0.01 -> +5 mag; mu = 2.5119 -> -1.0000 mag (Pogson's ratio)
    dm = mo.delta_m(np.array([100, 1000, 1, 0], dtype=np.uint32), 100.0)
    assert dm[0] == 0.0 and abs(dm[1] + 2.5) < 1e-15 and abs(dm[2] - 5.0) < 1e-15 and np.isposinf(dm[3])
    assert abs(mo.delta_m(np.array([100.0 ** 0.2 * 1e6]), 1e6)[0] + 1.0) < 1e-12
    # brighter (more rays) means smaller magnitude: the minus sign of eq. 10
    assert mo.delta_m([300], 100.0)[0] < mo.delta_m([200], 100.0)[0]


def test_rms_of_a_map_against_its_multiple_is_the_magnitude_of_the_factor():
    a = _maps(0)
    a[a == 0] = 1
    for k in (2, 3, 10):
        rms, n = mo.rms_delta_m(a, 100.0, a * k, 100.0)
        assert n == a.size and abs(rms - 2.5 * math.log10(k)) < 1e-12
        # the same factor hidden in n_rays cancels: identical magnification maps
        rms, _ = mo.rms_delta_m(a, 100.0, a * k, 100.0 * k)
        assert rms < 1e-12
    # hand-worked: two pixels, differences 2.5 log10(2) and 0 -> rms = 2.5 log10(2)/sqrt(2)
    rms, n = mo.rms_delta_m([100, 50], 100.0, [200, 50], 100.0)
    assert n == 2 and abs(rms - 2.5 * math.log10(2) / math.sqrt(2)) < 1e-14


def test_rms_leaves_out_pixels_empty_in_either_map():
    rms, n = mo.rms_delta_m([0, 100, 7, 100], 100.0, [5, 0, 7, 1000], 100.0)
    assert n == 2 and abs(rms - math.sqrt((0.0 + 2.5 ** 2) / 2)) < 1e-14
    assert mo.rms_delta_m([0, 0], 10.0, [1, 1], 10.0) == (0.0, 0)


@pytest.mark.parametrize("seed,na,nb", [(1, 100.0, 100.0), (2, 100.0, 250.0), (3, 37.5, 100.0)])
def test_ks_statistic_equals_scipy_ks_2samp(seed, na, nb):
    a, b = _maps(seed), _maps(seed + 100, mean=200.0 * nb / na * 1.03)
    a[:2, :3] = 0                                   # some empty pixels: samples at +inf
    d = mo.ks_statistic(a, na, b, nb)
    xa, xb = mo.delta_m(a.ravel(), na), mo.delta_m(b.ravel(), nb)
    big = 1e300                                      # scipy wants finite samples; +inf -> a value above all others
    ref = stats.ks_2samp(np.where(np.isfinite(xa), xa, big), np.where(np.isfinite(xb), xb, big), method="asymp")
    assert abs(d - ref.statistic) < 1e-15
    # invariant under the monotone map Delta m -> mu (the statistic only sees the order of the samples)
    ref_mu = stats.ks_2samp(a.ravel() / na, b.ravel() / nb, method="asymp")
    assert abs(d - ref_mu.statistic) < 1e-15


def test_ks_statistic_hand_worked_and_extremes():
    # samples (as counts, n_rays = 1): a = {1,2,3}, b = {2,3,4}; in mu the ECDFs differ by at most 1/3
    assert abs(mo.ks_statistic([1, 2, 3], 1.0, [2, 3, 4], 1.0) - 1.0 / 3.0) < 1e-15
    assert mo.ks_statistic([5, 6, 7], 1.0, [5, 6, 7], 1.0) == 0.0
    assert mo.ks_statistic([1, 2, 3], 1.0, [10, 20, 30, 40], 1.0) == 1.0
    # a = {1,1,2,5}, b = {1,3,3,4,9}: F_a - F_b at mu = 1,2,3,4,5,9 is .3,.55,.15,-.05,.2,0 -> D = 0.55
    assert abs(mo.ks_statistic([1, 1, 2, 5], 1.0, [1, 3, 3, 4, 9], 1.0) - 0.55) < 1e-15
    # same magnification maps recorded with different n_rays: identical distributions
    assert mo.ks_statistic([10, 20, 30], 10.0, [30, 60, 90], 30.0) == 0.0


def test_ks_probability_is_the_kolmogorov_series_with_stephens_correction():
    for d, na, nb in [(0.01, 4096, 4096), (0.02, 16384, 8000), (0.3, 20, 30), (0.001, 10 ** 6, 10 ** 6),
                      (2e-4, 16384, 16384), (0.004, 16384, 16384), (0.0008, 16384, 16384), (0.03, 300, 200)]:
        ne = na * nb / (na + nb)
        lam = (math.sqrt(ne) + 0.12 + 0.11 / math.sqrt(ne)) * d
        assert abs(mo.ks_probability(d, na, nb) - special.kolmogorov(lam)) < 1e-12
    # tabulated critical values of the Kolmogorov distribution: Q(1.3581) = 0.05, Q(1.6276) = 0.01
    big = 10 ** 12                                   # correction terms negligible: lambda = sqrt(Ne) d
    ne = big / 2
    assert abs(mo.ks_probability(1.3581 / math.sqrt(ne), big, big) - 0.05) < 2e-4
    assert abs(mo.ks_probability(1.6276 / math.sqrt(ne), big, big) - 0.01) < 1e-4
    assert mo.ks_probability(0.0, 100, 100) == 1.0 and mo.ks_probability(1.0, 10 ** 4, 10 ** 4) < 1e-300 + 1e-12
    # monotone: a larger distance is less probable
    p = [mo.ks_probability(d, 5000, 5000) for d in (0.005, 0.01, 0.02, 0.04)]
    assert all(x > y for x, y in zip(p, p[1:]))


def test_histogram_equals_numpy_histogram():
    a = _maps(7)
    a[0, :5] = 0
    lo, hi, nb = -3.003, 2.999, 97
    h = mo.histogram_delta_m(a, 150.0, lo, hi, nb)
    x = mo.delta_m(a.ravel(), 150.0)
    x = x[np.isfinite(x)]
    ref, _ = np.histogram(x[x < hi], bins=nb, range=(lo, hi))   # numpy closes the last bin; ours is half-open
    assert np.array_equal(h, ref.astype(np.uint64))
    assert h.sum() <= a.size - 5


def test_mean_mu():
    assert mo.mean_mu(np.full((4, 4), 250, dtype=np.uint32), 100.0) == 2.5
