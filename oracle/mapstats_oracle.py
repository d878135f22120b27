"""Map-comparison oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy fp64 restatement of the paper's two accuracy measures between magnification maps
(section 3.1): the root-mean-square difference of the maps in magnitudes and
a two-sample Kolmogorov-Smirnov test on the distributions of the change in magnitude

    Delta m_ij = -2.5 log10(mu_ij)         (eq. 10),   mu_ij = N_ij / N_rays (eq. 3, :47).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module; it shares nothing with paper_1005_5198_b200/ (the CUDA side is csrc/mapstats.cu).

Each function is the textbook definition written out, no blocking or shortcuts:
  delta_m            eq. 10, element by element; a pixel that received no ray has Delta m = +inf.
  rms_delta_m        sqrt(mean((Delta m_a - Delta m_b)^2)) over "corresponding" pixels;
                     reading M1: pixels where either map is empty (infinite Delta m) are left out and counted.
  ks_statistic       D = sup_x |F_a(x) - F_b(x)|, F = empirical distribution of Delta m over ALL pixels of a map
                     (reading M2: an empty pixel is a sample at +inf; it changes F's normalisation only).
                     Written as the definition: both samples sorted, both ECDFs evaluated at every sample point.
  ks_probability     significance of D: Q_KS(lambda) = 2 sum_{j>=1} (-1)^(j-1) exp(-2 j^2 lambda^2) with
                     lambda = (sqrt(Ne) + 0.12 + 0.11/sqrt(Ne)) D, Ne = na nb/(na + nb).  The paper only says
                     "K-S test ... probability"; reading M3 takes the standard asymptotic
                     form with Stephens' small-sample correction.
  histogram_delta_m  counts of Delta m in n_bins equal bins of [lo, hi): the "probability distributions for
                     change in magnitude" of PAPER.md:169 (reading M4: half-open bins, values outside dropped).

Pins (tests/test_mapstats_oracle.py): scipy.stats.ks_2samp (statistic) and scipy.special.kolmogorov (the
series) as independent library routines, the 5 % / 1 % critical values lambda = 1.358 / 1.628 of the Kolmogorov
distribution, hand-worked tiny samples, RMS of a map against its own multiple = 2.5 log10(k), numpy.histogram.
No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def delta_m(counts, n_rays):
    """eq. 10 with mu = N / N_rays (eq. 3); +inf where N = 0."""
    c = np.asarray(counts, dtype=np.float64)
    with np.errstate(divide="ignore"):
        return -2.5 * np.log10(c / float(n_rays))


def rms_delta_m(counts_a, n_rays_a, counts_b, n_rays_b):
    """(rms, n_valid): RMS difference in magnitudes over pixels lit in both maps (M1)."""
    a = np.asarray(counts_a).ravel()
    b = np.asarray(counts_b).ravel()
    assert a.shape == b.shape
    ok = (a > 0) & (b > 0)
    if not ok.any():
        return 0.0, 0
    d = delta_m(a[ok], n_rays_a) - delta_m(b[ok], n_rays_b)
    return float(np.sqrt(np.mean(d * d))), int(ok.sum())


def ks_statistic(counts_a, n_rays_a, counts_b, n_rays_b):
    """Two-sample K-S distance between the Delta m samples of two maps (M2)."""
    xa = np.sort(delta_m(np.asarray(counts_a).ravel(), n_rays_a))
    xb = np.sort(delta_m(np.asarray(counts_b).ravel(), n_rays_b))
    na, nb = xa.size, xb.size
    if na == 0 or nb == 0:
        return 0.0
    pts = np.concatenate([xa, xb])
    pts = pts[np.isfinite(pts)]            # F_a(+inf) = F_b(+inf) = 1: no difference there
    fa = np.searchsorted(xa, pts, side="right") / na   # F(x) = fraction of samples <= x
    fb = np.searchsorted(xb, pts, side="right") / nb
    return float(np.abs(fa - fb).max()) if pts.size else 0.0


def ks_probability(d, na, nb):
    """Q_KS: probability of a distance >= d under the null hypothesis (M3).  The alternating series is summed
    until its terms vanish in fp64 (about 3/lambda terms); below lambda = 0.04 Q_KS = 1 to 1e-300."""
    ne = float(na) * float(nb) / (float(na) + float(nb))
    lam = (np.sqrt(ne) + 0.12 + 0.11 / np.sqrt(ne)) * float(d)
    if lam < 0.04:
        return 1.0
    total, j = 0.0, 1
    while True:
        term = np.exp(-2.0 * j * j * lam * lam)
        total += term if j % 2 else -term
        if term < 1e-20:
            break
        j += 1
    return float(min(1.0, max(0.0, 2.0 * total)))


def histogram_delta_m(counts, n_rays, lo, hi, n_bins):
    """Counts of Delta m in n_bins equal half-open bins of [lo, hi) (M4)."""
    x = delta_m(np.asarray(counts).ravel(), n_rays)
    x = x[np.isfinite(x)]
    k = np.floor((x - lo) / ((hi - lo) / n_bins)).astype(np.int64)
    k = k[(x >= lo) & (k >= 0) & (k < n_bins)]
    return np.bincount(k, minlength=n_bins).astype(np.uint64)


def mean_mu(counts, n_rays):
    """Map-mean magnification (eq. 3; compared with eq. 12)."""
    return float(np.asarray(counts, dtype=np.float64).mean() / float(n_rays))
