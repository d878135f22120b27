"""Pins of the fp64 CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path.  Each test
names the mistake it would catch.  All run without a GPU.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle
from workloads import CONFIGS, lens_disk

from bruteforce import shoot_numpy

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                out.append(line.split())
    return out


# ---------------------------------------------------------------- eq.(5) units (pin h)
def test_n_star_reproduces_the_papers_lens_counts():
    """PAPER.md:156-157 and Fig. 1 (:25) print 21 lens counts.  With A = pi R^2 and
    <M> = 1, eq.(5) is N* = sigma_* R^2; the paper's (unstated) disk rule, inferred in
    SURVEY.md section 4, is R = 1.5 sqrt((L/2/(1-s-g))^2 + (L/2/(1-s+g))^2) + 2 at L = 20.
    A factor pi, a diameter-for-radius slip or a wrong rounding misses all of them."""
    exact = 0
    rows = _rows("paper_nstar.txt")
    for sig, gam, sig_c, n_paper, _cite in rows:
        sig, gam, sig_c, n_paper = float(sig), float(gam), float(sig_c), int(n_paper)
        r = 1.5 * math.hypot(10.0 / (1 - sig - gam), 10.0 / (1 - sig + gam)) + 2.0
        got = oracle.n_star(sig - sig_c, r)
        exact += got == n_paper
        assert abs(got / n_paper - 1) < 3e-4, (sig, gam, got, n_paper)
    # 20 of the 21 printed values are reproduced to the integer; sigma = 0.9 gives 41267
    # against the printed 41257 (one digit, 2.4e-4 -- a misprint or single precision).
    assert exact >= len(rows) - 1


def test_phi_bookkeeping_of_eq6_and_eq9():
    """eq.(6) with N_FLOP = 10 reproduces the printed range of eq.(9) and Phi_fiducial:
    fixes what 'one interaction = 10 flop' means for the metric."""
    for n_side, n_star, n_rays, phi, _cite in _rows("paper_phi.txt"):
        got = 10.0 * int(n_side) ** 2 * int(n_star) * float(n_rays)
        assert abs(got / float(phi) - 1) < 0.2


# ---------------------------------------------------------------- geometry vs BASELINE.json text
def test_geometry_matches_the_config_statements():
    """BASELINE.json:configs quotes N*~140 / ~540 / ~20 000 / ~10 000 / ~1 200, a1~120 R_E for
    config 3, and ~8e9 / ~1.2e10 / ~2.5e10 rays for configs 2, 4, 5."""
    g = [oracle.geometry(c.sigma, c.stellar_fraction, c.gamma, c.n_pix, c.n_rays, c.L)
         for c in CONFIGS]
    for gi, approx in zip(g, (140, 540, 20000, 10000, 1200)):
        assert abs(gi.n_star / approx - 1) < 0.05
    assert abs(g[2].a1 - 120.0) < 1e-9 and abs(g[2].a2 - 24.0) < 1e-9
    assert abs(g[1].n1 * g[1].n2 / 8e9 - 1) < 0.06
    assert abs(g[3].n1 * g[3].n2 / 1.2e10 - 1) < 0.02
    assert abs(g[4].n1 * g[4].n2 / 2.5e10 - 1) < 0.02
    # C1 by hand: a = 1.2*5/0.6 = 10, delta = (10/128)/10, n = 20/delta = 2560,
    # R* = 1.3*sqrt(200), N* = round(0.4*338) = 135; kappa split for C5: 0.18 / 0.42
    assert (g[0].n1, g[0].n2, g[0].n_star) == (2560, 2560, 135)
    assert g[0].delta == 0.0078125 and g[0].pixel == 0.078125
    assert abs(g[4].kappa_star - 0.18) < 1e-12 and abs(g[4].kappa_c - 0.42) < 1e-12
    # eq.(12), and its printed examples PAPER.md:308
    assert abs(g[0].mu_th - 1 / 0.36) < 1e-12 and abs(g[2].mu_th + 20.0) < 1e-9
    q = oracle.geometry(0.394, 1.0, 0.395, 64, 10, 10.0)
    assert abs(q.mu_th - 4.735) < 5e-3          # Q2237+0305 image A
    q = oracle.geometry(0.476, 1.0, 0.565, 64, 10, 10.0)
    assert abs(q.mu_th + 22.4) < 0.05           # SDSS J0924+0219 image D


def test_geometry_rejects_the_critical_line_and_bad_input():
    """1 - sigma -/+ gamma ~ 0 makes the rectangle infinite."""
    for bad in ((0.5, 1.0, 0.5, 64, 10, 10.0), (1.5, 1.0, -0.5, 64, 10, 10.0),
                (-0.1, 1.0, 0.0, 64, 10, 10.0), (0.4, 1.5, 0.0, 64, 10, 10.0),
                (0.4, 1.0, 0.0, 0, 10, 10.0), (0.4, 1.0, 0.0, 64, 0.0, 10.0),
                (0.4, 1.0, 0.0, 64, 10, -1.0), (0.4, 1.0, float("nan"), 64, 10, 10.0)):
        with pytest.raises(ValueError):
            oracle.geometry(*bad)


# ---------------------------------------------------------------- eq.(4) by hand
def test_lens_equation_worked_by_hand():
    """eq.(4) PAPER.md:51.  One unit lens at (1,2), ray at (4,6): d = (3,4), |d|^2 = 25,
    deflection (0.12, 0.16).  With gamma = 0.3, sigma_c = 0.2:
    y = ((1-0.3-0.2)*4 - 0.12, (1+0.3-0.2)*6 - 0.16) = (1.88, 6.44).
    Catches 1/r for 1/r^2, a sign, swapped components, gamma on the wrong axis."""
    y = oracle.deflect_points(0.3, 0.2, [[1.0, 2.0]], [[4.0, 6.0]])
    assert np.allclose(y, [[1.88, 6.44]], rtol=0, atol=1e-14)
    # no lenses: pure macro model
    y = oracle.deflect_points(0.3, 0.2, np.zeros((0, 2)), [[2.0, 3.0]])
    assert np.allclose(y, [[1.0, 3.3]], rtol=0, atol=1e-14)
    # two lenses add linearly (m_i = 1): second lens at (4,3), d = (0,3), deflection (0, 1/3)
    y = oracle.deflect_points(0.0, 0.0, [[1.0, 2.0], [4.0, 3.0]], [[4.0, 6.0]])
    assert np.allclose(y, [[4 - 0.12, 6 - 0.16 - 1 / 3]], rtol=0, atol=1e-14)


def test_ring_of_lenses_obeys_the_2d_gauss_theorem():
    """n unit lenses equally spaced on a circle of radius R deflect like nothing inside it
    and like a mass n at the centre outside it, up to (r/R)^n resp. (R/r)^n: with
    z = x1 + i x2 the sum is conj(n z^(n-1)/(z^n - R^n)).  A dropped lens, a wrong index or
    a transposed component breaks it."""
    n, R = 64, 10.0
    th = 2 * np.pi * (np.arange(n) + 0.25) / n
    ring = np.stack([R * np.cos(th), R * np.sin(th)], axis=1)
    inside = np.array([[3.0, -2.0], [-1.5, 4.0], [0.0, 0.0]])
    y = oracle.deflect_points(0.0, 0.0, ring, inside)
    assert np.abs(y - inside).max() < 1e-11
    outside = np.array([[25.0, 7.0], [-3.0, -30.0]])
    y = oracle.deflect_points(0.0, 0.0, ring, outside)
    alpha = n * outside / (outside ** 2).sum(axis=1, keepdims=True)
    assert np.abs((outside - y) - alpha).max() < 1e-11
    # exact closed form at a point where neither limit applies
    z = complex(8.0, 5.0)
    w = complex(R * math.cos(th[0]), R * math.sin(th[0]))
    s = (n * z ** (n - 1) / (z ** n - w ** n)).conjugate()
    y = oracle.deflect_points(0.0, 0.0, ring, [[z.real, z.imag]])
    assert abs((z.real - y[0, 0]) - s.real) < 1e-11 and abs((z.imag - y[0, 1]) - s.imag) < 1e-11


# ---------------------------------------------------------------- (a) no stars: eq.(12)
@pytest.mark.parametrize("sigma,gamma,n_pix,values", [
    (0.4, 0.0, 128, {256, 272, 289}),   # r1 = r2 = 10/0.6 = 16.67 -> {16,17}^2
    (0.6, 0.2, 128, {800, 850}),        # r1 = 10/0.2 = 50, r2 = 10/0.6 -> 50*{16,17}
    (0.8, 0.3, 64, {2000}),             # r1 = 100, r2 = 20: commensurate
])
def test_no_stars_gives_the_uniform_map_of_eq12(sigma, gamma, n_pix, values):
    """Without compact lenses (stellar fraction 0) a regular grid puts
    sqrt(N_rays)/|1-sigma-/+gamma| rays per pixel per axis, so counts are products of
    floor/ceil of those (exactly N_rays*|mu| when commensurate) and the mean
    magnification is eq.(12) PAPER.md:289.  Catches wrong delta, rectangle, macro terms
    and binning."""
    m, st = oracle.shoot(sigma, 0.0, gamma, n_pix, 100.0, 10.0, np.zeros((0, 2)))
    assert set(np.unique(m).tolist()) == values
    mu_th = 1.0 / abs((1 - sigma) ** 2 - gamma ** 2)
    assert abs(m.mean() / 100.0 / mu_th - 1) < 1e-3
    assert st["rays_in_map"] == int(m.sum()) and st["rays_dropped"] == 0
    # the rectangle is 1.2x the minimal one per side: 1/1.44 of the rays land in the map
    assert abs(st["rays_in_map"] / st["rays_shot"] - 1 / 1.44) < 2e-3


def test_no_stars_map_is_flipped_not_scrambled_for_negative_parity():
    """sigma=0.8, gamma=0.3: 1-sigma-gamma = -0.1 (PAPER.md:292 parity flip).  Ray i=0 sits
    at the most negative x1 and must land at the most positive y1 column it can reach."""
    g = oracle.geometry(0.8, 0.0, 0.3, 64, 100.0, 10.0)
    y = oracle.probe(0.8, 0.0, 0.3, 64, 100.0, 10.0, np.zeros((0, 2)), [0, g.n1 - 1], [0, 0])
    assert y[0, 0] > 0 > y[1, 0] and y[0, 1] < 0 and y[1, 1] < 0
    assert abs(y[0, 0] - 0.1 * g.a1) < g.delta and abs(y[0, 1] + 0.5 * g.a2) < g.delta


# ---------------------------------------------------------------- (b) one isolated lens
def test_single_lens_matches_point_lens_magnification():
    """north_star (b): one lens at the origin, no convergence, no shear.  The map must follow
    A(u) = (u^2+2)/(u sqrt(u^2+4)) averaged over each pixel, away from the caustic (u > 1).
    The regular grid makes per-pixel sampling noise of a few %, so compare 8x8-block
    averages (tolerance 0.5 %, SURVEY.md section 8(c) pin b) and the map integral."""
    n_pix, n_rays, L = 128, 100.0, 10.0
    m, st = oracle.shoot(0.0, 1.0, 0.0, n_pix, n_rays, L, [[0.0, 0.0]])
    assert st["rays_shot"] == 1536 * 1536
    pix = L / n_pix
    c = (np.arange(n_pix) + 0.5) * pix - L / 2
    sub = (np.arange(16) + 0.5) / 16 - 0.5
    u1 = c[None, :, None, None] + sub[None, None, None, :] * pix
    u2 = c[:, None, None, None] + sub[None, None, :, None] * pix
    u = np.sqrt(u1 ** 2 + u2 ** 2)
    A = ((u * u + 2) / (u * np.sqrt(u * u + 4))).mean(axis=(2, 3))
    mu = m / n_rays

    def blocks(z):
        return z.reshape(16, 8, 16, 8).mean(axis=(1, 3))

    uc = np.sqrt(c[None, :] ** 2 + c[:, None] ** 2)
    far = blocks(uc) > 1.4
    rel = (blocks(mu) / blocks(A) - 1)[far]
    assert np.abs(rel).max() < 5e-3 and rel.std() < 2e-3
    assert abs(mu.sum() / A.sum() - 1) < 5e-4
    # the map is symmetric under both mirrors and the transpose (lens at the centre)
    assert np.array_equal(m, m[:, ::-1]) and np.array_equal(m, m[::-1, :]) and np.array_equal(m, m.T)


# ---------------------------------------------------------------- (c) (d) (e) (g) config 1
@pytest.fixture(scope="module")
def c1():
    c = CONFIGS[0]
    g = oracle.geometry(c.sigma, c.stellar_fraction, c.gamma, c.n_pix, c.n_rays, c.L)
    xy = lens_disk(g.n_star, g.r_star, c.seed)
    m, st = oracle.shoot(c.sigma, c.stellar_fraction, c.gamma, c.n_pix, c.n_rays, c.L, xy)
    return c, g, xy, m, st


def test_c1_conservation_and_mean(c1):
    c, g, xy, m, st = c1
    assert st["rays_shot"] == g.n1 * g.n2 == 6553600
    assert st["rays_shot"] == st["rays_in_map"] + st["rays_out_of_map"] + st["rays_dropped"]
    assert int(m.sum(dtype=np.int64)) == st["rays_in_map"]
    assert st["interactions"] == 6553600 * 135
    # north_star (d): map mean vs eq.(12).  A sanity band, not a precision pin: a 10 R_E map
    # holds few caustics, so the sample variance of the lens field dominates (SURVEY section 8(c) d).
    ratio = m.mean() / c.n_rays / abs(g.mu_th)
    assert 0.6 < ratio < 1.1


def test_c1_equals_an_independent_numpy_brute_force(c1):
    """Pin (g)/(e): a second implementation, array-wise numpy, must give the same integers.
    Also fixes the worked-example numbers of SURVEY.md section 8(c) (e), which came from a third
    (survey-time) script: in-map 4 012 112, max 2351, min 75, sum of squares 1 636 545 372."""
    c, g, xy, m, st = c1
    assert np.allclose(xy[0], (-12.5297296, 7.63537337), atol=1e-7)
    assert np.allclose(xy[-1], (9.87350103, 0.01865395), atol=1e-7)
    ref, shot, n_in = shoot_numpy(c.sigma, c.stellar_fraction, c.gamma, c.n_pix, c.n_rays, c.L, xy)
    assert shot == st["rays_shot"] and n_in == st["rays_in_map"] == 4012112
    assert np.array_equal(ref, m.astype(np.int64))
    assert int(m.max()) == 2351 and int(m.min()) == 75
    assert int((m.astype(np.int64) ** 2).sum()) == 1636545372


def test_tiny_case_with_shear_and_smooth_matter_equals_brute_force():
    """n_pix = 8, N_rays = 4, 3 lenses, gamma and sigma_c both non-zero and the grid ragged
    (2a/delta not an integer)."""
    xy = np.array([[0.3, -0.2], [-1.1, 0.9], [2.0, 1.5]])
    args = (0.55, 0.4, 0.15, 8, 4.0, 6.0)
    m, st = oracle.shoot(*args, xy)
    ref, shot, n_in = shoot_numpy(*args, xy)
    assert shot == st["rays_shot"] and n_in == st["rays_in_map"]
    assert np.array_equal(ref, m.astype(np.int64))


# ---------------------------------------------------------------- (f) symmetries
def test_mirror_and_transpose_symmetries_are_exact():
    """The grid is symmetric about the origin, so mirroring the lenses in x1 mirrors the map in
    i', and swapping the lens axes together with gamma -> -gamma transposes it.  Catches
    axis / sign / layout slips that the scalar pins cannot see."""
    args = dict(sigma=0.5, stellar_fraction=0.8, gamma=0.2, n_pix=32, n_rays=16.0, L=8.0)
    g = oracle.geometry(**args)
    xy = lens_disk(g.n_star, g.r_star, 11)
    m, _ = oracle.shoot(lens_xy=xy, **args)
    assert m.sum() > 0 and not np.array_equal(m, m[:, ::-1])
    mx, _ = oracle.shoot(lens_xy=xy * np.array([-1.0, 1.0]), **args)
    assert np.array_equal(mx, m[:, ::-1])
    my, _ = oracle.shoot(lens_xy=xy * np.array([1.0, -1.0]), **args)
    assert np.array_equal(my, m[::-1, :])
    args_t = dict(args, gamma=-0.2)
    mt, _ = oracle.shoot(lens_xy=xy[:, ::-1].copy(), **args_t)
    assert np.array_equal(mt, m.T)


# ---------------------------------------------------------------- regions, capture, probe agree
def test_regions_tile_the_full_map_and_capture_probe_agree():
    """shoot = sum of shoot_region over any tiling; capture/probe/pixels_of describe the same
    rays.  (Consistency of the oracle's entry points, so that GPU parity on sub-regions speaks
    for the full map.)"""
    args = dict(sigma=0.45, stellar_fraction=1.0, gamma=0.1, n_pix=24, n_rays=9.0, L=6.0)
    g = oracle.geometry(**args)
    xy = lens_disk(g.n_star, g.r_star, 5)
    full, st = oracle.shoot(lens_xy=xy, **args)
    acc = np.zeros_like(full)
    tot = 0
    isplit, jsplit = [0, 37, g.n1], [0, 5, 64, g.n2]
    for a, b in zip(isplit[:-1], isplit[1:]):
        for c_, d in zip(jsplit[:-1], jsplit[1:]):
            _, s = oracle.shoot_region(lens_xy=xy, region=(a, b, c_, d), map_out=acc, **args)
            tot += s["rays_shot"]
    assert tot == st["rays_shot"] and np.array_equal(acc, full)
    reg = (3, 40, 7, 29)
    cap = oracle.capture_region(lens_xy=xy, region=reg, **args)
    pix = oracle.pixels_of(y=cap, **args)
    part, s = oracle.shoot_region(lens_xy=xy, region=reg, **args)
    ok = pix >= 0
    assert ok.sum() == s["rays_in_map"]
    assert np.array_equal(np.bincount(pix[ok], minlength=24 * 24).reshape(24, 24), part)
    ii, jj = np.meshgrid(np.arange(reg[0], reg[1]), np.arange(reg[2], reg[3]))
    pr = oracle.probe(lens_xy=xy, ray_i=ii.ravel(), ray_j=jj.ravel(), **args)
    assert np.array_equal(pr.reshape(cap.shape), cap)


def test_ray_on_a_lens_is_dropped_not_binned():
    """Reading R12: |x - x_i|^2 = 0 -> the ray is counted as dropped and poisons nothing."""
    args = dict(sigma=0.0, stellar_fraction=1.0, gamma=0.0, n_pix=16, n_rays=4.0, L=4.0)
    g = oracle.geometry(**args)
    i, j = 5, 9
    x = np.array([[(i - (g.n1 - 1) / 2) * g.delta, (j - (g.n2 - 1) / 2) * g.delta]])
    m, st = oracle.shoot(lens_xy=x, **args)
    assert st["rays_dropped"] == 1
    assert st["rays_shot"] == st["rays_in_map"] + st["rays_out_of_map"] + 1
    assert int(m.sum()) == st["rays_in_map"]


# ---------------------------------------------------------------- input generator
def test_lens_disk_is_uniform_in_the_disk():
    xy = lens_disk(200000, 7.0, 3)
    r = np.hypot(xy[:, 0], xy[:, 1])
    assert r.max() <= 7.0
    assert abs((r < 7.0 / math.sqrt(2)).mean() - 0.5) < 5e-3     # equal areas
    assert np.abs(xy.mean(axis=0)).max() < 0.05
    q = ((xy[:, 0] > 0) & (xy[:, 1] > 0)).mean()
    assert abs(q - 0.25) < 5e-3
    assert np.array_equal(xy, lens_disk(200000, 7.0, 3)) and not np.array_equal(xy, lens_disk(200000, 7.0, 4))
