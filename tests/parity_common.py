"""Shared helpers of the -m gpu parity tests: build the same problem on both sides
(CUDA library through its C ABI, fp64 CPU oracle) and evaluate the four criteria of
BASELINE.json:north_star.  No arithmetic of the method lives here: pixels are derived
with the oracle's own floor rule (oracle.pixels_of), maps come from each side.
"""
from __future__ import annotations

import os

import numpy as np

import paper_1005_5198_b200 as ml
from oracle import oracle
from workloads import lens_disk, parity_tiles

# north_star tolerances
TOL_POSITION_PIXELS = 1e-3      # |y_gpu - y_oracle| <= 1e-3 pixel widths on sampled rays
MIN_SAME_PIXEL = 0.9999         # >= 99.99 % of rays land in the oracle's pixel
TOL_INMAP_REL = 1e-5            # total in-map counts
TOL_BLOCK_MU = 1e-3             # |mu_gpu - mu_oracle| on 8x8-block averages

# interactions the oracle may spend per config on sub-region parity (about 10 s on 8 cores)
ORACLE_BUDGET = float(os.environ.get("ML_PARITY_BUDGET", "6e9"))


def problem_args(p):
    return (p.sigma, p.stellar_fraction, p.gamma, p.n_pix, p.n_rays, p.L)


def make_pair(p, precision=ml.ML_PREC_FP32_TILED, lenses=None):
    """(MagnificationMap, oracle geometry, lens array) for Problem p.  Each side derives
    its own geometry; they must agree before anything else is compared."""
    m = ml.MagnificationMap(*problem_args(p), precision=precision)
    g = oracle.geometry(*problem_args(p))
    info = m.info
    assert (info["n1"], info["n2"], info["n_star_expected"]) == (g.n1, g.n2, g.n_star)
    for a, b in (("a1", "a1"), ("a2", "a2"), ("ray_spacing", "delta"), ("r_star", "r_star"),
                 ("kappa_star", "kappa_star"), ("kappa_c", "kappa_c"), ("pixel_side", "pixel"),
                 ("mu_theory", "mu_th")):
        assert info[a] == getattr(g, b), (a, info[a], getattr(g, b))
    xy = lens_disk(g.n_star, g.r_star, p.seed) if lenses is None else np.asarray(lenses, dtype=np.float64)
    m.set_lenses(xy)
    return m, g, xy


def block_mu(counts, n_rays, block=8):
    n = counts.shape[0]
    assert n % block == 0
    c = counts.astype(np.float64).reshape(n // block, block, n // block, block)
    return c.mean(axis=(1, 3)) / n_rays


def check_maps(p, gpu_map, gpu_stats, ora_map, ora_stats):
    """Criteria 3 and 4 plus conservation.  Returns the figures for reporting."""
    assert int(gpu_stats["rays_shot"]) == ora_stats["rays_shot"]
    assert int(gpu_map.sum(dtype=np.uint64)) == int(gpu_stats["rays_in_map"])
    n_in_o = ora_stats["rays_in_map"]
    rel = abs(int(gpu_stats["rays_in_map"]) - n_in_o) / max(n_in_o, 1)
    assert rel <= TOL_INMAP_REL, ("in-map counts", gpu_stats["rays_in_map"], n_in_o, rel)
    d = np.abs(block_mu(gpu_map, p.n_rays) - block_mu(ora_map, p.n_rays)).max()
    assert d <= TOL_BLOCK_MU, ("8x8 block mu", d)
    return {"inmap_rel": rel, "block_mu_max": float(d),
            "pixels_differing": int((gpu_map != ora_map).sum())}


def check_rays(p, g, y_gpu, y_ora):
    """Criteria 1 and 2 on per-ray source-plane positions (same rays, same order)."""
    y_gpu = y_gpu.reshape(-1, 2)
    y_ora = y_ora.reshape(-1, 2)
    ok = np.isfinite(y_ora).all(axis=1)
    assert np.isfinite(y_gpu[ok]).all()
    pix_o = oracle.pixels_of(*problem_args(p), y_ora)
    pix_g = oracle.pixels_of(*problem_args(p), y_gpu)
    same = float((pix_o == pix_g).mean())
    # position criterion on rays that matter for the map: inside it or within one map side of it
    near = ok & (np.abs(y_ora) <= 1.5 * p.L).all(axis=1)
    err = np.abs(y_gpu[near] - y_ora[near]).max() / g.pixel if near.any() else 0.0
    assert err <= TOL_POSITION_PIXELS, ("position error / pixel", err)
    assert same >= MIN_SAME_PIXEL, ("same-pixel fraction", same)
    return {"same_pixel": same, "pos_err_pixels": float(err), "rays": int(y_ora.shape[0])}


def subregion_tiles(p, g, n_lens):
    """Seeded ray sub-rectangles whose total oracle cost stays within ORACLE_BUDGET."""
    side = 512 if n_lens < 4000 else 256
    n_tiles = int(ORACLE_BUDGET / (max(n_lens, 1) * side * side))
    n_tiles = max(4, min(32, n_tiles))
    return parity_tiles(g.n1, g.n2, n_tiles, side, p.seed)
