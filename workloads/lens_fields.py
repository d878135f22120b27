"""Synthetic lens fields and ray samples shaped like the paper's parameter space.

The paper's maps were made from lens-position files written by a tree-code run
(PAPER.md:138); those files are not available, so the inputs are synthetic:
unit-mass lenses drawn uniformly in a disk ("distributed in a
circle of area A"), seeded, with the problem statements of
BASELINE.json:configs (sigma, gamma, stellar fraction, L, N_pix, N_rays taken
from PAPER.md:152-158, :25, :308, :316).

Nothing here computes anything the method computes.  The disk radius and the
lens count are ARGUMENTS: the caller gets them from its own geometry code
(`oracle.geometry(...)` on the oracle side, `ml_get_info` on the CUDA side).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Problem:
    """The paper's statement of one map: raw inputs only."""

    name: str
    sigma: float             # total convergence
    gamma: float             # external shear
    stellar_fraction: float  # sigma_* / sigma  (= 1 - s, s = PAPER.md:158)
    L: float                 # source-plane side length, Einstein radii
    n_pix: int               # pixels per side
    n_rays: float            # mean rays per pixel in the absence of lensing
    seed: int                # lens-field seed


# BASELINE.json:configs, in order.  configs[0] is the seconds-on-CPU case,
# configs[1] the paper's Fig. 1 shape and the bench workload.
CONFIGS = (
    Problem("C1", 0.4, 0.0, 1.0, 10.0, 128, 100.0, 0),
    Problem("C2", 0.4, 0.0, 1.0, 20.0, 1024, 2000.0, 1),
    Problem("C3", 0.8, 0.3, 1.0, 20.0, 1024, 100.0, 2),
    Problem("C4", 0.4, 0.4, 1.0, 40.0, 4096, 100.0, 3),
    Problem("C5", 0.6, 0.2, 0.3, 20.0, 2048, 500.0, 4),
)


def lens_disk(n_star: int, r_star: float, seed: int) -> np.ndarray:
    """n_star points uniform in the disk of radius r_star about the origin.

    Returns a C-contiguous float64 array of shape (n_star, 2), interleaved
    (x, y) -- the layout both `ml_set_lenses` and the oracle take.
    Recipe (SURVEY.md section 8(c) point 5): PCG64 `default_rng(seed)`, all radii
    first, then all angles.
    """
    rng = np.random.default_rng(seed)
    u = rng.random(n_star)
    v = rng.random(n_star)
    r = r_star * np.sqrt(u)
    th = 2.0 * np.pi * v
    xy = np.empty((n_star, 2), dtype=np.float64)
    xy[:, 0] = r * np.cos(th)
    xy[:, 1] = r * np.sin(th)
    return xy


def lens_masses(n_star: int, seed: int) -> np.ndarray:
    """n_star seeded lens masses for the unequal-mass row (eq. 4's m_i).

    The paper sets all masses equal and names no spectrum; this stand-in is a
    log-uniform spectrum over a decade, 0.3 ... 3 in units of the reference mass, the range a stellar
    population would span.  Mean ~ 1.17; the caller uses the sample mean as <M> in eq. 5.
    """
    rng = np.random.default_rng(3000 + seed)
    return 0.3 * 10.0 ** rng.random(n_star)


def parity_tiles(n1: int, n2: int, n_tiles: int, side: int, seed: int):
    """Seeded ray-index sub-rectangles [i0,i1) x [j0,j1) inside the n1 x n2 grid.

    The first four touch the four edges of the shooting rectangle (ragged
    tails live there); the rest are uniform.  Offsets are deliberately NOT
    aligned to any kernel tile size.
    """
    rng = np.random.default_rng(1000 + seed)
    w = min(side, n1)
    h = min(side, n2)
    out = []
    for t in range(n_tiles):
        i0 = int(rng.integers(0, n1 - w + 1))
        j0 = int(rng.integers(0, n2 - h + 1))
        if t == 0:
            i0 = 0
        elif t == 1:
            i0 = n1 - w
        elif t == 2:
            j0 = 0
        elif t == 3:
            j0 = n2 - h
        out.append((i0, i0 + w, j0, j0 + h))
    return out


def probe_rays(n1: int, n2: int, n: int, seed: int, regions=None):
    """n seeded ray indices (int64 arrays i, j).

    With `regions` (a list from `parity_tiles`) the rays are drawn inside those
    rectangles, round-robin; otherwise anywhere in the grid.
    """
    rng = np.random.default_rng(2000 + seed)
    if not regions:
        return (rng.integers(0, n1, n, dtype=np.int64),
                rng.integers(0, n2, n, dtype=np.int64))
    ri = np.empty(n, dtype=np.int64)
    rj = np.empty(n, dtype=np.int64)
    for k in range(n):
        i0, i1, j0, j1 = regions[k % len(regions)]
        ri[k] = rng.integers(i0, i1)
        rj[k] = rng.integers(j0, j1)
    return ri, rj
