"""Make one magnification map from the command line (argument marshalling and file output only; every step of
the computation runs in the CUDA library).

    python -m paper_1005_5198_b200.cli --sigma 0.4 --gamma 0 --n-pix 1024 --n-rays 2000 --L 20 \
        [--stellar-fraction 1] [--lenses lenses.txt | --seed 1] [--masses masses.txt] \
        [--precision fp32_tiled|fp32_compensated|fp64] [--random-rays SEED] [--out map.npy] [--pgm map.pgm]

The arguments are the paper's statement of the problem.  Lens positions are read from a
text file of "x y" pairs in Einstein radii (the paper reads them from a file too) or, without one,
drawn uniformly in the lens disk of radius R* with numpy's PCG64 and the given seed.  --out writes the raw uint32
counts N_ij (mu_ij = N_ij / N_rays, eq. 3); --pgm writes an 8-bit greyscale picture like the paper's Fig. 1
(PAPER.md:23-25).  The picture is PRESENTATION ONLY: its grey levels are a numpy rendering of the counts on the host
(Delta m of eq. 10 clipped to +-3 mag); the method's own Delta m statistics (histogram, RMS, K-S test) are the library
calls ml_delta_m_histogram / ml_map_compare, and --dm-hist prints the former.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np

from . import binding as _b
from .map import MagnificationMap

PRECISIONS = {"fp32_tiled": _b.ML_PREC_FP32_TILED, "fp32_compensated": _b.ML_PREC_FP32_COMPENSATED,
              "fp64": _b.ML_PREC_FP64}


def _disk(n, radius, seed):
    """The repo's seeded synthetic lens field (workloads/lens_fields.py: the stand-in for the paper's lens files)."""
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    from workloads import lens_disk
    return lens_disk(n, radius, seed)


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--sigma", type=float, required=True, help="total convergence")
    ap.add_argument("--gamma", type=float, default=0.0, help="external shear")
    ap.add_argument("--stellar-fraction", type=float, default=1.0, help="sigma_* / sigma = 1 - s")
    ap.add_argument("--n-pix", type=int, required=True, help="pixels per side")
    ap.add_argument("--n-rays", type=float, required=True, help="mean rays per pixel without lensing")
    ap.add_argument("--L", type=float, required=True, help="source-plane side length, Einstein radii")
    ap.add_argument("--lenses", help="text file of lens positions, one 'x y' per line")
    ap.add_argument("--masses", help="text file of lens masses, one per line (default: unit masses)")
    ap.add_argument("--seed", type=int, default=0, help="seed of the synthetic lens disk when --lenses is absent")
    ap.add_argument("--precision", default="fp32_tiled", choices=sorted(PRECISIONS))
    ap.add_argument("--random-rays", type=int, default=None, metavar="SEED", help="random ray positions (GPU-D's way)")
    ap.add_argument("--uniform-rays", type=int, default=None, metavar="SEED",
                    help="every ray an independent uniform point of the shooting rectangle (Poisson noise, PAPER.md:167)")
    ap.add_argument("--device", type=int, default=0)
    ap.add_argument("--out", help="write the uint32 counts to this .npy file")
    ap.add_argument("--pgm", help="write a greyscale picture of Delta m to this .pgm file (presentation only)")
    ap.add_argument("--dm-hist", type=int, default=0, metavar="BINS",
                    help="print the Delta m histogram over [-3, 3) mag relative to mu_th (ml_delta_m_histogram)")
    a = ap.parse_args(argv)

    with MagnificationMap(a.sigma, a.stellar_fraction, a.gamma, a.n_pix, a.n_rays, a.L, device=a.device,
                          precision=PRECISIONS[a.precision]) as m:
        info = m.info
        xy = np.loadtxt(a.lenses, ndmin=2)[:, :2] if a.lenses else _disk(info["n_star_expected"], info["r_star"], a.seed)
        mass = np.loadtxt(a.masses, ndmin=1) if a.masses else None
        m.set_lenses(xy, mass)
        if a.random_rays is not None:
            m.set_ray_mode(_b.ML_RAYS_RANDOM, a.random_rays)
        if a.uniform_rays is not None:
            m.set_ray_mode(_b.ML_RAYS_UNIFORM, a.uniform_rays)
        m.shoot()
        st, counts = m.stats, m.counts()
    mu_mean = float(counts.mean()) / a.n_rays
    print("lenses %d  rays %d x %d = %d  in map %d  dropped %d" % (xy.shape[0], info["n1"], info["n2"], st["rays_shot"],
                                                                  st["rays_in_map"], st["rays_dropped"]))
    print("kernel %.3f ms  %.4e lens-ray interactions/s  mean mu %.5f  (1/((1-sigma)^2-gamma^2) = %.5f)"
          % (st["kernel_ms"], st["interactions"] / max(st["kernel_ms"], 1e-9) * 1e3, mu_mean, info["mu_theory"]))
    if a.dm_hist > 0:
        # Delta m relative to the theoretical mean: count / (n_rays |mu_th|)
        h = _b.ml_delta_m_histogram(counts, a.n_rays * abs(info["mu_theory"]), -3.0, 3.0, a.dm_hist, device=a.device)
        w = 6.0 / a.dm_hist
        for k, v in enumerate(h):
            print("dm [%+.3f, %+.3f)  %d" % (-3.0 + k * w, -3.0 + (k + 1) * w, int(v)))
    if a.out:
        np.save(a.out, counts)
    if a.pgm:
        with np.errstate(divide="ignore"):
            dm = -2.5 * np.log10(counts / a.n_rays / abs(info["mu_theory"]))
        dm = np.clip(dm, -3.0, 3.0)                     # bright (negative Delta m) = white
        img = np.round((3.0 - dm) / 6.0 * 255.0).astype(np.uint8)[::-1]
        with open(a.pgm, "wb") as f:
            f.write(b"P5\n%d %d\n255\n" % (a.n_pix, a.n_pix))
            f.write(img.tobytes())
    return 0


if __name__ == "__main__":
    sys.exit(main())
