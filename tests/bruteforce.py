"""A second, independent restatement of inverse ray-shooting (numpy, fp64).

Used only to pin the C oracle (SURVEY.md section 8(c) pin (g)): it is written array-wise
(whole rows of rays at once, lens by lens) from PAPER.md eq.(3)-(4) and the rules
of BASELINE.json:configs[0]; it shares nothing with oracle/microlens_oracle.c.
"""
import math

import numpy as np


def shoot_numpy(sigma, f_star, gamma, n_pix, n_rays, L, lens_xy, rows=256, mass=None):
    kc = sigma - sigma * f_star
    pix = L / n_pix
    d = pix / math.sqrt(n_rays)
    a1 = 1.2 * (L / 2) / abs(1 - sigma - gamma)
    a2 = 1.2 * (L / 2) / abs(1 - sigma + gamma)
    n1 = math.ceil(2 * a1 / d - 1e-9)
    n2 = math.ceil(2 * a2 / d - 1e-9)
    x1 = (np.arange(n1) - (n1 - 1) / 2) * d
    x2 = (np.arange(n2) - (n2 - 1) / 2) * d
    counts = np.zeros(n_pix * n_pix, dtype=np.int64)
    n_in = 0
    for j0 in range(0, n2, rows):
        X, Y = np.meshgrid(x1, x2[j0:j0 + rows])
        ax = np.zeros_like(X)
        ay = np.zeros_like(X)
        lenses = np.asarray(lens_xy, dtype=np.float64).reshape(-1, 2)
        masses = np.ones(len(lenses)) if mass is None else np.asarray(mass, dtype=np.float64)
        for (lx, ly), m in zip(lenses, masses):
            dx = X - lx
            dy = Y - ly
            r2 = dx * dx + dy * dy
            if mass is None:
                ax += dx / r2
                ay += dy / r2
            else:           # eq.(4) with its m_i
                ax += m * dx / r2
                ay += m * dy / r2
        y1 = (1 - gamma) * X - kc * X - ax
        y2 = (1 + gamma) * Y - kc * Y - ay
        ii = np.floor((y1 + L / 2) / pix)
        jj = np.floor((y2 + L / 2) / pix)
        ok = (ii >= 0) & (ii < n_pix) & (jj >= 0) & (jj < n_pix)
        flat = (jj[ok] * n_pix + ii[ok]).astype(np.int64)
        counts += np.bincount(flat, minlength=n_pix * n_pix)
        n_in += int(ok.sum())
    return counts.reshape(n_pix, n_pix), n1 * n2, n_in
