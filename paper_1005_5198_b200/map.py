"""Convenience object around one ml_ctx: owns the handle, forwards to the C calls."""
from __future__ import annotations

from . import binding as _b


class MagnificationMap:
    """One magnification map (eq.3): create, set lenses, shoot, read counts.

    All work is done by the C library; this class only keeps the handle alive.
    """

    def __init__(self, sigma, stellar_fraction, gamma, n_pix, n_rays, L, device=0,
                 precision=_b.ML_PREC_FP32_TILED):
        self._ctx = _b.ml_create(sigma, stellar_fraction, gamma, n_pix, n_rays, L, device)
        self.n_rays = float(n_rays)
        if precision != _b.ML_PREC_FP32_TILED:
            _b.ml_set_precision(self._ctx, precision)

    # -- lifetime
    def close(self):
        if self._ctx is not None:
            _b.ml_destroy(self._ctx)
            self._ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- forwards
    @property
    def ctx(self):
        return self._ctx

    @property
    def info(self) -> dict:
        return _b.ml_get_info(self._ctx)

    @property
    def stats(self) -> dict:
        return _b.ml_get_stats(self._ctx)

    def set_lenses(self, xy, mass=None):
        if mass is None:
            _b.ml_set_lenses(self._ctx, xy)
        else:
            _b.ml_set_lens_masses(self._ctx, xy, mass)

    def set_ray_mode(self, mode, seed=0):
        _b.ml_set_ray_mode(self._ctx, mode, seed)

    def set_precision(self, mode):
        _b.ml_set_precision(self._ctx, mode)

    def attach_stream(self, cuda_stream):
        _b.ml_attach_stream(self._ctx, cuda_stream)

    def use_device_map(self, dptr):
        _b.ml_use_device_map(self._ctx, dptr)

    def shoot(self):
        _b.ml_shoot(self._ctx)

    def shoot_region(self, i0, i1, j0, j1, accumulate=False):
        _b.ml_shoot_region(self._ctx, i0, i1, j0, j1, accumulate)

    def counts(self, out=None):
        return _b.ml_get_map(self._ctx, out)

    def capture_region(self, i0, i1, j0, j1):
        return _b.ml_capture_region(self._ctx, i0, i1, j0, j1)

    def probe(self, ray_i, ray_j):
        return _b.ml_probe(self._ctx, ray_i, ray_j)
