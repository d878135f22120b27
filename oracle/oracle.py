"""ctypes front end of the fp64 CPU oracle (oracle/microlens_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_1005_5198_b200/ and the package never imports it.

Every function is argument marshalling around the C routine of the same name;
the arithmetic, with its PAPER.md citations, lives in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "microlens_oracle.c")
_LIB = os.path.join(_HERE, "libmloracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no -march flags: the .so must run on any x86-64 box)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
             "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [("sigma", C.c_double), ("stellar_fraction", C.c_double), ("gamma", C.c_double),
                ("n_pix", C.c_int32), ("n_rays", C.c_double), ("L", C.c_double),
                ("ray_mode", C.c_int32), ("ray_seed", C.c_uint64)]


class _Geometry(C.Structure):
    _fields_ = [("kappa_star", C.c_double), ("kappa_c", C.c_double), ("pixel", C.c_double),
                ("delta", C.c_double), ("a1", C.c_double), ("a2", C.c_double),
                ("r_star", C.c_double), ("mu_th", C.c_double),
                ("n1", C.c_int64), ("n2", C.c_int64), ("n_star", C.c_int64)]


@dataclass(frozen=True)
class Geometry:
    kappa_star: float
    kappa_c: float
    pixel: float
    delta: float
    a1: float
    a2: float
    r_star: float
    mu_th: float
    n1: int
    n2: int
    n_star: int


_lib = None


def _load():
    global _lib
    if _lib is None:
        # ML_ORACLE_LIBRARY: another build of the same C file (tests/test_oracle_sanitizers.py loads an ASan/UBSan one)
        lib = C.CDLL(os.environ.get("ML_ORACLE_LIBRARY") or build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int64)
        pp = C.POINTER(_Problem)
        lib.ora_n_star.restype = C.c_int64
        lib.ora_n_star.argtypes = [C.c_double, C.c_double]
        lib.ora_derive.argtypes = [pp, C.POINTER(_Geometry)]
        lib.ora_shoot_region.argtypes = [pp, dp, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                         C.c_int64, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)]
        lib.ora_capture_region.argtypes = [pp, dp, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                           C.c_int64, dp]
        lib.ora_probe.argtypes = [pp, dp, C.c_int64, C.c_int64, ip, ip, dp]
        lib.ora_deflect_points.argtypes = [C.c_double, C.c_double, dp, C.c_int64, C.c_int64, dp, dp]
        lib.ora_pixels_of.argtypes = [pp, C.c_int64, dp, ip]
        lib.ora_ray_positions.argtypes = [pp, C.c_int64, ip, ip, dp]
        lib.ora_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        lib.ora_philox4x32_10.restype = None
        lib.ora_ray_uniforms.argtypes = [C.c_uint64, C.c_uint64, dp]
        lib.ora_ray_uniforms.restype = None
        lib.ora_n_star_m.restype = C.c_int64
        lib.ora_n_star_m.argtypes = [C.c_double, C.c_double, C.c_double]
        lib.ora_shoot_region_m.argtypes = [pp, dp, dp, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                           C.c_int64, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)]
        lib.ora_capture_region_m.argtypes = [pp, dp, dp, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                             C.c_int64, dp]
        lib.ora_deflect_points_m.argtypes = [C.c_double, C.c_double, dp, dp, C.c_int64, C.c_int64, dp, dp]
        lib.ora_num_threads.restype = C.c_int
        _lib = lib
    return _lib


RAY_MODES = {"regular": 0, "cell": 1, "uniform": 2}


def _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L, ray_seed=None, ray_mode=None):
    """ray_seed = None: regular ray grid; an int: random rays -- ray_mode "cell" (default): one random position inside
    each grid cell (reading R17); "uniform": every ray an independent uniform point of the whole shooting rectangle
    (reading R20, the literal GPU-D generation of PAPER.md:131, :167)."""
    if ray_seed is None:
        assert ray_mode in (None, "regular")
        return _Problem(float(sigma), float(stellar_fraction), float(gamma), int(n_pix), float(n_rays), float(L), 0, 0)
    return _Problem(float(sigma), float(stellar_fraction), float(gamma), int(n_pix),
                    float(n_rays), float(L), RAY_MODES[ray_mode or "cell"], int(ray_seed))


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _lenses(lens_xy):
    a = np.ascontiguousarray(lens_xy, dtype=np.float64).reshape(-1, 2)
    return a, a.shape[0]


def _masses(mass, n):
    """None (unit masses, the paper's maps) or n positive masses m_i of eq. 4."""
    if mass is None:
        return None, None
    m = np.ascontiguousarray(mass, dtype=np.float64).ravel()
    assert m.size == n
    return m, _dptr(m)


def _check(rc, what):
    if rc != 0:
        raise ValueError("oracle %s: invalid argument" % what)


def num_threads() -> int:
    return int(_load().ora_num_threads())


def n_star(kappa_star: float, r_disk: float, mean_mass: float = None) -> int:
    """Eq. (5), with A = pi R^2 and <M> = 1 (or the given mean mass)."""
    if mean_mass is not None:
        return int(_load().ora_n_star_m(float(kappa_star), float(r_disk), float(mean_mass)))
    return int(_load().ora_n_star(float(kappa_star), float(r_disk)))


def geometry(sigma, stellar_fraction, gamma, n_pix, n_rays, L) -> Geometry:
    g = _Geometry()
    p = _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L)
    _check(_load().ora_derive(C.byref(p), C.byref(g)), "geometry")
    return Geometry(**{f: getattr(g, f) for f, _ in _Geometry._fields_})


def shoot_region(sigma, stellar_fraction, gamma, n_pix, n_rays, L, lens_xy,
                 region=None, map_out=None, mass=None, ray_seed=None, ray_mode=None):
    """Counts map (uint32, shape (n_pix, n_pix), [j', i']) and stats dict.

    region = (i0, i1, j0, j1) ray-index rectangle (default: the whole grid);
    map_out: existing map to accumulate into.
    """
    p = _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L, ray_seed, ray_mode)
    g = geometry(sigma, stellar_fraction, gamma, n_pix, n_rays, L)
    xy, n = _lenses(lens_xy)
    i0, i1, j0, j1 = region if region is not None else (0, g.n1, 0, g.n2)
    m = map_out if map_out is not None else np.zeros((n_pix, n_pix), dtype=np.uint32)
    assert m.dtype == np.uint32 and m.flags.c_contiguous and m.size == n_pix * n_pix
    st = np.zeros(4, dtype=np.uint64)
    mk, mp = _masses(mass, n)
    if mk is None:
        rc = _load().ora_shoot_region(C.byref(p), _dptr(xy), n, i0, i1, j0, j1,
                                      m.ctypes.data_as(C.POINTER(C.c_uint32)), st.ctypes.data_as(C.POINTER(C.c_uint64)))
    else:
        rc = _load().ora_shoot_region_m(C.byref(p), _dptr(xy), mp, n, i0, i1, j0, j1,
                                        m.ctypes.data_as(C.POINTER(C.c_uint32)), st.ctypes.data_as(C.POINTER(C.c_uint64)))
    _check(rc, "shoot_region")
    stats = {"rays_shot": int(st[0]), "rays_in_map": int(st[1]),
             "rays_out_of_map": int(st[2]), "rays_dropped": int(st[3]),
             "interactions": int(st[0]) * n}
    return m, stats


def shoot(sigma, stellar_fraction, gamma, n_pix, n_rays, L, lens_xy, mass=None, ray_seed=None, ray_mode=None):
    return shoot_region(sigma, stellar_fraction, gamma, n_pix, n_rays, L, lens_xy, mass=mass, ray_seed=ray_seed,
                        ray_mode=ray_mode)


def capture_region(sigma, stellar_fraction, gamma, n_pix, n_rays, L, lens_xy, region, mass=None, ray_seed=None,
                   ray_mode=None):
    """y of every ray in region, shape (j1-j0, i1-i0, 2)."""
    p = _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L, ray_seed, ray_mode)
    xy, n = _lenses(lens_xy)
    i0, i1, j0, j1 = region
    out = np.empty((j1 - j0, i1 - i0, 2), dtype=np.float64)
    mk, mp = _masses(mass, n)
    if mk is None:
        rc = _load().ora_capture_region(C.byref(p), _dptr(xy), n, i0, i1, j0, j1, _dptr(out))
    else:
        rc = _load().ora_capture_region_m(C.byref(p), _dptr(xy), mp, n, i0, i1, j0, j1, _dptr(out))
    _check(rc, "capture_region")
    return out


def probe(sigma, stellar_fraction, gamma, n_pix, n_rays, L, lens_xy, ray_i, ray_j):
    """y of the listed rays, shape (n, 2)."""
    p = _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L)
    xy, n = _lenses(lens_xy)
    ri = np.ascontiguousarray(ray_i, dtype=np.int64)
    rj = np.ascontiguousarray(ray_j, dtype=np.int64)
    out = np.empty((ri.size, 2), dtype=np.float64)
    ip = C.POINTER(C.c_int64)
    _check(_load().ora_probe(C.byref(p), _dptr(xy), n, ri.size, ri.ctypes.data_as(ip),
                             rj.ctypes.data_as(ip), _dptr(out)), "probe")
    return out


def deflect_points(gamma, kappa_c, lens_xy, x, mass=None):
    """Eq. (4) at arbitrary image-plane points x (n, 2) -> y (n, 2)."""
    xy, n = _lenses(lens_xy)
    xs = np.ascontiguousarray(x, dtype=np.float64).reshape(-1, 2)
    out = np.empty_like(xs)
    mk, mp = _masses(mass, n)
    if mk is None:
        rc = _load().ora_deflect_points(float(gamma), float(kappa_c), _dptr(xy), n, xs.shape[0], _dptr(xs), _dptr(out))
    else:
        rc = _load().ora_deflect_points_m(float(gamma), float(kappa_c), _dptr(xy), mp, n, xs.shape[0], _dptr(xs), _dptr(out))
    _check(rc, "deflect_points")
    return out


def pixels_of(sigma, stellar_fraction, gamma, n_pix, n_rays, L, y):
    """Flat pixel index j'*n_pix+i' of source positions y (..., 2); -1 = outside or NaN."""
    p = _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L)
    ys = np.ascontiguousarray(y, dtype=np.float64).reshape(-1, 2)
    out = np.empty(ys.shape[0], dtype=np.int64)
    _check(_load().ora_pixels_of(C.byref(p), ys.shape[0], _dptr(ys),
                                 out.ctypes.data_as(C.POINTER(C.c_int64))), "pixels_of")
    return out.reshape(np.asarray(y).shape[:-1])


def philox4x32_10(ctr, key):
    """Philox-4x32-10 block: 4 counter words, 2 key words -> 4 output words (ints)."""
    c = (C.c_uint32 * 4)(*[int(v) for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) for v in key])
    o = (C.c_uint32 * 4)()
    _load().ora_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def ray_uniforms(ray_id, seed):
    u = (C.c_double * 2)()
    _load().ora_ray_uniforms(int(ray_id), int(seed), u)
    return float(u[0]), float(u[1])


def ray_positions(sigma, stellar_fraction, gamma, n_pix, n_rays, L, ray_i, ray_j, ray_seed=None, ray_mode=None):
    """Image-plane positions x (n, 2) of the listed rays (regular grid, or random with ray_seed: ray_mode "cell" /
    "uniform")."""
    p = _problem(sigma, stellar_fraction, gamma, n_pix, n_rays, L, ray_seed, ray_mode)
    ri = np.ascontiguousarray(ray_i, dtype=np.int64)
    rj = np.ascontiguousarray(ray_j, dtype=np.int64)
    out = np.empty((ri.size, 2), dtype=np.float64)
    ip = C.POINTER(C.c_int64)
    _check(_load().ora_ray_positions(C.byref(p), ri.size, ri.ctypes.data_as(ip), rj.ctypes.data_as(ip), _dptr(out)),
           "ray_positions")
    return out
