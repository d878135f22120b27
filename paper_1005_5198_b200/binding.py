"""ctypes binding of libmicrolens_b200.so -- argument marshalling only.

Function names and arguments are those of include/microlens.h; every step of the
hot path runs in the CUDA kernels behind them.  There is no CPU fallback: if the
library is missing and cannot be built, or no CUDA device is present, the calls
raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

ML_OK = 0
ML_ERR_INVALID_ARG = -1
ML_ERR_CUDA = -2
ML_ERR_OOM = -3
ML_ERR_STATE = -4
ML_ERR_LIMIT = -5
ML_STATIC_MAX_COUNT = 1 << 18

ML_PREC_FP32_TILED = 0
ML_PREC_FP32_COMPENSATED = 1
ML_PREC_FP64 = 2

EXPORTS = (
    "ml_create", "ml_destroy", "ml_get_info", "ml_set_lenses", "ml_set_precision", "ml_shoot",
    "ml_shoot_region", "ml_get_map", "ml_get_map_device", "ml_use_device_map", "ml_attach_stream",
    "ml_get_stats", "ml_capture_region", "ml_probe", "ml_strerror", "ml_version",
    "ml_map_compare", "ml_delta_m_histogram", "ml_set_lens_masses", "ml_set_ray_mode",
    "ml_delta_m_histogram_static",
)

ML_RAYS_REGULAR = 0
ML_RAYS_RANDOM = 1
ML_RAYS_UNIFORM = 2

ML_MEM_HOST = 0
ML_MEM_DEVICE = 1


class MlInfo(C.Structure):
    _fields_ = [
        ("kappa_star", C.c_double), ("kappa_c", C.c_double), ("a1", C.c_double), ("a2", C.c_double),
        ("ray_spacing", C.c_double), ("r_star", C.c_double), ("pixel_side", C.c_double),
        ("mu_theory", C.c_double),
        ("n1", C.c_int64), ("n2", C.c_int64), ("n_star_expected", C.c_int64), ("n_lenses", C.c_int64),
        ("n_pix", C.c_int32), ("tile_w", C.c_int32), ("tile_h", C.c_int32), ("precision", C.c_int32),
        ("device", C.c_int32), ("sm_count", C.c_int32), ("sm_clock_khz", C.c_int32),
        ("ray_mode", C.c_int32), ("ray_seed", C.c_uint64),
    ]


class MlStats(C.Structure):
    _fields_ = [
        ("rays_shot", C.c_uint64), ("rays_in_map", C.c_uint64), ("rays_dropped", C.c_uint64),
        ("interactions", C.c_uint64), ("kernel_launches", C.c_uint64),
        ("kernel_ms", C.c_double), ("total_ms", C.c_double), ("capture_ctas", C.c_uint64),
    ]


class MlMapCompareResult(C.Structure):
    _fields_ = [
        ("n_pixels", C.c_uint64), ("n_valid", C.c_uint64), ("n_empty_a", C.c_uint64), ("n_empty_b", C.c_uint64),
        ("sum_a", C.c_uint64), ("sum_b", C.c_uint64), ("max_a", C.c_uint32), ("max_b", C.c_uint32),
        ("mean_mu_a", C.c_double), ("mean_mu_b", C.c_double), ("rms_delta_m", C.c_double),
        ("ks_d", C.c_double), ("ks_prob", C.c_double), ("kernel_ms", C.c_double), ("pass_kernel_ms", C.c_double),
    ]


class MicrolensError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        super().__init__("%s: %s (%d)" % (what, strerror(code), code))


_lib = None


def library_path() -> str:
    """The in-tree library, or the build MICROLENS_B200_LIBRARY points at (a test build of the same sources)."""
    return os.environ.get("MICROLENS_B200_LIBRARY") or _build.LIB_PATH


def load():
    """dlopen the in-tree library (building it first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if path != _build.LIB_PATH:
        if not os.path.exists(path):
            raise RuntimeError("MICROLENS_B200_LIBRARY=%s does not exist (there is no CPU fallback)" % path)
    elif _build.is_stale():
        try:
            _build.build_library()
        except Exception as e:  # no nvcc on this box: use the shipped .so if there is one
            if not os.path.exists(path):
                raise RuntimeError("libmicrolens_b200.so is missing and cannot be built (%s); "
                                   "there is no CPU fallback" % e)
    lib = C.CDLL(path)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    lib.ml_create.argtypes = [dbl, dbl, dbl, i32, dbl, dbl, i32, C.POINTER(vp)]
    lib.ml_destroy.argtypes = [vp]
    lib.ml_destroy.restype = None
    lib.ml_get_info.argtypes = [vp, C.POINTER(MlInfo)]
    lib.ml_set_lenses.argtypes = [vp, C.POINTER(dbl), i64]
    lib.ml_set_lens_masses.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl), i64]
    lib.ml_set_precision.argtypes = [vp, C.c_int]
    lib.ml_set_ray_mode.argtypes = [vp, C.c_int, C.c_uint64]
    lib.ml_shoot.argtypes = [vp]
    lib.ml_shoot_region.argtypes = [vp, i64, i64, i64, i64, C.c_int]
    lib.ml_get_map.argtypes = [vp, C.POINTER(C.c_uint32), C.c_size_t]
    lib.ml_get_map_device.argtypes = [vp, C.POINTER(vp)]
    lib.ml_use_device_map.argtypes = [vp, vp]
    lib.ml_attach_stream.argtypes = [vp, vp]
    lib.ml_get_stats.argtypes = [vp, C.POINTER(MlStats)]
    lib.ml_capture_region.argtypes = [vp, i64, i64, i64, i64, C.POINTER(dbl)]
    lib.ml_probe.argtypes = [vp, i64, C.POINTER(i64), C.POINTER(i64), C.POINTER(dbl)]
    u32p = C.POINTER(C.c_uint32)
    lib.ml_map_compare.argtypes = [vp, dbl, vp, dbl, i64, C.c_int, i32, vp, C.POINTER(MlMapCompareResult)]
    lib.ml_delta_m_histogram.argtypes = [vp, dbl, i64, dbl, dbl, i32, C.c_int, i32, vp, C.POINTER(C.c_uint64)]
    lib.ml_delta_m_histogram_static.argtypes = [vp, dbl, i64, dbl, dbl, i32, i32, vp, vp]
    del u32p
    lib.ml_strerror.argtypes = [C.c_int]
    lib.ml_strerror.restype = C.c_char_p
    lib.ml_version.argtypes = []
    lib.ml_version.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("ml_destroy", "ml_strerror", "ml_version"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load().ml_strerror(int(code)).decode()


def ml_version() -> str:
    return load().ml_version().decode()


def _check(rc: int, what: str):
    if rc != ML_OK:
        raise MicrolensError(rc, what)


def _struct_dict(s):
    return {f: getattr(s, f) for f, _ in s._fields_}


# ---- the C calls, one Python function each (same names) -------------------------------
def ml_create(sigma, stellar_fraction, gamma, n_pix, n_rays, L, device=0):
    h = C.c_void_p()
    _check(load().ml_create(float(sigma), float(stellar_fraction), float(gamma), int(n_pix),
                            float(n_rays), float(L), int(device), C.byref(h)), "ml_create")
    return h


def ml_destroy(ctx):
    load().ml_destroy(ctx)


def ml_get_info(ctx) -> dict:
    s = MlInfo()
    _check(load().ml_get_info(ctx, C.byref(s)), "ml_get_info")
    return _struct_dict(s)


def ml_set_lenses(ctx, xy):
    a = np.ascontiguousarray(xy, dtype=np.float64).reshape(-1, 2)
    _check(load().ml_set_lenses(ctx, a.ctypes.data_as(C.POINTER(C.c_double)), a.shape[0]), "ml_set_lenses")


def ml_set_lens_masses(ctx, xy, mass=None):
    """Lens positions plus the masses m_i of eq. 4 (None = unit masses)."""
    a = np.ascontiguousarray(xy, dtype=np.float64).reshape(-1, 2)
    mp = None
    if mass is not None:
        m = np.ascontiguousarray(mass, dtype=np.float64).ravel()
        if m.size != a.shape[0]:
            raise ValueError("ml_set_lens_masses: one mass per lens")
        mp = m.ctypes.data_as(C.POINTER(C.c_double))
    _check(load().ml_set_lens_masses(ctx, a.ctypes.data_as(C.POINTER(C.c_double)), mp, a.shape[0]), "ml_set_lens_masses")


def ml_set_precision(ctx, mode):
    _check(load().ml_set_precision(ctx, int(mode)), "ml_set_precision")


def ml_set_ray_mode(ctx, mode, seed=0):
    _check(load().ml_set_ray_mode(ctx, int(mode), int(seed)), "ml_set_ray_mode")


def ml_shoot(ctx):
    _check(load().ml_shoot(ctx), "ml_shoot")


def ml_shoot_region(ctx, i0, i1, j0, j1, accumulate=False):
    _check(load().ml_shoot_region(ctx, int(i0), int(i1), int(j0), int(j1), 1 if accumulate else 0),
           "ml_shoot_region")


def ml_get_map(ctx, out=None) -> np.ndarray:
    """Counts as a (n_pix, n_pix) uint32 array, [j', i'] (host)."""
    n = ml_get_info(ctx)["n_pix"]
    if out is None:
        out = np.empty((n, n), dtype=np.uint32)
    assert out.dtype == np.uint32 and out.flags.c_contiguous
    _check(load().ml_get_map(ctx, out.ctypes.data_as(C.POINTER(C.c_uint32)), out.size), "ml_get_map")
    return out


def ml_get_map_device(ctx) -> int:
    p = C.c_void_p()
    _check(load().ml_get_map_device(ctx, C.byref(p)), "ml_get_map_device")
    return int(p.value or 0)


def ml_use_device_map(ctx, dptr):
    _check(load().ml_use_device_map(ctx, C.c_void_p(int(dptr) if dptr else None)), "ml_use_device_map")


def ml_attach_stream(ctx, cuda_stream):
    _check(load().ml_attach_stream(ctx, C.c_void_p(int(cuda_stream) if cuda_stream else None)),
           "ml_attach_stream")


def ml_get_stats(ctx) -> dict:
    s = MlStats()
    _check(load().ml_get_stats(ctx, C.byref(s)), "ml_get_stats")
    return _struct_dict(s)


def ml_capture_region(ctx, i0, i1, j0, j1) -> np.ndarray:
    """y of every ray of the region, shape (j1-j0, i1-i0, 2), computed by the shoot kernel."""
    out = np.empty((int(j1) - int(j0), int(i1) - int(i0), 2), dtype=np.float64)
    _check(load().ml_capture_region(ctx, int(i0), int(i1), int(j0), int(j1),
                                    out.ctypes.data_as(C.POINTER(C.c_double))), "ml_capture_region")
    return out


def ml_probe(ctx, ray_i, ray_j) -> np.ndarray:
    ri = np.ascontiguousarray(ray_i, dtype=np.int64)
    rj = np.ascontiguousarray(ray_j, dtype=np.int64)
    assert ri.shape == rj.shape
    out = np.empty((ri.size, 2), dtype=np.float64)
    ip = C.POINTER(C.c_int64)
    _check(load().ml_probe(ctx, ri.size, ri.ctypes.data_as(ip), rj.ctypes.data_as(ip),
                           out.ctypes.data_as(C.POINTER(C.c_double))), "ml_probe")
    return out


def _map_arg(m, n=None):
    """(pointer, n, where, keepalive): a host uint32 array, or an int DEVICE pointer with n given."""
    if isinstance(m, (int, np.integer)):
        if n is None:
            raise ValueError("a device pointer needs n")
        return C.c_void_p(int(m)), int(n), ML_MEM_DEVICE, None
    a = np.ascontiguousarray(m, dtype=np.uint32)
    return C.c_void_p(a.ctypes.data), a.size, ML_MEM_HOST, a


def ml_map_compare(a, n_rays_a, b, n_rays_b, n=None, device=0, cuda_stream=None) -> dict:
    """RMS difference in magnitudes and two-sample K-S test between two count maps.
    a, b: host uint32 arrays, or int device pointers (then pass n)."""
    pa, na_, wa, ka = _map_arg(a, n)
    pb, nb_, wb, kb = _map_arg(b, n)
    if wa != wb or na_ != nb_:
        raise ValueError("ml_map_compare: both maps must live in the same memory space and have the same size")
    r = MlMapCompareResult()
    _check(load().ml_map_compare(pa, float(n_rays_a), pb, float(n_rays_b), na_, wa, int(device),
                                 C.c_void_p(int(cuda_stream) if cuda_stream else None), C.byref(r)), "ml_map_compare")
    return _struct_dict(r)


def ml_delta_m_histogram(counts, n_rays, lo, hi, n_bins, n=None, device=0, cuda_stream=None) -> np.ndarray:
    """Histogram (uint64[n_bins]) of Delta m = -2.5 log10(count / n_rays) over [lo, hi) (eq. 10)."""
    pc, n_, w, keep = _map_arg(counts, n)
    out = np.zeros(int(n_bins), dtype=np.uint64)
    _check(load().ml_delta_m_histogram(pc, float(n_rays), n_, float(lo), float(hi), int(n_bins), w, int(device),
                                       C.c_void_p(int(cuda_stream) if cuda_stream else None),
                                       out.ctypes.data_as(C.POINTER(C.c_uint64))), "ml_delta_m_histogram")
    return out


def ml_delta_m_histogram_static(counts_ptr, n_rays, n, lo, hi, n_bins, hist_out_ptr, device=0, cuda_stream=None) -> None:
    """ml_delta_m_histogram without a single device allocation inside the library, for programs whose own pool
    (torch's caching allocator, a server's arena) already owns the GPU memory or that cannot take the device-wide
    stall of cudaMalloc / cudaFree.  counts_ptr: int DEVICE pointer to n uint32 counts; hist_out_ptr: int DEVICE
    pointer to n_bins uint64 the caller allocated (e.g. tensor.data_ptr() of a torch int64 tensor) -- overwritten.
    Scratch is a fixed 1 MiB array inside the library: every count must be < ML_STATIC_MAX_COUNT (2^18), else
    MicrolensError with code ML_ERR_LIMIT.  The first call on a device does a one-time symbol look-up; make it
    before any stream capture.  See include/microlens.h."""
    _check(load().ml_delta_m_histogram_static(C.c_void_p(int(counts_ptr)), float(n_rays), int(n), float(lo), float(hi),
                                              int(n_bins), int(device),
                                              C.c_void_p(int(cuda_stream) if cuda_stream else None),
                                              C.c_void_p(int(hist_out_ptr))), "ml_delta_m_histogram_static")
