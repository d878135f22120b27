"""B200-native direct inverse ray-shooting (arxiv/paper_1005_5198, GPU-D path).

The product is the C-ABI library built from csrc/ (include/microlens.h); this package
is its thin ctypes binding.  PyTorch is not imported here: callers use it only for
device memory and streams (ml_use_device_map / ml_attach_stream).
"""
from .binding import (  # noqa: F401
    EXPORTS,
    ML_ERR_CUDA,
    ML_ERR_INVALID_ARG,
    ML_ERR_LIMIT,
    ML_ERR_OOM,
    ML_ERR_STATE,
    ML_MEM_DEVICE,
    ML_MEM_HOST,
    ML_OK,
    ML_PREC_FP32_COMPENSATED,
    ML_PREC_FP32_TILED,
    ML_PREC_FP64,
    ML_RAYS_RANDOM,
    ML_RAYS_REGULAR,
    ML_RAYS_UNIFORM,
    ML_STATIC_MAX_COUNT,
    MicrolensError,
    library_path,
    load,
    ml_attach_stream,
    ml_capture_region,
    ml_create,
    ml_delta_m_histogram,
    ml_delta_m_histogram_static,
    ml_destroy,
    ml_get_info,
    ml_get_map,
    ml_get_map_device,
    ml_get_stats,
    ml_map_compare,
    ml_probe,
    ml_set_lens_masses,
    ml_set_lenses,
    ml_set_precision,
    ml_set_ray_mode,
    ml_shoot,
    ml_shoot_region,
    ml_use_device_map,
    ml_version,
    strerror,
)
from .map import MagnificationMap  # noqa: F401
