"""Seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and bench.py.

This package holds NO microlensing arithmetic: no geometry derivation, no
deflection, no binning.  It only (1) restates the five problem statements of
BASELINE.json:configs as plain numbers and (2) draws seeded random numbers.
Each side (oracle/ and the CUDA library) derives its own geometry and is handed
the same arrays.
"""
from .lens_fields import (  # noqa: F401
    CONFIGS,
    Problem,
    lens_disk,
    lens_masses,
    parity_tiles,
    probe_rays,
)
