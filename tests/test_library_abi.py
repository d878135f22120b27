"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol that
include/microlens.h declares, validates arguments, and fails loudly without a GPU.
No compute call is made here (those are the -m gpu tests)."""
import ctypes as C
import os
import re

import pytest

import paper_1005_5198_b200 as ml
from paper_1005_5198_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "microlens.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ml_[a-z_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    lib = ml.load()
    declared = _declared_symbols()
    assert len(declared) >= 16 and {"ml_create", "ml_set_lenses", "ml_shoot", "ml_get_map", "ml_destroy"} <= set(declared)
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared
    assert "sm_100a" in ml.ml_version()
    assert os.path.dirname(ml.library_path()).endswith("paper_1005_5198_b200")  # in-tree, not site-packages


def test_library_is_built_for_sm_100a_only():
    import shutil
    import subprocess
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    out = subprocess.run(["cuobjdump", "-lelf", ml.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, out


def test_error_strings_and_argument_validation():
    assert ml.strerror(ml.ML_OK) == "ok"
    for code in (ml.ML_ERR_INVALID_ARG, ml.ML_ERR_CUDA, ml.ML_ERR_OOM, ml.ML_ERR_STATE, -99):
        assert ml.strerror(code)
    lib = ml.load()
    h = C.c_void_p()
    bad = [
        (0.5, 1.0, 0.5, 64, 10.0, 10.0),           # 1 - sigma - gamma = 0: critical line
        (1.5, 1.0, -0.5, 64, 10.0, 10.0),          # 1 - sigma + gamma = 0
        (-0.1, 1.0, 0.0, 64, 10.0, 10.0),
        (0.4, 1.5, 0.0, 64, 10.0, 10.0),
        (0.4, 1.0, 0.0, 0, 10.0, 10.0),
        (0.4, 1.0, 0.0, 64, 0.0, 10.0),
        (0.4, 1.0, 0.0, 64, 10.0, -1.0),
        (0.4, 1.0, float("nan"), 64, 10.0, 10.0),
        (0.4, 1.0, 0.0, 64, float("inf"), 10.0),
        (0.4, 1.0, 0.0, 40000, 10.0, 10.0),
        (0.4, 1.0, 0.0, 64, 1e30, 10.0),           # n1*n2 overflows
    ]
    for args in bad:
        rc = lib.ml_create(*args, 0, C.byref(h))
        assert rc == ml.ML_ERR_INVALID_ARG and not h.value, args
    assert lib.ml_create(0.4, 1.0, 0.0, 64, 10.0, 10.0, 0, None) == ml.ML_ERR_INVALID_ARG
    # NULL contexts are rejected, never dereferenced
    assert lib.ml_shoot(None) == ml.ML_ERR_INVALID_ARG
    assert lib.ml_get_info(None, None) == ml.ML_ERR_INVALID_ARG
    assert lib.ml_set_lenses(None, None, 0) == ml.ML_ERR_INVALID_ARG
    assert lib.ml_get_map(None, None, 0) == ml.ML_ERR_INVALID_ARG
    lib.ml_destroy(None)


def test_no_cpu_fallback_without_a_device():
    """On a box without a GPU a valid ml_create must fail with ML_ERR_CUDA, not compute."""
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        pytest.skip("this box has a GPU")
    with pytest.raises(ml.MicrolensError) as e:
        ml.ml_create(0.4, 1.0, 0.0, 64, 10.0, 10.0)
    assert e.value.code == ml.ML_ERR_CUDA


def test_product_never_imports_the_oracle():
    """The oracle is test infrastructure: nothing under the package may mention it."""
    pkg = os.path.join(ROOT, "paper_1005_5198_b200")
    for dirpath, _dirs, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), (dirpath, f)


def test_test_builds_cannot_overwrite_the_shipped_library(tmp_path):
    """build_library(defines=...) makes a crippled TEST build (tiny grid limits, tiny list memory).  Written over the
    shipped .so it would be newer than its sources and every later load would silently use it: refused."""
    from paper_1005_5198_b200 import build as mlbuild
    before = os.path.getmtime(mlbuild.LIB_PATH)
    with pytest.raises(ValueError):
        mlbuild.build_library(defines=["ML_MAX_GRID_X=7"])
    with pytest.raises(ValueError):
        mlbuild.build_library(defines=["ML_MAX_GRID_X=7"], out=mlbuild.LIB_PATH)
    assert os.path.getmtime(mlbuild.LIB_PATH) == before
