"""The C oracle under AddressSanitizer + UndefinedBehaviorSanitizer (sanitizers on the oracle and
the host side; compute-sanitizer is not available on this pool, gcc's are).

oracle/microlens_oracle.c is rebuilt with -fsanitize=address,undefined into a scratch .so and a subprocess re-runs the
pins that exercise its array handling -- the brute-force maps (regular, masses, random and uniform rays), the region /
capture / probe consistency pins, ray-on-a-lens -- through that build (ML_ORACLE_LIBRARY), with libasan preloaded as gcc
requires for a sanitized library under an unsanitized python.  Any out-of-bounds access, signed overflow, bad shift or
misaligned load aborts the subprocess (-fno-sanitize-recover)."""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PINS = ["tests/test_oracle_pins.py", "tests/test_oracle_mass_pins.py", "tests/test_oracle_random_rays.py",
        "tests/test_oracle_uniform_rays.py"]
SELECT = "brute_force or regions or ray_on_a_lens or worked_by_hand or known_answer or own_grid_cell or cover_the_shooting"


def test_oracle_pins_pass_under_asan_and_ubsan(tmp_path):
    if not shutil.which("gcc"):
        pytest.skip("gcc not on PATH")
    libasan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(libasan) or not os.path.exists(libasan):
        pytest.skip("gcc has no libasan here")
    so = str(tmp_path / "libmloracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer",
                           "-o", so, os.path.join(ROOT, "oracle", "microlens_oracle.c"), "-lm"])
    env = dict(os.environ)
    env.update(ML_ORACLE_LIBRARY=so, LD_PRELOAD=libasan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",   # python itself never frees everything: leaks are not the subject
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", OMP_NUM_THREADS="4")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-k", SELECT] + PINS,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "AddressSanitizer" not in tail and "runtime error" not in tail, tail
    # the sanitized build really was the one loaded
    probe = subprocess.run([sys.executable, "-c",
                            "from oracle import oracle; oracle.geometry(0.4, 1.0, 0.0, 64, 10.0, 10.0); "
                            "print([l.split()[-1] for l in open('/proc/self/maps') if 'mloracle' in l][0])"],
                           cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert probe.returncode == 0 and probe.stdout.strip() == so, probe.stdout + probe.stderr
