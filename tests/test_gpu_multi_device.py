"""-m gpu test: one process, contexts on two devices (the C ABI and MagnificationMap(device=...) allow it).

The random- and uniform-ray kernels need more than 48 KB of dynamic shared memory; that opt-in is a per-device
attribute of each kernel, so a process that has shot random rays on one GPU must still be able to on another.  On a
box with one GPU both contexts sit on device 0 (the test then only checks that two live contexts do not disturb each
other); with more GPUs the second context is on the last one.  PAPER.md:259, :271 (several GPUs per host)."""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from workloads import CONFIGS, lens_disk

from parity_common import problem_args

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("ray_mode", [ml.ML_RAYS_RANDOM, ml.ML_RAYS_UNIFORM], ids=["random", "uniform"])
def test_two_contexts_in_one_process_first_and_last_device(ray_mode):
    import torch
    last = torch.cuda.device_count() - 1
    p = CONFIGS[0]
    maps = []
    with ml.MagnificationMap(*problem_args(p), device=0) as m0, ml.MagnificationMap(*problem_args(p), device=last) as m1:
        assert m0.info["device"] == 0 and m1.info["device"] == last
        xy = lens_disk(m0.info["n_star_expected"], m0.info["r_star"], p.seed)
        for m in (m0, m1, m0):   # device 0 first (opts in there), then the other device, then device 0 again
            m.set_lenses(xy)
            m.set_ray_mode(ray_mode, 77)
            m.shoot()
            st = m.stats
            assert st["rays_shot"] == m.info["n1"] * m.info["n2"] and st["rays_dropped"] == 0
            maps.append(m.counts())
    # same seed, same arithmetic: the device a context lives on does not change a single count
    assert np.array_equal(maps[0], maps[1]) and np.array_equal(maps[0], maps[2])
    assert int(maps[0].sum()) > 0
