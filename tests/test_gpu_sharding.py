"""-m gpu test of the N > 1 DEVICE path (ray batches over 2-4 GPUs).
Two processes share cuda:0 (the test boxes have one GPU); each one calls ml_shoot_region on its own
`sharding.row_band` through the C ABI, reads its private device map back and sums the maps with
`sharding.allreduce_map` over gloo (host tensors -- the ranks never wait on one another's kernels).
The all-reduced map must equal the single-process ml_shoot map bit for bit: rays are independent
(PAPER.md:78), tiles are aligned to the global grid and counts are integers.  bench.py --gpus N runs
the same two calls with NCCL in place of gloo.
"""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import paper_1005_5198_b200 as ml
from paper_1005_5198_b200.sharding import allreduce_map, row_band
from workloads import CONFIGS, lens_disk

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _args(p):
    return (p.sigma, p.stellar_fraction, p.gamma, p.n_pix, p.n_rays, p.L)


def _worker(rank, world, port, out_dir, precision, ray_mode):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = CONFIGS[0]
        with ml.MagnificationMap(*_args(p), device=0, precision=precision) as m:
            info = m.info
            m.set_lenses(lens_disk(info["n_star_expected"], info["r_star"], p.seed))
            if ray_mode:
                m.set_ray_mode(ray_mode, 99)
            info = m.info
            j0, j1 = row_band(info["n2"], rank, world, info["tile_h"])
            m.shoot_region(0, info["n1"], j0, j1)           # the device path of this rank's band
            st = m.stats
            counts = torch.from_numpy(m.counts().view(np.int32).copy())
        assert st["kernel_launches"] >= 1 and st["rays_shot"] == info["n1"] * (j1 - j0)
        allreduce_map(counts)
        tot = torch.tensor([st["rays_shot"], st["rays_in_map"]], dtype=torch.int64)
        dist.all_reduce(tot)
        np.save(os.path.join(out_dir, "map_%d.npy" % rank), counts.numpy().view(np.uint32))
        np.save(os.path.join(out_dir, "tot_%d.npy" % rank), tot.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("precision,ray_mode",
                         [(ml.ML_PREC_FP32_TILED, 0), (ml.ML_PREC_FP64, 0), (ml.ML_PREC_FP32_TILED, ml.ML_RAYS_RANDOM),
                          (ml.ML_PREC_FP32_TILED, ml.ML_RAYS_UNIFORM)],
                         ids=["fp32_tiled", "fp64", "fp32_tiled-random_rays", "fp32_tiled-uniform_rays"])
def test_row_bands_on_the_device_plus_allreduce_equal_the_single_process_map(tmp_path, world, precision, ray_mode):
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), precision, ray_mode), nprocs=world, join=True)
    p = CONFIGS[0]
    with ml.MagnificationMap(*_args(p), device=0, precision=precision) as m:
        info = m.info
        m.set_lenses(lens_disk(info["n_star_expected"], info["r_star"], p.seed))
        if ray_mode:
            m.set_ray_mode(ray_mode, 99)
        m.shoot()
        full, st = m.counts(), m.stats
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / ("map_%d.npy" % r)), full)
        tot = np.load(tmp_path / ("tot_%d.npy" % r))
        assert tot[0] == st["rays_shot"] and tot[1] == st["rays_in_map"]


def test_bench_refuses_more_gpus_than_the_box_has():
    """`python bench.py --gpus N` is how the driver starts the scaling run: with fewer than N devices it must exit
    non-zero and say why -- never run on fewer GPUs and print n_gpus = N."""
    n = torch.cuda.device_count() + 1
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(n), "--steps", "1", "--warmup", "1"],
                         capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode != 0
    assert "refusing to run fewer GPUs than reported" in out.stderr
    assert not [ln for ln in out.stdout.splitlines() if ln.strip().startswith("{")]
