"""CPU tests of the N > 1 path: the host logic that cuts the ray grid
into per-rank row bands (`sharding.row_band`) and sums the private count maps
(`sharding.allreduce_map`), run with world_size 2 over the `gloo` backend.  Each rank bins its
band with the fp64 oracle standing in for the GPU (the device path of the same logic is
`bench.py --gpus N`); the all-reduced map must equal the single-process map bit for bit,
because rays are independent and counts are integers.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle
from paper_1005_5198_b200.sharding import allreduce_map, row_band
from workloads import lens_disk

ARGS = (0.4, 1.0, 0.1, 32, 16.0, 4.0)  # sigma, stellar fraction, gamma, n_pix, n_rays, L
TILE_H = 16                             # the FP32 kernel's tile height (ml_info.tile_h)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir, ray_mode=None):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = oracle.geometry(*ARGS)
        xy = lens_disk(g.n_star, g.r_star, 7)
        j0, j1 = row_band(g.n2, rank, world, TILE_H)
        local = np.zeros((ARGS[3], ARGS[3]), dtype=np.uint32)
        _, st = oracle.shoot_region(*ARGS, xy, region=(0, g.n1, j0, j1), map_out=local,
                                    ray_seed=None if ray_mode is None else 11, ray_mode=ray_mode)
        counts = torch.from_numpy(local.view(np.int32).copy())
        allreduce_map(counts)
        shot = torch.tensor([st["rays_shot"], st["rays_in_map"]], dtype=torch.int64)
        dist.all_reduce(shot)
        np.save(os.path.join(out_dir, "map_%d.npy" % rank), counts.numpy().view(np.uint32))
        np.save(os.path.join(out_dir, "shot_%d.npy" % rank), shot.numpy())
        np.save(os.path.join(out_dir, "band_%d.npy" % rank), np.array([j0, j1]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("ray_mode", [None, "uniform"], ids=["regular", "uniform-rays"])
def test_two_ranks_row_bands_plus_allreduce_equal_the_single_map(tmp_path, ray_mode):
    """With uniform rays (reading R20) a row band is a band of ray IDS, not of the image plane: every rank's rays fall
    all over the rectangle, and the bands still partition the rays."""
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), ray_mode), nprocs=world, join=True)
    g = oracle.geometry(*ARGS)
    xy = lens_disk(g.n_star, g.r_star, 7)
    full, st = oracle.shoot(*ARGS, xy, ray_seed=None if ray_mode is None else 11, ray_mode=ray_mode)
    bands = [tuple(np.load(tmp_path / ("band_%d.npy" % r))) for r in range(world)]
    assert bands[0][0] == 0 and bands[0][1] == bands[1][0] and bands[1][1] == g.n2
    assert bands[0][1] % TILE_H == 0
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / ("map_%d.npy" % r)), full)
        shot = np.load(tmp_path / ("shot_%d.npy" % r))
        assert shot[0] == st["rays_shot"] == g.n1 * g.n2 and shot[1] == st["rays_in_map"]


@pytest.mark.parametrize("n2,world,align", [(2560, 2, 16), (91590, 8, 16), (24576, 4, 32), (17, 4, 16), (5, 8, 1), (0, 3, 16)])
def test_row_bands_are_disjoint_aligned_and_cover(n2, world, align):
    prev = 0
    heights = []
    for r in range(world):
        j0, j1 = row_band(n2, r, world, align)
        assert j0 == prev and j0 <= j1 <= n2
        assert j0 % align == 0 or j0 == n2
        heights.append(j1 - j0)
        prev = j1
    assert prev == n2
    full = [h for h in heights if h and h % align == 0]
    if full:
        assert max(full) - min(full) <= align


def test_row_band_rejects_bad_arguments():
    for bad in [(10, 2, 2, 1), (10, -1, 2, 1), (10, 0, 0, 1), (-1, 0, 1, 1), (10, 0, 1, 0)]:
        with pytest.raises(ValueError):
            row_band(*bad)


def test_allreduce_map_is_identity_without_a_process_group():
    c = torch.arange(16, dtype=torch.int32).reshape(4, 4)
    assert allreduce_map(c.clone()).equal(c)
