#!/usr/bin/env python
"""bench.py -- lens-ray interactions/s of the fused shoot kernel on BASELINE.json:configs[1].

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl reference]

A step is one pass of the whole hot path (lens staging, fused ray
generation, deflection sum, macro terms, binning; map zeroing included) over the full ray
grid of the workload: one ml_shoot (N = 1) or one row band per rank plus the map all-reduce
(N > 1, strong scaling).  Prints ONE JSON line (rank 0).  DESIGN.md "Measurement" explains
every field.

N > 1: one process per GPU over NCCL.  Started under torchrun the ranks come from the
environment; started as plain `python bench.py --gpus N` the script launches the N ranks
itself (torch.distributed.run on 127.0.0.1).  Fewer than N visible GPUs is an error -- the
script never runs fewer GPUs than it prints.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from workloads import CONFIGS, lens_disk, lens_masses, parity_tiles  # noqa: E402

METRIC = "lens-ray interactions/sec"
UNIT = "interactions/s"
N_FLOP = 10.0          # flop per lens-ray interaction
FP32_LANES_PER_SM = 128
# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the dominant kernel, from the
# committed `ncu --set full` capture of this very command; None where no capture exists.
NCU_DRAM_BYTES_PER_LAUNCH = {
    ("C2", "fp32_tiled"): (4384512 + 0, "profiles/r02_ncu_full_c2.txt"),
    ("C2", "fp32_compensated"): (4423168 + 0, "profiles/r02_ncu_full_c2_compensated.txt"),
    ("C2", "fp64"): (4385792 + 0, "profiles/r02_ncu_full_c2_fp64.txt"),
    # widened rows (key: workload, precision, row): the shoot kernel of that row
    ("C2", "fp32_tiled", "random_rays"): (5490000, "profiles/r02_ncu_full_c2_random.txt"),
    ("C2", "fp32_tiled", "uniform_rays"): (68970000000 + 750000000, "profiles/r02_ncu_full_c2_uniform.txt (shoot_kernel_upipe; "
                                           "the scatter kernel moves another 283 GB, r02_ncu_full_c2_uniform_scatter.txt)"),
}
NCU_MAPSTATS_DRAM_BYTES = (134431232 + 3515904, "profiles/r02_ncu_full_mapstats.txt")


def problem_args(p):
    return (p.sigma, p.stellar_fraction, p.gamma, p.n_pix, p.n_rays, p.L)


def sig(x, digits=6):
    """A float rounded to `digits` significant digits: the per_config / extra_rows blocks must fit the ~5 KB tail of
    stdout that the driver's record keeps."""
    return float("%.*g" % (digits, x))


def brief_clocks(clocks):
    return {"sm_mhz": clocks.get("sm_mhz"), "reasons": clocks.get("reasons")} if clocks else None


def pick(name):
    for p in CONFIGS:
        if p.name == name:
            return p
    raise SystemExit("unknown workload %r" % name)


# ------------------------------------------------------------------ clocks (recipe: B200_PROFILING.md)
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"], stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        try:
            for line in open(self.path):
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm),
                       power_w_max=float(max(pw)), sm_mhz_min=float(min(sm)), reasons=sorted(reasons))
        return out


# ------------------------------------------------------------------ oracle legs
def oracle_rate(p, seconds, log=None):
    """Time the fp64 CPU oracle, as it stands, on a bounded sample of workload p: seeded
    512 x 512-ray sub-rectangles of its ray grid, as many as fit in about `seconds`."""
    from oracle import oracle
    g = oracle.geometry(*problem_args(p))
    xy = lens_disk(g.n_star, g.r_star, p.seed)   # the BASELINE config's own field (no --masses / --n-lenses here)
    side = 512
    tiles = parity_tiles(g.n1, g.n2, 64, side, p.seed)
    omap = np.zeros((p.n_pix, p.n_pix), dtype=np.uint32)
    t0 = time.perf_counter()
    oracle.shoot_region(*problem_args(p), xy, region=(0, 128, 0, 128), map_out=omap)  # calibrate
    per_inter = (time.perf_counter() - t0) / (128 * 128 * max(g.n_star, 1))
    n_tiles = int(max(1, min(len(tiles), seconds / (per_inter * side * side * max(g.n_star, 1)))))
    omap[:] = 0
    inter = 0
    t0 = time.perf_counter()
    for r in tiles[:n_tiles]:
        _, st = oracle.shoot_region(*problem_args(p), xy, region=r, map_out=omap)
        inter += st["interactions"]
    dt = time.perf_counter() - t0
    return {"value": inter / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": "%s: %d seeded sub-rectangles of %dx%d rays x %d lenses = %.3g interactions in %.1f s"
                      % (p.name, n_tiles, side, side, g.n_star, inter, dt),
            "seconds": dt, "interactions": inter}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / unit / config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    p = pick(args.workload)
    from oracle import oracle
    g = oracle.geometry(*problem_args(p))
    per_step = max(1.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    if args.ref_seconds_per_step is not None:
        per_step = args.ref_seconds_per_step
    for _ in range(args.warmup):
        oracle_rate(p, per_step)
    inter, secs, last = 0, 0.0, None
    for _ in range(args.steps):
        last = oracle_rate(p, per_step)
        inter += last["interactions"]
        secs += last["seconds"]
    value = inter / secs
    base = {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"] + " per step"}
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(p, {"n_lenses": g.n_star, "n1": g.n1, "n2": g.n2}, args),
            "precision": "fp64", "config_note": "config is the CUDA arm's, key for key (its l2 / parallelism entries describe that arm; "
                                                  "this arm runs the oracle on the host cores)",
            "cpu_baseline": base,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def config_dict(p, info, args):
    c = {"workload": "%s: sigma=%g gamma=%g stellar_fraction=%g L=%g n_pix=%d^2 n_rays=%g seed=%d (BASELINE.json configs[%d])"
                     % (p.name, p.sigma, p.gamma, p.stellar_fraction, p.L, p.n_pix, p.n_rays, p.seed, CONFIGS.index(p)),
         "l2": "flushed between steps (256 MiB write)",
         "parallelism": "ray row bands x%d + map all-reduce" % args.gpus if args.gpus > 1 else "single GPU"}
    if getattr(args, "masses", False):
        c["masses"] = "log-uniform 0.3-3 (workloads.lens_masses), eq. 4 with m_i"
    if getattr(args, "random_rays", False):
        c["ray_mode"] = "random position in every grid cell (GPU-D's ray generation, PAPER.md:131; reading R17), generic kernel"
    if getattr(args, "uniform_rays", False):
        c["ray_mode"] = ("every ray an independent uniform point of the shooting rectangle (the literal GPU-D ray generation, "
                         "PAPER.md:131, :167; reading R20): bucket sort on the device + shoot_kernel_upipe, both inside the step")
    if getattr(args, "n_lenses", 0) > 0:
        c["n_lenses_override"] = "lens count set to %d in the same disk (large-N* row, not a BASELINE config)" % args.n_lenses
    # the geometry keys are the same in both arms (ours: ml_get_info; --impl reference: the oracle's own geometry), so
    # that the two `config` objects are identical; what differs between the arms (precision, tile) is top-level
    if info is not None:
        c.update(n_lenses=int(info["n_lenses"]), n1=int(info["n1"]), n2=int(info["n2"]), rays=int(info["n1"]) * int(info["n2"]))
    return c


# ------------------------------------------------------------------ the CUDA arm
PRECISIONS = {"fp32_tiled": 0, "fp32_compensated": 1, "fp64": 2}
# per_config block of the default line: (workload, timed steps, full warm-up steps); configs without a full warm-up step
# are warmed by three shoots of 1/32 of their ray rows (the device is already warm from the C2 region before them)
PER_CONFIG_PLAN = (("C1", 50, 5), ("C5", 2, 0), ("C3", 1, 0), ("C4", 1, 0))


def fp32_peak_tflops(info):
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    max_mhz = float(peaks.get("sm_max_mhz") or (info["sm_clock_khz"] / 1e3))
    return int(info["sm_count"]) * FP32_LANES_PER_SM * 2 * max_mhz * 1e6 / 1e12, max_mhz


class ShootRig:
    """One workload set up the way a user of the library would: context, lenses, a torch-owned device map, a torch
    stream attached to the context, pinned host buffers for the end-to-end leg."""

    def __init__(self, ml, torch, p, args, local, rank=0, world=1, flush=None):
        from paper_1005_5198_b200.sharding import row_band
        self.torch, self.p, self.world = torch, p, world
        self.dev = torch.device("cuda", local)
        self.m = ml.MagnificationMap(*problem_args(p), device=local, precision=PRECISIONS[args.precision])
        info = self.m.info
        n_field = args.n_lenses if args.n_lenses > 0 else info["n_star_expected"]
        self.xy = lens_disk(n_field, info["r_star"], p.seed)
        self.mass = lens_masses(n_field, p.seed) if args.masses else None
        self.m.set_lenses(self.xy, self.mass)
        if args.random_rays:
            self.m.set_ray_mode(ml.ML_RAYS_RANDOM, 20100527)
        if args.uniform_rays:
            self.m.set_ray_mode(ml.ML_RAYS_UNIFORM, 20100527)
        self.info = info = self.m.info
        self.n1, self.n2, self.n_lens = int(info["n1"]), int(info["n2"]), int(info["n_lenses"])
        self.j0, self.j1 = row_band(self.n2, rank, world, int(info["tile_h"]))
        self.stream = torch.cuda.Stream(device=self.dev)
        self.counts = torch.zeros((p.n_pix, p.n_pix), dtype=torch.int32, device=self.dev)  # torch owns the map memory
        self.m.use_device_map(self.counts.data_ptr())
        self.m.attach_stream(self.stream.cuda_stream)
        self.flush = flush if flush is not None else torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)
        self.host_xy = torch.from_numpy(self.xy).pin_memory()
        self.host_map = torch.empty((p.n_pix, p.n_pix), dtype=torch.int32).pin_memory()
        self.host_map_np = self.host_map.numpy().view(np.uint32)

    def flush_l2(self):
        with self.torch.cuda.stream(self.stream):
            self.flush.fill_(1)                  # 256 MiB write: evicts the 126 MB L2

    def step(self, rows=None):
        """flush L2, zero the map, shoot this rank's band, (N > 1) all-reduce the maps; returns ml_stats."""
        from paper_1005_5198_b200.sharding import allreduce_map
        j0, j1 = rows if rows is not None else (self.j0, self.j1)
        self.flush_l2()
        self.m.shoot_region(0, self.n1, j0, j1)  # zero map + fused kernel (synchronises the stream)
        st = self.m.stats
        if self.world > 1:
            with self.torch.cuda.stream(self.stream):
                allreduce_map(self.counts)
        return st

    def e2e_step(self):
        """The same through the C ABI with HOST buffers: lenses host -> device, shoot, map device -> host."""
        from paper_1005_5198_b200.sharding import allreduce_map
        self.m.set_lenses(self.host_xy.numpy(), self.mass)   # H2D (ml_set_lenses / ml_set_lens_masses)
        self.m.shoot_region(0, self.n1, self.j0, self.j1)
        st = self.m.stats
        if self.world > 1:
            with self.torch.cuda.stream(self.stream):
                allreduce_map(self.counts)
        self.m.counts(out=self.host_map_np)                  # D2H (ml_get_map)
        return st

    def e2e_bytes(self):
        h2d = int(self.xy.nbytes) + (int(self.mass.nbytes) if self.mass is not None else 0)
        return h2d, int(self.host_map_np.nbytes + 24)

    def close(self):
        self.m.close()


def per_config_entry(ml, torch, name, steps, full_warmup, args, local, flush):
    """One entry of the default line's per_config block (single GPU; keys kept short, see `sig`: unit = the line's unit,
    e2e_value / e2e_ms = the end-to-end rate and wall time per step with h2d / d2h bytes copied per step; each config is
    shot 2 x steps times, once end to end and once device-timed).  Every timed step is an END-TO-END step (host
    lenses -> ml_set_lenses -> ml_shoot -> ml_get_map -> host map, L2 flushed before it, outside the clock): `e2e` is
    its wall clock, `kernel_ms` the library's CUDA events around the kernel launch of the same step, `value` the
    device-timed rate of the whole step without the copies (memset + kernel, events on the launching stream)."""
    p = pick(name)
    rig = ShootRig(ml, torch, p, args, local, flush=flush)
    dev, n_lens, rays = rig.dev, rig.n_lens, rig.n1 * rig.n2
    for _ in range(full_warmup):
        rig.step()
    if not full_warmup:
        band = max(int(rig.info["tile_h"]), rig.n2 // 32)
        for k in range(3):
            rig.step(rows=(k * band, (k + 1) * band))
    sampler = ClockSampler(local)
    short = rays * n_lens < 1e11          # ms-long steps: a polling nvidia-smi triples their host latency
    if short:
        sampler.start()
        t_end = time.perf_counter() + 1.2
        while time.perf_counter() < t_end:
            rig.step()
        clocks = sampler.stop()
        clocks["when"] = "1.2 s of the same steps immediately before the timed region"
    else:
        sampler.start()
    kernel_ms, dev_ms, wall = 0.0, 0.0, 0.0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(steps):
        rig.flush_l2()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        st = rig.e2e_step()
        wall += time.perf_counter() - t0
        assert int(st["rays_shot"]) == rays
        kernel_ms += st["kernel_ms"]
        rig.flush_l2()                    # the device-timed form of the same step: memset + kernel, no copies
        e0.record(rig.stream)
        rig.m.shoot_region(0, rig.n1, 0, rig.n2)
        e1.record(rig.stream)
        torch.cuda.synchronize(dev)
        dev_ms += e0.elapsed_time(e1)
        kernel_ms += rig.m.stats["kernel_ms"]
    if not short:
        clocks = sampler.stop()
    peak, _ = fp32_peak_tflops(rig.info)
    inter = float(rays) * n_lens
    h2d, d2h = rig.e2e_bytes()
    k_ms = kernel_ms / (2 * steps)
    out = {"workload": p.name, "n_lenses": n_lens, "rays": rays, "steps": steps,
           "kernel_ms": sig(k_ms), "ms_per_step": sig(dev_ms / steps), "value": sig(inter * steps / (dev_ms * 1e-3)),
           "frac": sig(N_FLOP * inter / (k_ms * 1e-3) / 1e12 / peak, 4),
           "step_frac": sig(N_FLOP * inter * steps / (dev_ms * 1e-3) / 1e12 / peak, 4),
           "e2e_value": sig(inter * steps / wall), "e2e_ms": sig(1e3 * wall / steps),
           "h2d": h2d, "d2h": d2h, "clocks": brief_clocks(clocks)}
    rig.close()
    return out


# extra_rows of the default line: the widened rows of DESIGN.md section 11 on C2, one device-timed full step each (after
# two warm-up shoots of 1/32 of the rows and one full step; the device is warm from the regions before), so that the
# driver's own run observes them too.  Their full bench lines are `bench.py --masses` etc.
EXTRA_ROWS = (("C2 masses", {"masses": True}), ("C2 random rays (R17)", {"random_rays": True}),
              ("C2 uniform rays (R20), sort included", {"uniform_rays": True}),
              ("C2 fp32_compensated", {"precision": "fp32_compensated"}), ("C2 fp64", {"precision": "fp64"}))


def extra_row(ml, torch, label, overrides, args, local, flush):
    a = argparse.Namespace(**vars(args))
    for k, v in overrides.items():
        setattr(a, k, v)
    p = pick("C2")
    rig = ShootRig(ml, torch, p, a, local, flush=flush)
    band = max(int(rig.info["tile_h"]), rig.n2 // 32)
    for k in range(2):
        rig.step(rows=(k * band, (k + 1) * band))
    rig.step()                                   # one full step: also sizes the uniform mode's bucket lists
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rig.flush_l2()
    e0.record(rig.stream)
    rig.m.shoot_region(0, rig.n1, 0, rig.n2)
    e1.record(rig.stream)
    torch.cuda.synchronize(rig.dev)
    st = rig.m.stats
    assert int(st["rays_shot"]) == rig.n1 * rig.n2
    ms = e0.elapsed_time(e1)
    peak, _ = fp32_peak_tflops(rig.info)
    inter = float(rig.n1) * rig.n2 * rig.n_lens
    out = {"row": label, "ms_per_step": sig(ms), "kernel_ms": sig(st["kernel_ms"]), "gpu_launches": int(st["kernel_launches"]),
           "value": sig(inter / (ms * 1e-3)), "frac": sig(N_FLOP * inter / (st["kernel_ms"] * 1e-3) / 1e12 / peak, 4)}
    rig.close()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1005_5198_b200 as ml

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; --impl reference times the oracle)")
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d: launch with --nproc-per-node equal to --gpus"
                         % (args.gpus, world))
    if local >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d needs cuda:%d but only %d device(s) are visible"
                         % (rank, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    p = pick(args.workload)
    rig = ShootRig(ml, torch, p, args, local, rank, world)
    info, n1, n2, n_lens, stream = rig.info, rig.n1, rig.n2, rig.n_lens, rig.stream
    if world > 1:   # one line per rank on stderr, so that a scaling record shows the N ranks, their devices and bands
        print("bench.py: rank %d/%d on cuda:%d (%s), communicator size %d, ray rows [%d, %d) of %d"
              % (rank, world, local, torch.cuda.get_device_name(local), dist.get_world_size(), rig.j0, rig.j1, n2),
              file=sys.stderr, flush=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        rig.step()
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms, launches, rays = 0.0, 0, 0
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        st = rig.step()
        kernel_ms += st["kernel_ms"]
        launches += int(st["kernel_launches"])
        rays += int(st["rays_shot"])
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    agg = torch.tensor([ms, kernel_ms], dtype=torch.float64, device=dev)
    tot = torch.tensor([rays, launches], dtype=torch.int64, device=dev)
    if world > 1:
        dist.all_reduce(agg, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    ms, kernel_ms_max = float(agg[0]), float(agg[1])
    rays_all, launches_all = int(tot[0]), int(tot[1])
    assert rays_all == n1 * n2 * args.steps, (rays_all, n1 * n2 * args.steps)
    value = rays_all * n_lens / (ms * 1e-3)

    # ---- end to end through the public C ABI with HOST buffers, copies inside the timed region
    e2e_steps = max(1, min(args.steps, 3))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        rig.e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    e2e_value = n1 * n2 * n_lens * e2e_steps / float(e2e_t[0])
    h2d, d2h = rig.e2e_bytes()
    flush = rig.flush
    rig.close()
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return 0

    peak_tflops, max_mhz = fp32_peak_tflops(info)
    sm_count = int(info["sm_count"])
    kernel_s_per_launch = kernel_ms_max * 1e-3 / max(1, launches_all // max(world, 1))
    inter_per_launch = (rays_all // world) * n_lens / max(1, launches_all // max(world, 1))
    achieved = N_FLOP * inter_per_launch / kernel_s_per_launch / 1e12
    # ncu DRAM bytes exist only for the exact kernel that was captured: the BASELINE workload, unit masses, regular grid
    plain = world == 1 and not (args.masses or args.random_rays or args.uniform_rays or args.n_lenses > 0)
    traffic, traffic_src = NCU_DRAM_BYTES_PER_LAUNCH.get((p.name, args.precision), (None, None)) if plain else (None, None)
    if world == 1 and not plain and not args.masses and args.n_lenses <= 0 and not (args.random_rays and args.uniform_rays):
        row = "random_rays" if args.random_rays else "uniform_rays"
        traffic, traffic_src = NCU_DRAM_BYTES_PER_LAUNCH.get((p.name, args.precision, row), (None, None))
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "traffic": traffic,
                "traffic_unit": "DRAM bytes per launch (ncu --set full; %s); algorithmic = n_pix^2*4 + 16 N* = %d"
                                % (traffic_src or "no capture of this kernel instantiation", p.n_pix * p.n_pix * 4 + 16 * n_lens),
                "note": "%g flop/interaction (PAPER.md:66); peak = %d SMs x 128 lanes x 2 x %.0f MHz (sm_max_mhz); "
                        "kernel time = CUDA events on the launching stream" % (N_FLOP, sm_count, max_mhz),
                "kernel_ms_per_launch": 1e3 * kernel_s_per_launch}
    if clocks and clocks.get("sm_mhz"):
        roofline["frac_at_sampled_clock"] = achieved / (peak_tflops * clocks["sm_mhz"] / max_mhz)
    per_config = None
    if plain and args.workload == "C2" and args.precision == "fp32_tiled" and not args.no_per_config:
        per_config = [{"workload": p.name, "n_lenses": n_lens, "rays": n1 * n2,        # the line's own timed region
                       "steps": args.steps, "kernel_ms": sig(1e3 * kernel_s_per_launch), "ms_per_step": sig(ms / args.steps),
                       "value": sig(value), "frac": sig(achieved / peak_tflops, 4),
                       "step_frac": sig(N_FLOP * value / 1e12 / peak_tflops, 4),
                       "e2e_value": sig(e2e_value), "e2e_ms": sig(1e3 * float(e2e_t[0]) / e2e_steps),
                       "h2d": h2d, "d2h": d2h, "clocks": brief_clocks(clocks)}]
        for name, steps, full_warmup in PER_CONFIG_PLAN:
            per_config.append(per_config_entry(ml, torch, name, steps, full_warmup, args, local, flush))
    extra = None
    if per_config is not None:
        extra = [extra_row(ml, torch, label, ov, args, local, flush) for label, ov in EXTRA_ROWS]
        del flush
        torch.cuda.empty_cache()
        ms_args = argparse.Namespace(**vars(args))
        ms_args.steps, ms_args.warmup, ms_args.no_cpu_baseline = 10, 3, True
        ml_line = mapstats_line(ms_args)
        extra.append({"row": "ml_map_compare, two 4096^2 maps", "ms_per_step": sig(ml_line["ms_per_step"]),
                      "value": sig(ml_line["value"]), "unit": ml_line["unit"], "frac": sig(ml_line["roofline"]["frac"], 4), "bound": "hbm",
                      "pass_kernel_ms": sig(ml_line["roofline"]["pass_kernel_ms"]), "call_ms_without_flush": sig(ml_line["call_ms_without_flush"])})
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = oracle_rate(p, args.cpu_seconds)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32" if args.precision != "fp64" else "f64",
            "data": "synthetic", "config": config_dict(p, info, args),
            "precision": args.precision, "tile": [int(info["tile_w"]), int(info["tile_h"])],
            "rays_per_s": rays_all / (ms * 1e-3), "map_wall_ms": ms / args.steps,
            "nominal_tflops": N_FLOP * value / 1e12, "frac_fp32_peak": N_FLOP * value / 1e12 / (peak_tflops * args.gpus),
            "roofline": roofline, "cpu_baseline": cpu, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "steps": e2e_steps},
            "gpu_launches": launches_all}
    if per_config is not None:
        line["per_config"] = per_config
        line["extra_rows"] = extra
    print(json.dumps(line))
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun around it: start the N ranks here (one process per GPU,
    NCCL over 127.0.0.1) and pass their exit code on.  Refuses to run with fewer than N devices."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        print("bench.py: --gpus %d requested but %d CUDA device(s) are visible; refusing to run fewer GPUs than reported"
              % (args.gpus, have), file=sys.stderr)
        return 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


# ------------------------------------------------------------------ the map-comparison row
def run_mapstats(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    print(json.dumps(mapstats_line(args)))
    return 0


def mapstats_line(args):
    """--row mapstats: pixels/s of ml_map_compare (RMS in magnitudes + two-sample K-S) on two
    seeded synthetic 4096^2 count maps (the map size of C4) resident in HBM; HBM roofline."""
    import torch
    import paper_1005_5198_b200 as ml
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    n_pix, n_rays = 4096, 100.0
    rng = np.random.default_rng(5)
    a = rng.poisson(5.0 * n_rays * rng.lognormal(0.0, 0.7, size=(n_pix, n_pix))).astype(np.uint32)
    b = np.clip(a.astype(np.int64) + rng.integers(-30, 31, size=a.shape), 0, None).astype(np.uint32)
    n = a.size
    ta = torch.from_numpy(a.view(np.int32)).to(dev)
    tb = torch.from_numpy(b.view(np.int32)).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.Stream(device=dev)

    def step():
        with torch.cuda.stream(stream):
            flush.fill_(1)
        return ml.ml_map_compare(ta.data_ptr(), n_rays, tb.data_ptr(), n_rays, n=n, device=dev.index,
                                 cuda_stream=stream.cuda_stream)

    for _ in range(args.warmup):
        r = step()
    # The timed region lasts a few ms and a polling nvidia-smi slows the host side of short calls threefold, so the
    # clocks are sampled over one second of the same load immediately BEFORE the timed region, then the sampler stops.
    sampler = ClockSampler(dev.index)
    sampler.start()
    t_end = time.perf_counter() + 1.5
    while time.perf_counter() < t_end:
        step()
    clocks = sampler.stop()
    clocks["when"] = "1.5 s of the same calls immediately before the timed region (see bench.py)"
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms, pass_ms = 0.0, 0.0
    e0.record(stream)
    for _ in range(args.steps):
        r = step()
        kernel_ms += r["kernel_ms"]
        pass_ms += r["pass_kernel_ms"]
    e1.record(stream)
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1)
    # wall clock of the call alone (device-resident maps, no L2 flush in between): what a user of the call waits for
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for _ in range(max(args.steps, 20)):
        ml.ml_map_compare(ta.data_ptr(), n_rays, tb.data_ptr(), n_rays, n=n, device=dev.index, cuda_stream=stream.cuda_stream)
    call_ms = 1e3 * (time.perf_counter() - t0) / max(args.steps, 20)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r_host = ml.ml_map_compare(a, n_rays, b, n_rays, device=dev.index)   # host buffers: H2D inside
    e2e_s = time.perf_counter() - t0
    assert r_host["rms_delta_m"] == r["rms_delta_m"] and r_host["ks_d"] == r["ks_d"]
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs") or 6500.0)
    algo_bytes = 2 * 4 * n
    achieved = algo_bytes / (pass_ms / args.steps * 1e-3) / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import mapstats_oracle as mo
        sa, sb = a[:2048, :2048], b[:2048, :2048]
        t0 = time.perf_counter()
        rms, _ = mo.rms_delta_m(sa, n_rays, sb, n_rays)
        d = mo.ks_statistic(sa, n_rays, sb, n_rays)
        mo.ks_probability(d, sa.size, sb.size)
        dt = time.perf_counter() - t0
        cpu = {"value": sa.size / dt, "unit": "pixels/s", "cores": 1, "kind": "oracle",
               "sample": "2048x2048 corner of the same two maps: rms + K-S distance + Q_KS in %.2f s" % dt}
    line = {"metric": "map-comparison pixels/sec (RMS in magnitudes + two-sample K-S, PAPER.md:169-173)",
            "value": n * args.steps / (ms * 1e-3), "unit": "pixels/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "mapstats: two seeded synthetic 4096^2 uint32 count maps (C4's map size), n_rays=100",
                       "l2": "flushed between steps (256 MiB write); the two maps (134 MB) exceed L2 anyway"},
            "result": {k: r[k] for k in ("rms_delta_m", "ks_d", "ks_prob", "n_valid")},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": NCU_MAPSTATS_DRAM_BYTES[0], "pass_kernel_ms": pass_ms / args.steps,
                         "all_kernels_ms_per_call": kernel_ms / args.steps,
                         "note": "dominant kernel = mlstats::pass_kernel (fused RMS + statistics + count histograms); "
                                 "algorithmic bytes = 2 maps x 4 B x n pixels read once; time = CUDA events around that "
                                 "launch on the launching stream (ml_map_compare_result.pass_kernel_ms); traffic = ncu "
                                 "dram bytes read + written of that launch (%s); "
                                 "peak = MEASURED_PEAKS.json hbm_gbs" % NCU_MAPSTATS_DRAM_BYTES[1]},
            "cpu_baseline": cpu, "clocks": clocks,
            "e2e": {"value": n * args.steps / e2e_s, "unit": "pixels/s", "h2d_bytes_per_step": 2 * 4 * n,
                    "d2h_bytes_per_step": 112},
            "gpu_launches": 7 * args.steps,   # pass, reduce, three scan kernels, K-S, finalize (+ one memset) per call
            "call_ms_without_flush": call_ms}
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", help="C1..C5 (BASELINE.json configs); the metric is quoted on C2")
    ap.add_argument("--precision", default="fp32_tiled", choices=sorted(PRECISIONS))
    ap.add_argument("--row", default="shoot", choices=["shoot", "mapstats"],
                    help="shoot = the hot path (default, the BASELINE.json metric); mapstats = the map-comparison row")
    ap.add_argument("--masses", action="store_true", help="unequal lens masses (eq. 4 with m_i): the MASS kernel instantiations")
    ap.add_argument("--random-rays", action="store_true", help="ML_RAYS_RANDOM: the paper's GPU-D ray generation")
    ap.add_argument("--uniform-rays", action="store_true",
                    help="ML_RAYS_UNIFORM: independent uniform ray positions over the whole rectangle (Poisson noise)")
    ap.add_argument("--n-lenses", type=int, default=0, help="override the lens count (large-N* row); 0 = eq. 5")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true",
                    help="skip the per_config block (C1, C5, C3, C4 after the C2 timed region) of the default line")
    ap.add_argument("--ref-seconds-per-step", type=float, default=None,
                    help="--impl reference: oracle seconds per step (default: 120 s spread over steps + warmup, 1-20 s each)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: --warmup < 3 breaks the timing rules", file=sys.stderr)
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    if args.row == "mapstats":
        return run_mapstats(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
