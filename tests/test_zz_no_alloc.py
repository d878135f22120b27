"""-m gpu test of ml_delta_m_histogram_static, the entry point for callers that cannot allocate device memory.

Why the entry point exists: a program that gave the GPU's memory to its own pool at start-up (torch's caching allocator, a
serving arena) makes every later cudaMalloc inside a library fail, and a program that renders maps in a loop beside other
GPU work cannot afford the device-wide stall of cudaMalloc / cudaFree.  ml_delta_m_histogram allocates a per-device cache;
the _static variant runs the same kernels on a fixed 1 MiB array built into the library, so counts must stay below
ML_STATIC_MAX_COUNT = 2^18.

What is checked: the histogram is an integer result, so -- like tests/test_gpu_mapstats.py does against the oracle -- it has
to equal the existing path's (ml_delta_m_histogram) bit for bit, on two calls in a row that share the built-in array (the
second map is dimmer than the first, so anything the first call left behind would show), into an output buffer that held
garbage; the device's free memory must not shrink across the second call; a map beyond the limit is refused with
ML_ERR_LIMIT and the next call is still right.

This file sorts last on purpose (pytest -x stops at the first failure: nothing may hide behind it) and does not depend
on what ran before it: alone in a fresh process its first call performs the per-device set-up.
"""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml

pytestmark = pytest.mark.gpu


def synth_map(seed, shape, mean):
    """Seeded count map shaped like a magnification map: log-normal magnification field, Poisson counts, a few zeros."""
    rng = np.random.default_rng(seed)
    m = rng.poisson(mean * rng.lognormal(0.0, 0.7, size=shape)).astype(np.uint32)
    m.ravel()[rng.integers(0, m.size, 5)] = 0
    return m


def static_histogram(torch, counts_host, n_rays, lo, hi, n_bins, stream=None):
    """Caller-side allocations only: the input map and the output bins are torch tensors; the output starts as garbage."""
    d_counts = torch.from_numpy(counts_host.view(np.int32).ravel().copy()).cuda()
    d_out = torch.full((n_bins,), -7, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    ml.ml_delta_m_histogram_static(d_counts.data_ptr(), n_rays, d_counts.numel(), lo, hi, n_bins, d_out.data_ptr(),
                                   cuda_stream=stream.cuda_stream if stream is not None else None)
    return d_out.cpu().numpy().view(np.uint64)


def test_static_scratch_histogram_equals_the_allocating_path_twice_in_a_row():
    import torch
    bright = synth_map(21, (1031, 517), mean=6000.0)   # counts up to several 1e4: most of the 2^18 bins' low end is touched
    dim = synth_map(22, (640, 480), mean=40.0)         # second call: far fewer distinct counts than the first left behind
    assert int(bright.max()) < ml.ML_STATIC_MAX_COUNT and int(dim.max()) < int(bright.max())
    cases = [(bright, 2000.0, -3.003, 2.999, 97), (dim, 15.0, -2.5, 2.5, 1000)]
    side = torch.cuda.Stream()
    got = []
    for k, (m, n_rays, lo, hi, nb) in enumerate(cases):    # the two calls in a row, nothing of this library in between
        if k == 1:
            free_before = torch.cuda.mem_get_info()[0]
        got.append(static_histogram(torch, m, n_rays, lo, hi, nb, stream=side if k == 1 else None))
    # ours allocated nothing between the calls; torch's own tensors of call 2 come out of its cache or shrink `free`,
    # so only compare after handing them back
    torch.cuda.empty_cache()
    assert torch.cuda.mem_get_info()[0] >= free_before
    for (m, n_rays, lo, hi, nb), h in zip(cases, got):
        want = ml.ml_delta_m_histogram(m, n_rays, lo, hi, nb)    # the existing, allocating path (host map)
        assert h.dtype == want.dtype and np.array_equal(h, want), (n_rays, lo, hi, nb)
        assert int(h.sum()) > 0.9 * m.size                       # a real histogram, not two empty ones


def test_static_scratch_limit_and_arguments():
    import torch
    m = synth_map(23, (300, 300), mean=500.0)
    over = m.copy()
    over[17, 4] = ml.ML_STATIC_MAX_COUNT                       # first count the built-in histogram cannot hold
    d_over = torch.from_numpy(over.view(np.int32).ravel().copy()).cuda()
    d_out = torch.zeros(64, dtype=torch.int64, device="cuda")
    with pytest.raises(ml.MicrolensError) as e:
        ml.ml_delta_m_histogram_static(d_over.data_ptr(), 100.0, d_over.numel(), -3.0, 3.0, 64, d_out.data_ptr())
    assert e.value.code == ml.ML_ERR_LIMIT and "built-in scratch" in str(e.value)
    edge = m.copy()
    edge[17, 4] = ml.ML_STATIC_MAX_COUNT - 1                   # the largest count it can: last bin of the array
    for cur in (edge, m):                                        # and the refused call left nothing behind that matters
        h = static_histogram(torch, cur, 100.0, -9.0, 3.0, 64)
        assert np.array_equal(h, ml.ml_delta_m_histogram(cur, 100.0, -9.0, 3.0, 64))
    ok = (d_over.data_ptr(), 100.0, d_over.numel(), -3.0, 3.0, 64, d_out.data_ptr())
    for pos, bad in [(0, 0), (6, 0), (0, d_over.data_ptr() + 2), (6, d_out.data_ptr() + 4), (1, 0.0), (2, 0), (4, -3.0),
                     (5, 0), (5, (1 << 20) + 1)]:
        args = list(ok)
        args[pos] = bad
        with pytest.raises(ml.MicrolensError) as e:
            ml.ml_delta_m_histogram_static(*args)
        assert e.value.code == ml.ML_ERR_INVALID_ARG, (pos, bad)
    with pytest.raises(ml.MicrolensError) as e:
        ml.ml_delta_m_histogram_static(*ok, device=99)
    assert e.value.code == ml.ML_ERR_CUDA
