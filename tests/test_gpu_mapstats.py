"""-m gpu parity tests of the device map comparison (ml_map_compare, ml_delta_m_histogram; PAPER.md:169-173,
eq. 10) against oracle/mapstats_oracle.py on the same seeded maps, through the C ABI.

Bar: integer outputs (pixel counts, sums, maxima, histograms) bit-exact; the K-S distance is a difference of two
integer ratios, compared to 1e-14 absolute; RMS (fp64 log10 of up to 1.7e7 pixels, fixed summation order on the
device, numpy pairwise on the host) to 1e-11 relative -- both sides form Delta m_a - Delta m_b from two rounded
logarithms (absolute error <= ~2e-15 per pixel against differences of 1e-3 mag and more); Q_KS to 1e-10.
"""
import numpy as np
import pytest

import paper_1005_5198_b200 as ml
from oracle import mapstats_oracle as mo
from oracle import oracle
from workloads import CONFIGS, lens_disk

pytestmark = pytest.mark.gpu


def synth_map(seed, shape, mean=300.0, zeros=0):
    """Seeded synthetic count map shaped like a magnification map: log-normal magnification field, Poisson counts."""
    rng = np.random.default_rng(seed)
    lam = mean * rng.lognormal(0.0, 0.7, size=shape)
    m = rng.poisson(lam).astype(np.uint32)
    if zeros:
        idx = rng.integers(0, m.size, zeros)
        m.ravel()[idx] = 0
    return m


def check(a, na, b, nb, **kw):
    r = ml.ml_map_compare(a, na, b, nb, **kw)
    a_h, b_h = np.asarray(a), np.asarray(b)
    assert r["n_pixels"] == a_h.size
    assert r["sum_a"] == int(a_h.sum(dtype=np.uint64)) and r["sum_b"] == int(b_h.sum(dtype=np.uint64))
    assert r["max_a"] == int(a_h.max()) and r["max_b"] == int(b_h.max())
    assert r["n_empty_a"] == int((a_h == 0).sum()) and r["n_empty_b"] == int((b_h == 0).sum())
    rms, n_valid = mo.rms_delta_m(a_h, na, b_h, nb)
    assert r["n_valid"] == n_valid
    assert abs(r["rms_delta_m"] - rms) <= 1e-11 * max(rms, 1e-300) + 1e-15, (r["rms_delta_m"], rms)
    d = mo.ks_statistic(a_h, na, b_h, nb)
    assert abs(r["ks_d"] - d) <= 1e-14, (r["ks_d"], d)
    q = mo.ks_probability(d, a_h.size, b_h.size)
    assert abs(r["ks_prob"] - q) <= 1e-10, (r["ks_prob"], q)
    assert abs(r["mean_mu_a"] - mo.mean_mu(a_h, na)) <= 1e-13 * mo.mean_mu(a_h, na) + 1e-300
    assert abs(r["mean_mu_b"] - mo.mean_mu(b_h, nb)) <= 1e-13 * mo.mean_mu(b_h, nb) + 1e-300
    return r


@pytest.mark.parametrize("shape", [(1,), (5,), (1000,), (64, 64), (1031, 517), (1024, 1024)])
@pytest.mark.parametrize("rays", [(100.0, 100.0), (100.0, 250.0), (37.5, 100.0)])
def test_compare_matches_the_oracle_on_seeded_maps(shape, rays):
    na, nb = rays
    a = synth_map(1, shape, mean=3.0 * na, zeros=3 if np.prod(shape) > 100 else 0)
    b = synth_map(2, shape, mean=3.1 * nb, zeros=5 if np.prod(shape) > 100 else 0)
    r = check(a, na, b, nb)
    if np.prod(shape) >= 4096:
        assert 0.0 < r["ks_d"] < 1.0 and r["rms_delta_m"] > 0.0


def test_compare_full_size_map_pair():
    # C5-sized maps (2048^2): several tiles of every kernel, ragged scan tail
    a = synth_map(11, (2048, 2048), mean=4000.0, zeros=17)
    noise = np.random.default_rng(12).integers(-40, 41, size=a.shape)
    b = np.clip(a.astype(np.int64) + noise, 0, None).astype(np.uint32)
    r = check(a, 500.0, b, 500.0)
    print("2048^2 pair: rms %.6f mag, D %.3e, P %.4f, kernels %.3f ms" % (r["rms_delta_m"], r["ks_d"], r["ks_prob"], r["kernel_ms"]))


def test_degenerate_maps():
    z = np.zeros(1000, dtype=np.uint32)
    r = check(z, 10.0, z, 10.0)                       # nothing lit: no valid pixel, identical distributions
    assert r["n_valid"] == 0 and r["rms_delta_m"] == 0.0 and r["ks_d"] == 0.0 and r["ks_prob"] == 1.0
    u = np.full((300, 300), 272, dtype=np.uint32)     # the uniform map of eq. 12: every lane holds the same count
    r = check(u, 100.0, u, 100.0)
    assert r["rms_delta_m"] == 0.0 and r["ks_d"] == 0.0
    r = check(u, 100.0, 2 * u, 100.0)                  # disjoint distributions, constant 2.5 log10(2) apart
    assert r["ks_d"] == 1.0 and abs(r["rms_delta_m"] - 2.5 * np.log10(2.0)) < 1e-14 and r["ks_prob"] < 1e-100
    r = check(u, 100.0, 2 * u, 200.0)                  # the same magnification map recorded with twice the rays
    assert r["ks_d"] == 0.0 and r["rms_delta_m"] < 1e-15
    check(z, 10.0, u.ravel()[:1000], 10.0)


def test_counts_beyond_the_first_pass_histogram():
    a = synth_map(3, (257, 129), mean=500.0)
    b = synth_map(4, (257, 129), mean=500.0)
    a[7, 7] = 3_000_001                                # > 2^20 bins: second histogram pass
    b[100, 3] = (1 << 20)                              # exactly the first-pass bin count
    check(a, 100.0, b, 100.0)
    c = a.copy()
    c[0, 0] = 1 << 27
    with pytest.raises(ml.MicrolensError) as e:
        ml.ml_map_compare(a, 100.0, c, 100.0)
    assert e.value.code == ml.ML_ERR_OOM


def test_histogram_matches_the_oracle():
    for seed, shape, n_rays in [(5, (640, 480), 150.0), (6, (33,), 10.0), (7, (1024, 1024), 2000.0)]:
        a = synth_map(seed, shape, mean=2.5 * n_rays, zeros=4)
        for lo, hi, nb in [(-3.003, 2.999, 97), (-0.4871, 0.5123, 1000), (-10.01, 10.02, 1)]:
            h = ml.ml_delta_m_histogram(a, n_rays, lo, hi, nb)
            assert np.array_equal(h, mo.histogram_delta_m(a, n_rays, lo, hi, nb)), (seed, lo, hi, nb)


def test_device_pointers_on_real_maps_fp32_vs_fp64():
    """The use the paper makes of these measures (section 3.1), applied to the two precision modes: C1 shot in
    FP32 and in fp64, compared in place on the device (borrowed device pointers, unaligned offset included)."""
    import torch
    p = CONFIGS[0]
    args = (p.sigma, p.stellar_fraction, p.gamma, p.n_pix, p.n_rays, p.L)
    g = oracle.geometry(*args)
    xy = lens_disk(g.n_star, g.r_star, p.seed)
    with ml.MagnificationMap(*args) as m32, ml.MagnificationMap(*args, precision=ml.ML_PREC_FP64) as m64:
        for m in (m32, m64):
            m.set_lenses(xy)
            m.shoot()
        n = p.n_pix * p.n_pix
        r = ml.ml_map_compare(ml.ml_get_map_device(m32.ctx), p.n_rays, ml.ml_get_map_device(m64.ctx), p.n_rays, n=n)
        a, b = m32.counts(), m64.counts()
    rms, nv = mo.rms_delta_m(a, p.n_rays, b, p.n_rays)
    assert r["n_valid"] == nv and abs(r["rms_delta_m"] - rms) <= 1e-11 * rms + 1e-15
    assert abs(r["ks_d"] - mo.ks_statistic(a, p.n_rays, b, p.n_rays)) <= 1e-14
    # "excellent agreement" in the paper's sense: RMS < 0.2 mag and P(KS) > 99.7 %
    assert r["rms_delta_m"] < 0.2 and r["ks_prob"] > 0.997
    print("C1 fp32 vs fp64: rms %.3e mag, D %.3e, P(KS) %.6f" % (r["rms_delta_m"], r["ks_d"], r["ks_prob"]))
    # torch-owned memory, a pointer that is only 4-byte aligned (scalar-load path), and a torch stream
    ta = torch.from_numpy(a.view(np.int32).ravel().copy()).cuda()
    tb = torch.from_numpy(b.view(np.int32).ravel().copy()).cuda()
    s = torch.cuda.Stream()
    r2 = ml.ml_map_compare(ta.data_ptr() + 4, p.n_rays, tb.data_ptr() + 4, p.n_rays, n=n - 1, cuda_stream=s.cuda_stream)
    rms2, nv2 = mo.rms_delta_m(a.ravel()[1:], p.n_rays, b.ravel()[1:], p.n_rays)
    assert r2["n_valid"] == nv2 and abs(r2["rms_delta_m"] - rms2) <= 1e-11 * rms2 + 1e-15


def test_argument_validation():
    a = np.ones(16, dtype=np.uint32)
    for bad in [dict(n_rays_a=0.0), dict(n_rays_b=-1.0), dict(n_rays_a=float("nan"))]:
        kw = dict(n_rays_a=10.0, n_rays_b=10.0)
        kw.update(bad)
        with pytest.raises(ml.MicrolensError) as e:
            ml.ml_map_compare(a, kw["n_rays_a"], a, kw["n_rays_b"])
        assert e.value.code == ml.ML_ERR_INVALID_ARG
    with pytest.raises(ml.MicrolensError):
        ml.ml_map_compare(np.zeros(0, dtype=np.uint32), 1.0, np.zeros(0, dtype=np.uint32), 1.0)
    with pytest.raises(ml.MicrolensError):
        ml.ml_delta_m_histogram(a, 10.0, 1.0, 1.0, 10)
    with pytest.raises(ml.MicrolensError) as e:
        ml.ml_map_compare(a, 10.0, a, 10.0, device=99)
    assert e.value.code == ml.ML_ERR_CUDA
