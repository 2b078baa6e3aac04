"""GPU parity on the five BASELINE.json configurations (synthetic stand-ins, see
workloads/lightcurves.py).  Config 1 and a star subset of config 2 are compared at
every position; the full-size runs (the launch configuration bench.py times) are
compared on sampled positions the oracle computes one by one, plus the NaN pattern.
"""
import numpy as np
import pytest

from oracle import umi_oracle as orc
from tests import parity
from workloads import lightcurves as lc

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def umi():
    import paper_2604_06602_b200 as m
    m.lib()
    return m


def _run(umi, flux, cfg, n_iter=None):
    import torch
    f = torch.from_numpy(flux).cuda()
    out = umi.umi_detrend(None, f, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter if n_iter is None else n_iter)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _sampled(umi, cfg, flux, n_samples, seed):
    """Full-size device run, oracle on random (star, position) samples + tile seams."""
    S, N = flux.shape
    rng = np.random.default_rng(seed)
    sb = rng.integers(0, S, n_samples)
    sp = rng.integers(0, N, n_samples)
    T1, _, T2 = umi.umi_launch_geometry(cfg.W)
    seams = []
    for T in (T1, T2):
        for k in range(1, 4):
            seams += [k * T - 1, k * T]
    seams += [0, 1, cfg.W // 2, N - 1, N - 2, N - 1 - cfg.W // 2]
    seams = np.array([p for p in seams if 0 <= p < N], dtype=np.int64)
    sb = np.concatenate([sb, rng.integers(0, S, seams.size)])
    sp = np.concatenate([sp, seams])
    med = _run(umi, flux, cfg, n_iter=0)
    ref = orc.positions(flux, sb, sp, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(med[sb, sp], ref.median)
    del med
    got = _run(umi, flux, cfg)
    rep = parity.compare_trend(got[sb, sp], ref)
    # NaN pattern over the whole array: invalid own sample, or window below W/3 valid (R4, R5)
    valid = np.isfinite(flux)
    csum = np.concatenate([np.zeros((S, 1), np.int64), np.cumsum(valid, axis=1, dtype=np.int64)], axis=1)
    h = cfg.W // 2
    lo = np.clip(np.arange(N) - h, 0, N)
    hi = np.clip(np.arange(N) + h + 1, 0, N)
    n_valid = csum[:, hi] - csum[:, lo]
    expect_nan = ~valid | (n_valid < max(1, cfg.W // 3))
    assert np.array_equal(np.isnan(got), expect_nan)
    return rep


def test_config1_tess_single_every_position(umi):
    cfg, flux = lc.make(1)
    ref = orc.detrend(flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(_run(umi, flux, cfg, n_iter=0), ref.median)
    rep = parity.compare_trend(_run(umi, flux, cfg), ref)
    assert rep.n == 19440 and rep.n_nan == 0


def test_config2_tess_batch_subset_every_position(umi):
    cfg = lc.CONFIGS[2]
    idx = list(range(0, 1000, 21))           # 48 separately seeded stars
    flux = lc.stars(2, idx)
    ref = orc.detrend(flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(_run(umi, flux, cfg, n_iter=0), ref.median)
    rep = parity.compare_trend(_run(umi, flux, cfg), ref)
    assert rep.n_nan > 0                      # the 1-day gap


def test_config2_tess_batch_full_size_sampled(umi):
    cfg, flux = lc.make(2)
    assert flux.shape == (1000, 19440)
    _sampled(umi, cfg, flux, 20000, seed=2)


def test_config3_kepler_reduced_and_sampled(umi):
    cfg = lc.CONFIGS[3]
    flux = lc.stars(3, range(0, 10000, 1250))           # 8 stars, every position
    ref = orc.detrend(flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(_run(umi, flux, cfg, n_iter=0), ref.median)
    parity.compare_trend(_run(umi, flux, cfg), ref)
    flux = lc.stars(3, range(1000))                     # 1000 x 70000, sampled
    _sampled(umi, cfg, flux, 20000, seed=3)


def test_config4_tess20s_reduced_and_sampled(umi):
    cfg = lc.CONFIGS[4]
    flux = lc.stars(4, [0, 199])
    sl = flux[:, 50000:62000].copy()                    # spans the NaN gap; every position
    ref = orc.detrend(sl, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(_run(umi, sl, cfg, n_iter=0), ref.median)
    parity.compare_trend(_run(umi, sl, cfg), ref)
    cfg, flux = lc.make(4)                              # full size 200 x 116640, sampled
    _sampled(umi, cfg, flux, 4000, seed=4)


def test_config5_ffi_sweep_reduced_and_sampled(umi):
    cfg = lc.CONFIGS[5]
    flux = lc.stars(5, range(0, 100000, 5000))          # 20 stars, every position
    ref = orc.detrend(flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(_run(umi, flux, cfg, n_iter=0), ref.median)
    parity.compare_trend(_run(umi, flux, cfg), ref)
    flux = lc.stars(5, range(6000))                     # 6000 x 11664 through the host batch driver
    out = np.empty_like(flux)
    umi.umi_detrend_host(None, flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter, out=out,
                         stars_per_batch=700, n_streams=3)
    dev = _run(umi, flux, cfg)
    assert np.array_equal(out, dev, equal_nan=True)     # same kernels, same bits
    rng = np.random.default_rng(5)
    sb, sp = rng.integers(0, 6000, 8000), rng.integers(0, cfg.n_cadences, 8000)
    ref = orc.positions(flux, sb, sp, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_trend(out[sb, sp], ref)


def test_host_path_with_time_and_pinned_memory(umi):
    import torch
    cfg = lc.CONFIGS[2]
    flux = torch.from_numpy(lc.stars(2, range(10))).pin_memory()
    t = lc.times(2, 10)
    t[3, 500:900] = np.nan
    out = umi.umi_detrend_host(torch.from_numpy(t), flux, cfg.W, stars_per_batch=3, n_streams=2)
    ref = orc.detrend(flux.numpy(), cfg.W, time=t)
    parity.compare_trend(out.numpy(), ref)


@pytest.mark.parametrize("n_stars", [1, 2, 5, 23, 131])
def test_host_path_default_batches_ramp_up_and_down(umi, n_stars):
    # default batching (stars_per_batch <= 0): ramp / body / ramp sizes must cover every star exactly once,
    # also when the job is smaller than one ramp; called twice (the second call reuses the cached streams)
    import threading
    cfg = lc.CONFIGS[5]
    flux = lc.stars(5, range(n_stars))
    ref = orc.detrend(flux, cfg.W)
    for _ in range(2):
        out = umi.umi_detrend_host(None, flux, cfg.W)
        parity.compare_trend(out, ref)
    # another host thread gets streams of its own
    res = {}
    th = threading.Thread(target=lambda: res.setdefault("out", umi.umi_detrend_host(None, flux, cfg.W, n_streams=5)))
    th.start()
    th.join()
    parity.compare_trend(res["out"], ref)
