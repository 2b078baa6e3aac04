"""GPU parity on the five BASELINE.json configurations (synthetic stand-ins, see
workloads/lightcurves.py), every one at its FULL size on the device.  Configs 1 and 2:
every position of every star against the oracle.  Configs 3-5: every
position of the stars {b : b mod q = 0} (q stated in each test; stars are independent and
separately seeded), sampled positions + tile seams over all stars, and the closed-form NaN
pattern over the whole array.
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


def test_config1_tess_single_every_position(umi):
    cfg, flux = lc.make(1)
    ref = orc.detrend(flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(_run(umi, flux, cfg, n_iter=0), ref.median)
    rep = parity.compare_trend(_run(umi, flux, cfg), ref)
    assert rep.n == 19440 and rep.n_nan == 0


def _nan_pattern_on_device(flux_d, got_d, W):
    """Closed-form NaN pattern over the whole array (R4, R5): own sample invalid, or fewer than
    max(1, W/3) valid samples in the window.  Bookkeeping on validity flags only, in chunks of stars."""
    import torch
    S, N = flux_d.shape
    h = W // 2
    idx = torch.arange(N, device=flux_d.device)
    lo = torch.clamp(idx - h, 0, N)
    hi = torch.clamp(idx + h + 1, 0, N)
    for s0 in range(0, S, 512):
        valid = torch.isfinite(flux_d[s0:s0 + 512])
        csum = torch.zeros((valid.shape[0], N + 1), dtype=torch.int32, device=flux_d.device)
        csum[:, 1:] = torch.cumsum(valid, dim=1, dtype=torch.int32)
        n_valid = csum[:, hi] - csum[:, lo]
        expect = ~valid | (n_valid < max(1, W // 3))
        assert torch.equal(torch.isnan(got_d[s0:s0 + 512]), expect), "NaN pattern differs in stars %d.." % s0


def _full_size(umi, config_id, q, n_samples):
    """The whole configuration resident on the device, one umi_detrend call (the launch configuration
    bench.py times); oracle on every position of the stars b = 0 mod q and on n_samples random
    (star, position) pairs + tile seams of all stars."""
    import torch
    cfg, flux = lc.make(config_id)
    S, N = flux.shape
    assert (S, N) == (cfg.n_stars, cfg.n_cadences)
    fd = torch.from_numpy(flux).cuda()
    med_d = umi.umi_detrend(None, fd, cfg.W, alpha=cfg.alpha, n_iter=0)
    got_d = umi.umi_detrend(None, fd, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    torch.cuda.synchronize()
    _nan_pattern_on_device(fd, got_d, cfg.W)
    assert torch.equal(torch.isnan(med_d), torch.isnan(got_d))
    # every position of every q-th star
    sub = np.arange(0, S, q)
    ref = orc.detrend(flux[sub], cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    parity.compare_median(med_d[sub].cpu().numpy(), ref.median)
    rep = parity.compare_trend(got_d[sub].cpu().numpy(), ref)
    # random positions and tile seams of all stars
    rng = np.random.default_rng(config_id)
    T1, _, T2 = umi.umi_launch_geometry(cfg.W)
    seams = []
    for T in (T1, T2, 4 * T2, 512):
        for k in range(1, 4):
            seams += [k * T - 1, k * T]
    seams += [0, 1, cfg.W // 2, N - 1, N - 2, N - 1 - cfg.W // 2]
    seams = np.array([p for p in seams if 0 <= p < N], dtype=np.int64)
    sb = np.concatenate([rng.integers(0, S, n_samples), rng.integers(0, S, seams.size)])
    sp = np.concatenate([rng.integers(0, N, n_samples), seams])
    refp = orc.positions(flux, sb, sp, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    sbd, spd = torch.from_numpy(sb).cuda(), torch.from_numpy(sp).cuda()
    parity.compare_median(med_d[sbd, spd].cpu().numpy(), refp.median)
    parity.compare_trend(got_d[sbd, spd].cpu().numpy(), refp)
    return cfg, flux, got_d, rep


def test_config2_tess_batch_every_position_of_every_star(umi):
    # "all stars for configs 1-2" -- 1,000 x 19,440 positions, ~25 s of oracle on 16 cores
    cfg, flux, got_d, rep = _full_size(umi, 2, q=1, n_samples=1000)
    assert rep.n == 1000 * 19440 and rep.n_nan > 0        # the 1-day gap
    print("config 2: %d positions, %d NaN, max rel err %.2e, %d near-cutoff (max %.2e)"
          % (rep.n, rep.n_nan, rep.max_rel, rep.n_flagged, rep.max_rel_flagged))


def test_config3_kepler_full_size(umi):
    # 10,000 x 70,000 on the device (fused short-window kernel); q = 50: every position of 200 stars
    _full_size(umi, 3, q=50, n_samples=20000)


def test_config4_tess20s_full_size(umi):
    # 200 x 116,640, W = 2161; q = 100: every position of stars 0 and 100 (the oracle is O(W) per position)
    _full_size(umi, 4, q=100, n_samples=4000)


def test_config5_ffi_sweep_full_size(umi):
    # 100,000 x 11,664 resident on the device, one call; q = 500: every position of 200 stars;
    # then the same stars through the host batch driver (streams, H2D / kernels / D2H): same kernels, same bits
    import torch
    cfg, flux, got_d, rep = _full_size(umi, 5, q=500, n_samples=8000)
    n_host = 6000
    out = np.empty_like(flux[:n_host])
    umi.umi_detrend_host(None, flux[:n_host], cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter, out=out,
                         stars_per_batch=700, n_streams=3)
    assert np.array_equal(out, got_d[:n_host].cpu().numpy(), equal_nan=True)


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


@pytest.mark.parametrize("W,n_iter", [(361, 5), (361, 0), (25, 5), (2161, 5)])
def test_host_path_single_small_batch_pinned_and_pageable(umi, W, n_iter):
    # the latency case (config 1's shape): one batch, caller-supplied pinned output (CPU tensors go through by address,
    # no numpy round trip) and pageable numpy buffers.  Both must equal the device entry point bit for bit, and the
    # oracle to tolerance.
    import torch
    flux = lc.stars(1, range(1)).copy()
    flux[0, 4000:4700] = np.nan                             # a gap longer than the short windows
    ref = orc.detrend(flux, W, n_iter=n_iter)
    dev = umi.umi_detrend(None, torch.from_numpy(flux).cuda(), W, n_iter=n_iter).cpu().numpy()
    pinned_in = torch.from_numpy(flux).pin_memory()
    pinned_out = torch.full(flux.shape, 7.0, dtype=torch.float32).pin_memory()
    got = umi.umi_detrend_host(None, pinned_in, W, n_iter=n_iter, out=pinned_out)
    assert got is pinned_out
    np.testing.assert_array_equal(got.numpy(), dev)
    pageable = umi.umi_detrend_host(None, flux, W, n_iter=n_iter)
    np.testing.assert_array_equal(pageable, dev)
    if n_iter == 0:
        parity.compare_median(got.numpy(), ref.median)
    else:
        parity.compare_trend(got.numpy(), ref)
    # a view into the middle of a pinned allocation, and two stars forced into one batch
    two = lc.stars(1, range(2))
    big = torch.empty(3 * two.size, dtype=torch.float32).pin_memory()
    out2 = big[two.size // 2: two.size // 2 + two.size].view(two.shape)
    umi.umi_detrend_host(None, torch.from_numpy(two).pin_memory(), W, n_iter=n_iter, out=out2, stars_per_batch=2)
    dev2 = umi.umi_detrend(None, torch.from_numpy(two).cuda(), W, n_iter=n_iter).cpu().numpy()
    np.testing.assert_array_equal(out2.numpy(), dev2)


@pytest.mark.parametrize("want_trend", [True, False])
def test_flatten_host_caller_supplied_pinned_outputs(umi, want_trend):
    import torch
    flux = lc.stars(1, range(1))
    W = 361
    tr_dev, fl_dev = umi.umi_flatten(None, torch.from_numpy(flux).cuda(), W)
    out_trend = torch.empty(flux.shape, dtype=torch.float32).pin_memory() if want_trend else None
    out_flat = torch.empty(flux.shape, dtype=torch.float32).pin_memory()
    tr, fl = umi.umi_flatten_host(None, torch.from_numpy(flux).pin_memory(), W, want_trend=want_trend,
                                  out_trend=out_trend, out_flat=out_flat)
    assert fl is out_flat and (tr is out_trend)
    np.testing.assert_array_equal(fl.numpy(), fl_dev.cpu().numpy())
    if want_trend:
        np.testing.assert_array_equal(tr.numpy(), tr_dev.cpu().numpy())
    ref = orc.detrend(flux, W)
    parity.compare_trend((flux / fl.numpy()).astype(np.float32), ref, tol=2e-5)   # flat = flux / trend, rounded twice
