"""GPU parity for the rows SURVEY.md 8(f) marks "next": F1 fused normalisation
(umi_flatten) and F2 time-stamped gap handling (umi_detrend_gapped,
PAPER.md:155; R20), through the C ABI, against the fp64 oracle.
Bars: NaN pattern identical, median bit-exact, trend and flat within 1e-5 relative."""
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


def _cuda(a, dtype):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def _check_flat(flat_gpu, flux, ref):
    want = orc.normalize(flux, ref.trend64)
    got = flat_gpu.astype(np.float64)
    assert np.array_equal(np.isnan(got), np.isnan(want))
    ok = ~np.isnan(want) & ~ref.near_cutoff.astype(bool)
    if ok.any():
        rel = np.abs(got[ok] - want[ok]) / np.maximum(np.abs(want[ok]), 1e-30)
        assert rel.max() <= parity.TOL, rel.max()


@pytest.mark.parametrize("W", [1, 9, 25, 49, 51, 361, 1081])
@pytest.mark.parametrize("n_iter", [0, 5])
def test_flatten_matches_oracle(umi, W, n_iter):
    import torch
    x = lc.random_series(300 + W, 3, 2777)
    ref = orc.detrend(x, W, n_iter=n_iter)
    trend, flat = umi.umi_flatten(None, _cuda(x, np.float32), W, n_iter=n_iter)
    torch.cuda.synchronize()
    trend, flat = trend.cpu().numpy(), flat.cpu().numpy()
    if n_iter == 0:
        parity.compare_median(trend, ref.median)
    else:
        parity.compare_trend(trend, ref)
    _check_flat(flat, x, ref)


def test_flatten_constant_series_is_exactly_one(umi):
    import torch
    x = np.full((2, 1500), 0.3, np.float32)
    for W in (25, 361):
        trend, flat = umi.umi_flatten(None, _cuda(x, np.float32), W)
        torch.cuda.synchronize()
        assert np.array_equal(flat.cpu().numpy(), np.ones_like(x))
        assert np.array_equal(trend.cpu().numpy(), x)


@pytest.mark.parametrize("W,jitter", [(5, 0.0), (25, 0.3), (51, 0.45), (361, 0.4), (1081, 0.2)])
def test_gapped_matches_oracle(umi, W, jitter):
    import torch
    dt = 2.0 / 1440
    grid = lc.random_series(500 + W, 3, 4001, nan_frac=0.04, inf_frac=0.0)
    grid[1, 1000:1000 + W + 40] = np.nan                  # a gap wider than the window
    t, f, slot = lc.compact(grid, dt, t0=2458000.25, jitter=jitter, seed=W)
    t[2, 17] = np.inf                                     # bad time stamp
    f[0, 33] = np.nan                                     # bad flux that survived compaction
    n_grid = grid.shape[1] - 7                            # the last slots fall outside the grid
    ref = orc.gapped(t, f, 2458000.25, dt, n_grid, W)
    td, fd = _cuda(t, np.float64), _cuda(f, np.float32)
    med = umi.umi_detrend_gapped(td, fd, 2458000.25, dt, n_grid, W, n_iter=0)
    trend, flat = umi.umi_detrend_gapped(td, fd, 2458000.25, dt, n_grid, W, flat=True)
    torch.cuda.synchronize()
    parity.compare_median(med.cpu().numpy(), ref.median)
    parity.compare_trend(trend.cpu().numpy(), ref)
    _check_flat(flat.cpu().numpy(), f, ref)


def test_gapped_colliding_slots_and_empty_grid(umi):
    import torch
    dt = 0.02
    grid = lc.random_series(78, 2, 900, nan_frac=0.03, inf_frac=0.0)
    t, f, slot = lc.compact(grid, dt, t0=10.0, jitter=0.2, seed=2)
    t[0, 50] = t[0, 51] - 1e-9 * dt                       # two samples in one slot
    ref = orc.gapped(t, f, 10.0, dt, 900, 31)
    got = umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), 10.0, dt, 900, 31)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    parity.compare_trend(got, ref)
    assert np.isnan(got[0, 50]) and not np.isnan(got[0, 51])
    # n_grid = 0: every sample is outside the grid
    got = umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), 10.0, dt, 0, 31)
    torch.cuda.synchronize()
    assert np.isnan(got.cpu().numpy()).all()
    # a caller-owned workspace that is too small is refused on the host
    with pytest.raises(umi.UmiError):
        umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), 10.0, dt, 900, 31,
                               workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))


def test_gapped_tess_batch_stars_compacted(umi):
    # config-2 stars with their 1-day gap removed (PAPER.md:155 pipeline order), full length
    import torch
    cfg = lc.CONFIGS[2]
    grid = lc.stars(2, [3, 4])
    t, f, slot = lc.compact(grid, cfg.dt_days, t0=1468.27, jitter=0.1, seed=9)
    ref = orc.gapped(t, f, 1468.27, cfg.dt_days, cfg.n_cadences, cfg.W)
    trend, flat = umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), 1468.27, cfg.dt_days,
                                         cfg.n_cadences, cfg.W, flat=True)
    torch.cuda.synchronize()
    parity.compare_trend(trend.cpu().numpy(), ref)
    _check_flat(flat.cpu().numpy(), f, ref)


def _segment_rows(seed, S, N, dt):
    grid = lc.random_series(seed, S, N, nan_frac=0.03, inf_frac=0.0)
    rng = np.random.default_rng(seed)
    for b in range(S):                                      # wide gaps, and an island of a few samples
        for _ in range(4):
            a = int(rng.integers(50, N - 400))
            grid[b, a:a + int(rng.integers(30, 380))] = np.nan
        a = int(rng.integers(400, N - 400))
        grid[b, a - 200:a + 210] = np.nan
        grid[b, a:a + 9] = 1.0
    return lc.compact(grid, dt, t0=7.25, jitter=0.2, seed=seed)


@pytest.mark.parametrize("W,brk,mseg,ecut", [(25, 12, 12, 0), (25, 24, 0, 5), (51, 25, 17, 3), (361, 180, 120, 0),
                                              (361, 360, 120, 40), (361, -1, 0, 25), (217, 400, 72, 1)])
def test_gapped_segments_match_oracle(umi, W, brk, mseg, ecut):
    # reading R23: segments at gaps wider than break_slots, minimum segment length, edge cut
    import torch
    dt = 2.0 / 1440
    S, N = (5, 6001) if W > 49 else (3, 3001)
    t, f, slot = _segment_rows(600 + W + max(brk, 0), S, N, dt)
    ref = orc.gapped_ex(t, f, 7.25, dt, N, W, break_slots=brk, min_segment=mseg, edge_cut=ecut)
    td, fd = _cuda(t, np.float64), _cuda(f, np.float32)
    med = umi.umi_detrend_gapped(td, fd, 7.25, dt, N, W, n_iter=0, break_slots=brk, min_segment=mseg, edge_cut=ecut)
    trend, flat = umi.umi_detrend_gapped(td, fd, 7.25, dt, N, W, flat=True, break_slots=brk, min_segment=mseg, edge_cut=ecut)
    torch.cuda.synchronize()
    parity.compare_median(med.cpu().numpy(), ref.median)
    parity.compare_trend(trend.cpu().numpy(), ref)
    _check_flat(flat.cpu().numpy(), f, ref)
    if ecut > 0 or W == 25:                                               # the options did remove something the plain path keeps
        plain = orc.gapped(t, f, 7.25, dt, N, W)
        assert (np.isnan(ref.trend64) & ~np.isnan(plain.trend64)).any()


def test_gapped_segments_argument_rules(umi):
    import torch
    t, f, slot = _segment_rows(3, 2, 2001, 0.01)
    td, fd = _cuda(t, np.float64), _cuda(f, np.float32)
    with pytest.raises(umi.UmiError) as e:                                # a break a window could reach across
        umi.umi_detrend_gapped(td, fd, 7.25, 0.01, 2001, 51, break_slots=24)
    assert e.value.status == umi.UMI_ERR_UNSUPPORTED
    with pytest.raises(umi.UmiError):                                     # the plain workspace is too small for segments
        umi.umi_detrend_gapped(td, fd, 7.25, 0.01, 2001, 51, min_segment=17,
                               workspace=torch.empty(umi.umi_gapped_workspace_bytes(2, 2001), dtype=torch.uint8, device="cuda"))
    a = umi.umi_detrend_gapped(td, fd, 7.25, 0.01, 2001, 51)
    b = umi.umi_detrend_gapped(td, fd, 7.25, 0.01, 2001, 51, break_slots=10 ** 9)     # one segment: nothing changes
    torch.cuda.synchronize()
    assert torch.equal(torch.nan_to_num(a), torch.nan_to_num(b)) and torch.equal(torch.isnan(a), torch.isnan(b))


# ------------------------------------------------------------------ F4: sibling estimators
def _family_case(umi, x, W, sk, wk, alpha=2.0, c=5.0, n_iter=5, time=None):
    import torch
    ref = orc.family(x, W, sk, wk, alpha=alpha, c=c, n_iter=n_iter, time=time)
    t = None if time is None else _cuda(time, np.float64)
    trend, scale, flat = umi.umi_detrend_family(t, _cuda(x, np.float32), W, sk, wk, alpha=alpha, c=c,
                                                n_iter=n_iter, flat=True)
    torch.cuda.synchronize()
    trend, scale, flat = trend.cpu().numpy(), scale.cpu().numpy(), flat.cpu().numpy()
    if n_iter == 0:
        parity.compare_median(trend, ref.median)
    else:
        parity.compare_trend(trend, ref)
    _check_flat(flat, x, ref)
    # the scale: NaN pattern of the trend; the MAD is a difference of two samples (one fp32
    # rounding), the upper-RMS an fp32 sum of squares
    nan = np.isnan(ref.trend64)
    assert np.array_equal(np.isnan(scale), nan)
    want = ref.scale[~nan]
    got = scale[~nan].astype(np.float64)
    tol = 2e-7 if sk == 1 else 1e-5
    assert np.all(np.abs(got - want) <= tol * np.abs(want)), np.abs(got / np.maximum(want, 1e-300) - 1).max()


@pytest.mark.parametrize("W", [1, 5, 9, 25, 33, 49, 51, 217, 361, 1081])
@pytest.mark.parametrize("sk,wk", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_family_matches_oracle(umi, W, sk, wk):
    x = lc.random_series(700 + W + 2 * sk + wk, 3, 3001)
    _family_case(umi, x, W, sk, wk)


@pytest.mark.parametrize("W", [25, 361])
def test_family_median_and_scale_only(umi, W):
    x = lc.random_series(41 + W, 2, 2500, nan_frac=0.03)
    _family_case(umi, x, W, 1, 0, n_iter=0)
    _family_case(umi, x, W, 0, 0, n_iter=0)


@pytest.mark.parametrize("W", [25, 361])
def test_family_heavy_ties_and_presets(umi, W):
    x = lc.random_series(300 + W, 2, 2500, nan_frac=0.02, inf_frac=0.0, ties=True)
    _family_case(umi, x, W, 1, 0, alpha=1.0)          # classic symmetric biweight (MAD)
    _family_case(umi, x, W, 1, 1, alpha=1.0, c=2.5)
    y = lc.random_series(17, 2, 2000, nan_frac=0.02)
    _family_case(umi, y, W, 1, 0, alpha=10.0, c=2.5)
    _family_case(umi, y, W, 0, 1, alpha=3.0, n_iter=2)


def test_family_large_window_and_config_stars(umi):
    x = lc.random_series(8, 2, 9000, nan_frac=0.02)
    _family_case(umi, x, 2161, 1, 0)
    _family_case(umi, x, 4097, 1, 1)
    cfg = lc.CONFIGS[2]
    _family_case(umi, lc.stars(2, [5]), cfg.W, 1, 0, alpha=1.0)
    _family_case(umi, lc.stars(3, [2])[:, :20000], 25, 1, 0, alpha=1.0)


def test_family_constant_and_degenerate(umi):
    import torch
    x = np.full((2, 1200), 1.25, np.float32)
    for W in (9, 361):
        for sk in (0, 1):
            trend, scale = umi.umi_detrend_family(None, _cuda(x, np.float32), W, sk, 1)
            torch.cuda.synchronize()
            assert np.array_equal(trend.cpu().numpy(), x)
            assert np.array_equal(scale.cpu().numpy(), np.zeros_like(x))
    x = np.full((1, 800), np.nan, np.float32)
    trend, scale = umi.umi_detrend_family(None, _cuda(x, np.float32), 51, 1, 0)
    torch.cuda.synchronize()
    assert np.isnan(trend.cpu().numpy()).all() and np.isnan(scale.cpu().numpy()).all()


@pytest.mark.parametrize("case", range(16))
def test_fuzz_family_and_gapped(umi, case):
    # seeded fuzz over the next rows: random window, shape, kinds, parameters; odd cases through the
    # time-stamped path (compacted rows, jittered times, grid shorter than the data)
    import torch
    rng = np.random.default_rng(9100 + case)
    W = int(rng.choice([5, 9, 25, 33, 49, 51, 101, 217, 361, 801])) | 1
    S = int(rng.choice([1, 3, 40, 180]))
    N = int(rng.integers(2, 2200))
    alpha = float(rng.choice([1.0, 2.0, 3.0]))
    n_iter = int(rng.choice([0, 1, 5]))
    x = lc.random_series(9200 + case, S, N, nan_frac=float(rng.choice([0.0, 0.03, 0.15])), inf_frac=0.0)
    if case % 2 == 0:
        sk, wk = int(rng.integers(0, 2)), int(rng.integers(0, 2))
        _family_case(umi, x, W, sk, wk, alpha=alpha, n_iter=n_iter)
    else:
        dt = float(rng.choice([2.0 / 1440, 0.02, 1.0]))
        t0 = float(rng.choice([0.0, 2457000.5, -3.25]))
        t, f, slot = lc.compact(x, dt, t0=t0, jitter=float(rng.choice([0.0, 0.25, 0.45])), seed=case)
        n_grid = max(0, N - int(rng.integers(0, 5)))
        ref = orc.gapped(t, f, t0, dt, n_grid, W, alpha=alpha, n_iter=n_iter)
        trend, flat = umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), t0, dt, n_grid, W,
                                             alpha=alpha, n_iter=n_iter, flat=True)
        torch.cuda.synchronize()
        if n_iter == 0:
            parity.compare_median(trend.cpu().numpy(), ref.median)
        else:
            parity.compare_trend(trend.cpu().numpy(), ref)
        _check_flat(flat.cpu().numpy(), f, ref)


def test_flatten_host_driver(umi):
    # host buffers in, (trend, flat) back through the streamed batch driver; and flat only
    cfg = lc.CONFIGS[5]
    flux = lc.stars(5, range(40))
    ref = orc.detrend(flux, cfg.W, alpha=3.0, c=2.5)
    trend, flat = umi.umi_flatten_host(None, flux, cfg.W, alpha=3.0, c=2.5, stars_per_batch=7, n_streams=3)
    parity.compare_trend(trend, ref)
    _check_flat(flat, flux, ref)
    none, flat2 = umi.umi_flatten_host(None, flux, cfg.W, alpha=3.0, c=2.5, want_trend=False)
    # other batch size -> the other variant of the reweighting kernel (split-window vs throughput): same
    # arithmetic, another summation order, so equal to rounding, not bit for bit
    assert none is None and np.allclose(flat2, flat, rtol=2e-6, atol=0.0, equal_nan=True)


def test_hundred_random_cases_of_the_next_rows(umi):
    # sibling estimators and gap handling (plain and with segments) on random windows, shapes, gap structures and options
    import torch
    for case in range(100):
        rng = np.random.default_rng(55000 + case)
        W = int(rng.choice([5, 9, 25, 33, 49, 51, 101, 217, 361, 801])) | 1
        S = int(rng.choice([1, 3, 40, 180]))
        N = int(rng.integers(2, 2600))
        alpha = float(rng.choice([1.0, 2.0, 3.0]))
        n_iter = int(rng.choice([0, 1, 5]))
        x = lc.random_series(56000 + case, S, N, nan_frac=float(rng.choice([0.0, 0.03, 0.15])), inf_frac=0.0,
                             ties=bool(rng.integers(0, 3) == 0))
        kind = int(rng.integers(0, 3))
        if kind == 0:
            _family_case(umi, x, W, int(rng.integers(0, 2)), int(rng.integers(0, 2)), alpha=alpha, n_iter=n_iter)
            continue
        dt = float(rng.choice([2.0 / 1440, 0.02, 1.0]))
        tz = float(rng.choice([0.0, 2457000.5, -3.25]))
        for b in range(S):
            for _ in range(int(rng.integers(0, 4))):
                if N > 50:
                    a = int(rng.integers(0, N - 10))
                    x[b, a:a + int(rng.integers(1, max(2, N // 4)))] = np.nan
        t, f, slot = lc.compact(x, dt, t0=tz, jitter=float(rng.choice([0.0, 0.25, 0.45])), seed=case)
        n_grid = max(0, N - int(rng.integers(0, 5)))
        h = W // 2
        seg = {} if kind == 1 else dict(break_slots=int(rng.choice([-1, h, h + 3, W - 1, 3 * W])),
                                        min_segment=int(rng.choice([0, 1, W // 3, W])),
                                        edge_cut=int(rng.choice([0, 1, W // 10 + 1, W])))
        ref = orc.gapped_ex(t, f, tz, dt, n_grid, W, alpha=alpha, n_iter=n_iter, **seg)
        trend, flat = umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), tz, dt, n_grid, W, alpha=alpha,
                                             n_iter=n_iter, flat=True, **seg)
        torch.cuda.synchronize()
        if n_iter == 0:
            parity.compare_median(trend.cpu().numpy(), ref.median)
        else:
            parity.compare_trend(trend.cpu().numpy(), ref)
        _check_flat(flat.cpu().numpy(), f, ref)


def test_gapped_segments_rows_that_leave_whole_parts_empty(umi):
    # The segment scan of small batches runs one CTA per row, every warp one part of the row (umi_regrid.cu): rows whose
    # valid slots sit in one part only, at the part seams, nowhere, or everywhere; breaks exactly at / next to the limit.
    import torch
    dt, N, W = 0.01, 8000, 25                               # 250 chunks of 32 slots: parts of 32 chunks = 1024 slots
    rng = np.random.default_rng(5)
    grid = np.full((10, N), np.nan, np.float32)
    val = (1.0 + 1e-3 * rng.standard_normal(N)).astype(np.float32)
    grid[1, 4000] = val[4000]                               # one valid slot
    grid[2, 0] = val[0]; grid[2, N - 1] = val[N - 1]        # the two ends of the row
    grid[3, 1000:1048] = val[1000:1048]                     # across the seam of parts 0 and 1 (slot 1024)
    grid[4, 900:1024] = val[900:1024]; grid[4, 1024 + 13:1200] = val[1024 + 13:1200]     # a break of 13 empty slots exactly at a seam
    grid[5, 900:1024] = val[900:1024]; grid[5, 1024 + 12:1200] = val[1024 + 12:1200]     # 12: not a break
    grid[6] = val                                           # one segment over all parts
    grid[7, 100:300] = val[100:300]; grid[7, 7000:7300] = val[7000:7300]                 # parts 1 .. 5 empty
    grid[8] = val; grid[8, 1023::1024] = np.nan; grid[8, 2040:2060] = np.nan             # holes at the seams, a break next to one
    grid[9, ::40] = val[::40]                               # every valid slot a segment of its own (gaps of 39 > 12)
    t, f, slot = lc.compact(grid, dt, t0=3.5, jitter=0.0, seed=1)
    for brk, mseg, ecut in ((12, 0, 0), (12, 30, 4), (40, 2, 1), (-1, 0, 10)):
        ref = orc.gapped_ex(t, f, 3.5, dt, N, W, break_slots=brk, min_segment=mseg, edge_cut=ecut)
        got = umi.umi_detrend_gapped(_cuda(t, np.float64), _cuda(f, np.float32), 3.5, dt, N, W,
                                     break_slots=brk, min_segment=mseg, edge_cut=ecut)
        torch.cuda.synchronize()
        parity.compare_trend(got.cpu().numpy(), ref)


def test_gapped_segments_warp_per_row_and_cta_per_row_scans_agree(umi):
    # 4,200 rows take the warp-per-row scan, the same rows 100 at a time the CTA-per-row scan: identical results, and the oracle's
    import torch
    dt, N, W = 2.0 / 1440, 1301, 25
    t, f, slot = _segment_rows(77, 4200, N, dt)
    kw = dict(break_slots=12, min_segment=12, edge_cut=3)
    td, fd = _cuda(t, np.float64), _cuda(f, np.float32)
    big = umi.umi_detrend_gapped(td, fd, 7.25, dt, N, W, **kw).cpu().numpy()
    for a in (0, 2100, 4100):
        small = umi.umi_detrend_gapped(td[a:a + 100].contiguous(), fd[a:a + 100].contiguous(), 7.25, dt, N, W, **kw).cpu().numpy()
        np.testing.assert_array_equal(small, big[a:a + 100])
    ref = orc.gapped_ex(t[:150], f[:150], 7.25, dt, N, W, **kw)
    parity.compare_trend(big[:150], ref)
