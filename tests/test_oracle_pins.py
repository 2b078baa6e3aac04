"""Pins for the fp64 oracle (oracle/umi_oracle.c) against things other than itself:
paper-printed values, a hand-computed worked example, an independent numpy brute
force, numpy/scipy library routines, Gaussian closed forms and invariants.
All CPU (-m "not gpu").  Citations are /root/reference/PAPER.md lines.
"""
import itertools
import math
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.ndimage
import scipy.stats

from oracle import brute
from oracle import umi_oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows


# ---------------------------------------------------------------- paper-printed values
def test_paper_printed_values():
    for row in _read_golden("paper_values.txt"):
        kind = row[0]
        if kind == "window_len":
            minutes, W = float(row[1]), int(row[2])
            assert orc.window_len(minutes / 1440.0) == W
        elif kind == "window_days":
            minutes, days, tol = float(row[1]), float(row[2]), float(row[3])
            W = orc.window_len(minutes / 1440.0)
            assert abs(W * minutes / 1440.0 - days) <= tol
        elif kind == "weight":
            u, alpha, w, tol = map(float, row[1:5])
            assert abs(orc.weight(u, alpha) - w) <= tol
        elif kind == "dip_u":
            # a 1-sigma dip in Gaussian noise: |u| = sigma / (c * 0.6745 * sigma_upper), sigma_upper -> sigma
            c, u, tol = map(float, row[1:4])
            rng = np.random.default_rng(5)
            x = rng.normal(1.0, 1e-3, 200001).astype(np.float32)
            r = orc.positions(x, [0], [100000], W=200001, n_iter=0)
            assert abs(1e-3 / (c * r.scale[0]) - u) <= tol
        else:
            raise AssertionError("unknown golden row %r" % row)


def test_window_len_configs_and_guard():
    # BASELINE.json configs: 2 min, 29.4 min, 20 s, 200 s
    assert orc.window_len(2.0 / 1440) == 361
    assert orc.window_len(29.4 / 1440) == 25
    assert orc.window_len(20.0 / 86400) == 2161
    assert orc.window_len(200.0 / 86400) == 217
    # (R15) a cadence that passed through fp32 must not drop to 359 / 215
    assert orc.window_len(float(np.float32(2.0 / 1440))) == 361
    assert orc.window_len(float(np.float32(200.0 / 86400))) == 217
    # always odd, >= 1; bad input -> 0
    for dt in [0.3, 0.25, 0.1, 1.0, 7.3e-4, 0.0123]:
        W = orc.window_len(dt)
        assert W % 2 == 1 and W >= 1
        assert W in (math.floor(0.5 / dt) | 1, math.floor(0.5 / dt * (1 + 2 ** -20)) | 1)
    for bad in [0.0, -1.0, float("nan"), float("inf")]:
        assert orc.window_len(bad) == 0


def test_weight_function_shape():
    # Eq. 3: zero at and beyond |u_eff| = 1; Eq. 2: the cut-off on the low side is at -1/alpha
    for alpha in [1.0, 2.0, 3.0, 10.0]:
        assert orc.weight(0.0, alpha) == 1.0
        assert orc.weight(1.0, alpha) == 0.0
        assert orc.weight(1.5, alpha) == 0.0
        assert orc.weight(-1.0 / alpha, alpha) == 0.0
        assert orc.weight(-1.0 / alpha + 1e-9, alpha) > 0.0
        assert orc.weight(0.5, alpha) == pytest.approx((1 - 0.25) ** 2)
        assert orc.weight(-0.5 / alpha, alpha) == pytest.approx((1 - 0.25) ** 2)


# ---------------------------------------------------------------- worked example (hand-checkable)
def test_worked_example_golden():
    g = {k: float(v) for k, v in _read_golden("worked_example.txt")}
    x = np.array([0, 1, 2, 3, 4], dtype=np.float32)
    # hand-computed in tests/golden/make_golden.py's docstring
    assert g["median"] == 2.0
    assert g["scale"] == pytest.approx(0.6745 * math.sqrt(2.5), rel=1e-15)
    assert g["alpha2_pass1"] == pytest.approx(2.3575634, abs=2e-7)
    for k in range(1, 6):
        r = orc.positions(x, [0], [2], W=5, alpha=2.0, n_iter=k)
        assert r.median[0] == 2.0
        assert r.scale[0] == pytest.approx(g["scale"], rel=1e-14)
        assert r.trend64[0] == pytest.approx(g["alpha2_pass%d" % k], rel=1e-14)
        r1 = orc.positions(x, [0], [2], W=5, alpha=1.0, n_iter=k)
        assert r1.trend64[0] == pytest.approx(2.0, abs=1e-14)   # symmetric data, symmetric weights


# ---------------------------------------------------------------- brute force on tiny inputs
@pytest.mark.parametrize("W", [3, 5, 9, 15])
def test_brute_force_with_all_nan_placements(W):
    rng = np.random.default_rng(100 + W)
    N = 7
    base = (1.0 + 0.01 * rng.standard_normal(N)).astype(np.float32)
    base[2] = base[4]                                   # a tie
    for mask in itertools.product([0, 1], repeat=N):
        x = base.copy()
        x[np.array(mask, bool)] = np.nan
        for alpha, n_iter in [(2.0, 5), (1.0, 3), (3.0, 0)]:
            o = orc.detrend(x, W, alpha=alpha, n_iter=n_iter)
            t, m, s = brute.detrend(x, W, alpha=alpha, n_iter=n_iter)
            np.testing.assert_array_equal(np.isnan(o.trend64), np.isnan(t))
            ok = ~np.isnan(t)
            np.testing.assert_array_equal(o.median[ok].astype(np.float64), m[ok])
            np.testing.assert_allclose(o.scale[ok], s[ok], rtol=1e-13, atol=0)
            np.testing.assert_allclose(o.trend64[ok], t[ok], rtol=1e-13, atol=0)


def test_brute_force_random_series_with_gaps_time_and_inf():
    rng = np.random.default_rng(7)
    S, N = 3, 120
    flux = (1.0 + 0.002 * rng.standard_normal((S, N))).astype(np.float32)
    flux[0, 30:45] = np.nan
    flux[1, 5] = np.inf
    flux[1, 77] = -np.inf                              # (R16) +-Inf are invalid too
    flux[2, 60:70] -= 0.02                             # a dip
    time = np.tile(np.arange(N) * 0.02, (S, 1))
    time[2, 100:104] = np.nan                          # non-finite time marks the slot invalid
    for W, alpha, c in [(11, 2.0, 5.0), (25, 3.0, 5.0), (25, 10.0, 2.5), (151, 2.0, 5.0)]:
        o = orc.detrend(flux, W, alpha=alpha, c=c, n_iter=5, time=time)
        t, m, s = brute.detrend(flux, W, alpha=alpha, c=c, n_iter=5, time=time)
        np.testing.assert_array_equal(np.isnan(o.trend64), np.isnan(t))
        ok = ~np.isnan(t)
        assert ok.sum() > 0
        np.testing.assert_array_equal(o.median[ok].astype(np.float64), m[ok])
        np.testing.assert_allclose(o.trend64[ok], t[ok], rtol=1e-12)
        np.testing.assert_array_equal(o.trend32, o.trend64.astype(np.float32))
    # own slot invalid -> NaN (R5); W > N is legal (window clipped)
    o = orc.detrend(flux, 151, time=time)
    assert np.isnan(o.trend64[0, 30:45]).all() and np.isnan(o.trend64[2, 100:104]).all()
    assert np.isfinite(o.trend64[0, 0])


def test_positions_equals_full():
    rng = np.random.default_rng(3)
    flux = (1 + 1e-3 * rng.standard_normal((4, 300))).astype(np.float32)
    flux[1, 100:140] = np.nan
    full = orc.detrend(flux, 31)
    b = rng.integers(0, 4, 200)
    i = rng.integers(0, 300, 200)
    sub = orc.positions(flux, b, i, 31)
    np.testing.assert_array_equal(sub.trend64, full.trend64[b, i])
    np.testing.assert_array_equal(sub.median, full.median[b, i])
    np.testing.assert_array_equal(sub.n_valid, full.n_valid[b, i])


# ---------------------------------------------------------------- library routines
def test_median_equals_library_median_filter():
    # quickselect median == sort median.  n_iter = 0 returns Phase 1.
    rng = np.random.default_rng(11)
    x = rng.standard_normal(500).astype(np.float32)
    x[::7] = x[3]                                       # many ties
    for W in [3, 25, 101]:
        h = W // 2
        o = orc.detrend(x, W, n_iter=0)
        ref = scipy.ndimage.median_filter(x, size=W, mode="nearest")
        np.testing.assert_array_equal(o.trend32[0, h:-h], ref[h:-h])
        sw = np.lib.stride_tricks.sliding_window_view(x, W)
        np.testing.assert_array_equal(o.median[0, h:-h], np.median(sw, axis=1).astype(np.float32))
    # with gaps and an odd number of valid samples nanmedian agrees; with an even number the
    # oracle returns the LOWER middle sample (R6), nanmedian the mean of the two
    y = x.copy()
    y[100:103] = np.nan
    o = orc.detrend(y, 25, n_iter=0, min_valid=1)
    sw = np.lib.stride_tricks.sliding_window_view(y, 25)
    nv = np.isfinite(sw).sum(axis=1)
    nm = np.nanmedian(sw, axis=1)
    own = np.isfinite(y[12:-12])
    odd = (nv % 2 == 1) & own
    np.testing.assert_array_equal(o.median[0, 12:-12][odd], nm[odd].astype(np.float32))
    even = (nv % 2 == 0) & own
    assert even.any()
    lower = np.array([np.sort(w[np.isfinite(w)])[(np.isfinite(w).sum() - 1) // 2] for w in sw[even]])
    np.testing.assert_array_equal(o.median[0, 12:-12][even], lower.astype(np.float32))
    assert (o.median[0, 12:-12][even] <= nm[even]).all()


def test_c_to_infinity_gives_windowed_mean():
    # with c huge every weight is 1 and one pass of Eq. 4 is the plain mean of the valid samples
    rng = np.random.default_rng(13)
    x = (5.0 + rng.standard_normal(400)).astype(np.float32)
    x[50:60] = np.nan
    W = 41
    o = orc.detrend(x, W, alpha=2.0, c=1e9, n_iter=1)
    for i in [0, 3, 20, 45, 64, 200, 380, 399]:
        lo, hi = max(0, i - 20), min(400, i + 21)
        ref = np.nanmean(x[lo:hi].astype(np.float64))
        assert o.trend64[0, i] == pytest.approx(ref, rel=1e-12)
    assert np.isnan(o.trend64[0, 55])


def test_min_valid_rule():
    # minimum length W/3 (R4): fewer valid samples -> NaN
    x = np.full(100, np.nan, dtype=np.float32)
    x[40:48] = 1.0 + 0.01 * np.arange(8)               # 8 valid samples; W = 25 -> m_min = 8
    o = orc.detrend(x, 25)
    assert np.isfinite(o.trend64[0, 40:48]).all()       # every window around them holds all 8
    x[47] = np.nan                                      # 7 < 8
    o = orc.detrend(x, 25)
    assert np.isnan(o.trend64).all()
    o = orc.detrend(x, 25, min_valid=7)
    assert np.isfinite(o.trend64[0, 40:47]).all()
    assert (o.n_valid[0, 40:47] == 7).all()


# ---------------------------------------------------------------- Gaussian closed forms
def test_sigma_upper_tends_to_sigma():
    # E[(x-m)^2 | x>m] = sigma^2 for a Gaussian, so s -> 0.6745 sigma
    rng = np.random.default_rng(17)
    sigma = 3e-3
    x = rng.normal(2.0, sigma, 100001).astype(np.float32)
    r = orc.positions(x, [0], [50000], W=100001, n_iter=0)
    assert r.scale[0] / (0.6745 * sigma) == pytest.approx(1.0, abs=0.01)
    assert r.n_plus[0] == int(np.sum(x > np.median(x)))     # strict (R7): ties are not counted
    assert 49990 <= r.n_plus[0] <= 50000


def _population_offset(alpha, c, n_iter=5):
    """Eq. 2-4 applied to the N(0,1) population itself: median 0, sigma_upper 1."""
    cs = c * 0.6745
    pdf = scipy.stats.norm.pdf
    mu = 0.0
    for _ in range(n_iter):
        lo, hi = mu - cs / alpha, mu + cs

        def w(x):
            u = (x - mu) / cs
            ue = alpha * u if u < 0 else u
            return (1 - ue * ue) ** 2

        num = scipy.integrate.quad(lambda x: w(x) * x * pdf(x), lo, hi, points=[mu])[0]
        den = scipy.integrate.quad(lambda x: w(x) * pdf(x), lo, hi, points=[mu])[0]
        mu = num / den
    return mu


@pytest.mark.parametrize("alpha,c", [(1.0, 5.0), (2.0, 5.0), (3.0, 5.0), (10.0, 2.5)])
def test_gaussian_noise_offset_matches_population_integral(alpha, c):
    # a constant offset on flat stars, growing with alpha; ~0 at alpha = 1.
    # The detrended flux is biased low (paper: -451 ppm), i.e. the trend sits ABOVE the truth.
    expect = _population_offset(alpha, c)
    rng = np.random.default_rng(23)
    sigma = 1e-3
    x = (1.0 + sigma * rng.standard_normal((8, 3000))).astype(np.float32)
    o = orc.detrend(x, 361, alpha=alpha, c=c, n_iter=5)
    off = np.mean(o.trend64[:, 200:-200] - 1.0) / sigma
    assert off == pytest.approx(expect, abs=0.03)
    if alpha == 1.0:
        assert abs(expect) < 1e-9
    else:
        assert expect > 0.3


def test_paper_bias_ratios_consistent_with_population_integral():
    # -1857 ppm at (alpha=10, c=2.5) vs -451 ppm at (alpha=2, c=5): ratio 4.1
    ratio = _population_offset(10.0, 2.5) / _population_offset(2.0, 5.0)
    assert ratio == pytest.approx(1857.0 / 451.0, rel=0.05)


# ---------------------------------------------------------------- invariants
def _series(seed, n=400, nan=True):
    rng = np.random.default_rng(seed)
    t = np.arange(n)
    x = 1.0 + 0.003 * np.sin(t / 37.0) + 0.001 * rng.standard_normal(n)
    x[n * 3 // 10:n * 3 // 10 + 10] -= 0.01
    x[n * 3 // 4] += 0.02
    x = x.astype(np.float32)
    if nan:
        x[n // 2:n // 2 + 15] = np.nan
    return x


def test_constant_series_returns_itself():
    x = np.full(300, 1.2345678, dtype=np.float32)
    x[100:110] = np.nan
    o = orc.detrend(x, 51)
    ok = np.isfinite(x)
    np.testing.assert_array_equal(o.trend32[0, ok], x[ok])
    assert np.isnan(o.trend32[0, ~ok]).all()


def test_affine_equivariance_positive_scale_only():
    x = _series(1)
    x = (np.round(x.astype(np.float64) * 2 ** 20) / 2 ** 20).astype(np.float32)   # on a 2^-20 grid
    o = orc.detrend(x, 51)
    # exact for a power-of-two factor
    o2 = orc.detrend(x * np.float32(4.0), 51)
    np.testing.assert_array_equal(o2.trend64, 4.0 * o.trend64)
    # k > 0, offset: to rounding (inputs are re-rounded to fp32, so compare on fp64-exact inputs)
    y64 = x.astype(np.float64) * 0.5 + 0.25
    y = y64.astype(np.float32)                          # multiples of 2^-21 below 1: exact in fp32
    assert np.array_equal(y.astype(np.float64)[np.isfinite(y64)], y64[np.isfinite(y64)])
    o3 = orc.detrend(y, 51)
    np.testing.assert_allclose(o3.trend64, 0.5 * o.trend64 + 0.25, rtol=1e-12, equal_nan=True)
    # k < 0 is NOT an equivariance, not even at alpha = 1 (one-sided scale)
    o4 = orc.detrend(-x, 51, alpha=1.0)
    o5 = orc.detrend(x, 51, alpha=1.0)
    ok = np.isfinite(o4.trend64)
    assert np.max(np.abs(o4.trend64[ok] + o5.trend64[ok])) > 1e-6


def test_reversal_and_permutation():
    x = _series(2)
    o = orc.detrend(x, 51)
    orv = orc.detrend(x[::-1].copy(), 51)
    np.testing.assert_allclose(orv.trend64[0, ::-1], o.trend64[0], rtol=1e-13, equal_nan=True)
    np.testing.assert_array_equal(orv.median[0, ::-1], o.median[0])
    # permuting the samples of one full-length window leaves its result unchanged (to summation order)
    y = _series(3, n=101, nan=False)
    a = orc.positions(y, [0], [50], W=101)
    rng = np.random.default_rng(0)
    yp = y.copy()
    rng.shuffle(yp)
    b = orc.positions(yp, [0], [50], W=101)
    assert a.median[0] == b.median[0]
    assert b.scale[0] == pytest.approx(a.scale[0], rel=1e-13)
    assert b.trend64[0] == pytest.approx(a.trend64[0], rel=1e-13)


def test_deepening_below_median_leaves_scale_unchanged():
    # "transit dips (below the median) never contribute to the scale estimate" (G2)
    y = _series(4, n=201, nan=False)
    a = orc.positions(y, [0], [100], W=201, n_iter=0)
    z = y.copy()
    below = np.where(z < a.median[0])[0]
    z[below[::2]] -= np.float32(1000.0)                 # arbitrarily deep
    z[below[1::2]] -= np.float32(0.5)
    b = orc.positions(z, [0], [100], W=201, n_iter=0)
    assert b.median[0] == a.median[0]
    assert b.n_plus[0] == a.n_plus[0]
    assert b.scale[0] == a.scale[0]                     # bit-identical


def test_redescending_zero_weight_points_can_move():
    y = _series(5, n=201, nan=False)
    y[10] = 5.0                                         # far above: weight 0 in every pass
    y[20] = -3.0                                        # far below
    a = orc.positions(y, [0], [100], W=201)
    z = y.copy()
    z[20] = -3000.0
    b = orc.positions(z, [0], [100], W=201)
    assert b.trend64[0] == a.trend64[0]
    # the upward outlier enters the one-sided scale, so moving it changes s - but shrinking the
    # scale only pushes it further past the cut-off; check the weight is zero instead
    u = (5.0 - a.trend64[0]) / (5.0 * a.scale[0])
    assert u > 1.0 and orc.weight(u, 2.0) == 0.0


def test_alpha_one_is_symmetric_biweight():
    # alpha = 1 recovers the standard symmetric biweight (with the upper-RMS scale)
    y = _series(6, n=151, nan=False).astype(np.float64)
    a = orc.positions(y.astype(np.float32), [0], [75], W=151, alpha=1.0, n_iter=7)
    y = y.astype(np.float32).astype(np.float64)
    med = np.median(y)
    s = 0.6745 * np.sqrt(np.mean((y[y > med] - med) ** 2))
    mu = med
    for _ in range(7):                                  # textbook Tukey biweight location step
        u = (y - mu) / (5.0 * s)
        w = np.where(np.abs(u) < 1, (1 - u * u) ** 2, 0.0)
        mu = np.sum(w * y) / np.sum(w)
    assert a.trend64[0] == pytest.approx(mu, rel=1e-13)


def test_fixed_point_of_estimating_equation():
    y = _series(7, n=361, nan=False)
    a = orc.positions(y, [0], [180], W=361, n_iter=200)
    mu, s = a.trend64[0], a.scale[0]
    yd = y.astype(np.float64)
    w = brute.bisquare_weights((yd - mu) / (5.0 * s), 2.0)
    assert abs(np.sum(w * (yd - mu))) / np.sum(w) < 1e-12


def test_breakdown_forty_percent_dip():
    # breakdown point exceeding 40% for contamination beyond 3 sigma
    rng = np.random.default_rng(31)
    sigma = 1e-3
    base = 1.0 + sigma * rng.standard_normal(361)
    clean = orc.positions(base.astype(np.float32), [0], [180], W=361).trend64[0]
    for depth in [5e-3, 5e-2, 10.0]:
        y = base.copy()
        y[100:100 + 144] -= depth                      # 40 % of the window
        t = orc.positions(y.astype(np.float32), [0], [180], W=361).trend64[0]
        assert abs(t - clean) < 1.0 * sigma


def test_near_cutoff_flag():
    # the flag marks windows where some |u_eff| lies within tol of 1
    x = np.array([0, 1, 2, 3, 4], dtype=np.float32)
    r = orc.positions(x, [0], [2], W=5, cutoff_tol=1e-5)
    assert r.near_cutoff[0] == 0
    r = orc.positions(x, [0], [2], W=5, cutoff_tol=0.3)   # pass-1 u_eff = -0.75 is within 0.3 of -1
    assert r.near_cutoff[0] == 1


# ---------------------------------------------------------------- next rows: F1 normalisation, F2 gap handling
def test_normalize_is_flux_over_trend():
    # PAPER.md:155 "normalization": flat * trend = flux; a constant series flattens to exactly 1
    from workloads import lightcurves as lc
    x = lc.random_series(3, 2, 400)
    r = orc.detrend(x, 25)
    flat = orc.normalize(x, r.trend64)
    ok = ~np.isnan(r.trend64)
    assert np.array_equal(np.isnan(flat), ~ok | np.isnan(x))
    np.testing.assert_allclose(flat[ok] * r.trend64[ok], x[ok].astype(np.float64), rtol=4e-16)
    cst = np.full((1, 300), 0.75, np.float32)
    assert np.array_equal(orc.normalize(cst, orc.detrend(cst, 9).trend64), np.ones((1, 300)))


@pytest.mark.parametrize("W,jitter", [(5, 0.0), (25, 0.3), (51, 0.45)])
def test_gapped_equals_base_oracle_on_the_nan_filled_grid(W, jitter):
    # R20: removing the invalid slots and giving real time stamps must not change anything:
    # the base oracle on the uniform NaN-filled grid (pinned above) fixes every value.
    from workloads import lightcurves as lc
    dt = 2.0 / 1440
    grid = lc.random_series(40 + W, 3, 900, nan_frac=0.04, inf_frac=0.0)
    grid[1, 300:420] = np.nan                         # a gap wider than the window
    t, f, slot = lc.compact(grid, dt, t0=1234.5, jitter=jitter, seed=W)
    base = orc.detrend(grid, W)
    got = orc.gapped(t, f, 1234.5, dt, grid.shape[1], W)
    for b in range(grid.shape[0]):
        m = slot[b] >= 0
        np.testing.assert_array_equal(got.trend64[b, m], base.trend64[b, slot[b, m]])
        np.testing.assert_array_equal(got.median[b, m], base.median[b, slot[b, m]])
        np.testing.assert_array_equal(got.n_valid[b, m], base.n_valid[b, slot[b, m]])
        assert np.isnan(got.trend64[b, ~m]).all()     # padding (NaN time) -> NaN


def test_gapped_brute_force_out_of_range_and_colliding_slots():
    from workloads import lightcurves as lc
    dt = 0.02
    grid = lc.random_series(77, 2, 260, nan_frac=0.05, inf_frac=0.0)
    t, f, slot = lc.compact(grid, dt, t0=10.0, jitter=0.2, seed=1)
    t[0, 50] = t[0, 51] - 1e-9 * dt                   # two samples in one slot: the first is dropped
    t[1, 5] = np.inf
    f[1, 9] = np.nan
    n_grid = 240                                      # slots >= 240 fall outside the grid
    for W, mv in ((7, -1), (31, 3)):
        got = orc.gapped(t, f, 10.0, dt, n_grid, W, min_valid=mv)
        bt, bm = brute.detrend_gapped(t, f, 10.0, dt, n_grid, W, min_valid=None if mv < 0 else mv)
        assert np.array_equal(np.isnan(got.trend64), np.isnan(bt))
        ok = ~np.isnan(bt)
        np.testing.assert_allclose(got.trend64[ok], bt[ok], rtol=1e-13)
        np.testing.assert_array_equal(got.median[ok].astype(np.float64), bm[ok])
        assert np.isnan(got.trend64[0, 50]) and not np.isnan(got.trend64[0, 51])
        for b in range(2):
            assert np.isnan(got.trend64[b, slot[b] >= n_grid]).all()


def test_gapped_on_uniform_times_is_the_positional_window():
    from workloads import lightcurves as lc
    x = lc.random_series(9, 2, 500, nan_frac=0.0, inf_frac=0.0)
    t = np.tile(5.0 + np.arange(500) * 0.01, (2, 1))
    a = orc.gapped(t, x, 5.0, 0.01, 500, 21)
    b = orc.detrend(x, 21)
    np.testing.assert_array_equal(a.trend64, b.trend64)


# ---------------------------------------------------------------- next row F4: sibling estimators (MAD scale, Welsch weights)
def test_family_default_is_the_paper_estimator():
    from workloads import lightcurves as lc
    x = lc.random_series(12, 2, 600)
    a, b = orc.family(x, 25, 0, 0), orc.detrend(x, 25)
    np.testing.assert_array_equal(a.trend64, b.trend64)
    np.testing.assert_array_equal(a.scale, b.scale)


def test_mad_scale_library_routine_and_gaussian_constant():
    # n_iter = 0 leaves (median, s); the MAD of an odd gap-free window is scipy's routine
    rng = np.random.default_rng(11)
    x = rng.normal(1.0, 2e-3, (1, 801)).astype(np.float32)
    r = orc.family(x, 51, orc.SCALE_MAD, 0, n_iter=0)
    for i in (25, 26, 400, 775):
        win = x[0, i - 25:i + 26].astype(np.float64)
        assert r.scale[0, i] == scipy.stats.median_abs_deviation(win)
    # 0.6745 sigma is "the MAD convention at the Gaussian model"
    big = rng.normal(0.0, 1.0, 200001).astype(np.float32)
    rr = orc.family(big[None, 99000:101001].copy(), 2001, orc.SCALE_MAD, 0, n_iter=0)
    full = orc.positions(big, [0], [100000], W=200001, n_iter=0)        # reference sigma_upper ~ 1
    mad = np.sort(np.abs(big.astype(np.float64) - np.median(big)))[100000]
    assert abs(mad - scipy.stats.norm.ppf(0.75)) < 0.01 and abs(0.6745 - scipy.stats.norm.ppf(0.75)) < 1e-4
    assert abs(full.scale[0] / 0.6745 - 1.0) < 0.01 and np.isfinite(rr.scale[0, 1000])


@pytest.mark.parametrize("sk,wk", [(0, 1), (1, 0), (1, 1)])
def test_family_brute_force_with_gaps(sk, wk):
    from workloads import lightcurves as lc
    x = lc.random_series(90 + sk * 2 + wk, 2, 160, nan_frac=0.08, inf_frac=0.02)
    for W, alpha in ((7, 2.0), (15, 1.0), (31, 3.0)):
        r = orc.family(x, W, sk, wk, alpha=alpha)
        h = (W - 1) // 2
        for b in range(2):
            for i in range(160):
                win = brute.window_samples(x[b], i, W)
                if not np.isfinite(x[b, i]) or win.size < max(1, W // 3):
                    assert np.isnan(r.trend64[b, i])
                    continue
                mu, med, s = brute.location_family(win, "mad" if sk else "upper_rms",
                                                   "welsch" if wk else "bisquare", alpha=alpha)
                assert r.median[b, i] == np.float32(med)
                assert r.scale[b, i] == pytest.approx(s, rel=1e-13, abs=0.0)
                assert r.trend64[b, i] == pytest.approx(mu, rel=1e-12)


def test_welsch_worked_example_and_limits():
    # x = {0,1,2,3,4}, MAD scale: median 2, deviations {2,1,0,1,2} -> MAD = 1; c = 5, alpha = 2:
    # u = (x-2)/5, u_eff = {-.8,-.4,0,.2,.4}, w = exp(-u_eff^2); one pass by hand
    x = np.array([[0, 1, 2, 3, 4]], np.float32)
    w = [math.exp(-0.64), math.exp(-0.16), 1.0, math.exp(-0.04), math.exp(-0.16)]
    mu1 = sum(wi * xi for wi, xi in zip(w, range(5))) / sum(w)
    r = orc.family(x, 5, orc.SCALE_MAD, orc.WEIGHT_WELSCH, alpha=2.0, n_iter=1, min_valid=5)
    assert r.scale[0, 2] == 1.0 and r.median[0, 2] == 2.0
    assert r.trend64[0, 2] == pytest.approx(mu1, rel=1e-15) and abs(mu1 - 2.180888) < 1e-6
    # symmetric data, alpha = 1: the location stays at the centre for both weights and both scales
    for sk in (0, 1):
        for wk in (0, 1):
            assert orc.family(x, 5, sk, wk, alpha=1.0, min_valid=5).trend64[0, 2] == pytest.approx(2.0, abs=1e-15)
    # c -> infinity: every weight -> 1, one pass gives the window mean
    rng = np.random.default_rng(3)
    y = rng.normal(1.0, 1e-2, (1, 41)).astype(np.float32)
    big = orc.family(y, 41, orc.SCALE_MAD, orc.WEIGHT_WELSCH, c=1e9, n_iter=1)
    assert big.trend64[0, 20] == pytest.approx(y.astype(np.float64).mean(), rel=1e-12)


def test_mad_biweight_invariants():
    rng = np.random.default_rng(8)
    x = (1.0 + 1e-3 * rng.standard_normal((1, 400))).astype(np.float32)
    for wk in (0, 1):
        r = orc.family(x, 41, orc.SCALE_MAD, wk, alpha=1.0)
        # two-sided scale + symmetric weights: reflection equivariance on interior odd windows
        m = orc.family((-x).astype(np.float32), 41, orc.SCALE_MAD, wk, alpha=1.0)
        np.testing.assert_allclose(m.trend64[0, 20:-20], -r.trend64[0, 20:-20], rtol=1e-13)
        # positive affine map (power of two: exact)
        a = orc.family((4.0 * x).astype(np.float32), 41, orc.SCALE_MAD, wk, alpha=1.0)
        np.testing.assert_array_equal(a.trend64, 4.0 * r.trend64)
        # fixed point of the estimating equation after many passes
        f = orc.family(x, 41, orc.SCALE_MAD, wk, alpha=1.0, n_iter=300)
        i = 200
        win = x[0, i - 20:i + 21].astype(np.float64)
        u = (win - f.trend64[0, i]) / (5.0 * f.scale[0, i])
        wgt = np.exp(-u ** 2) if wk else brute.bisquare_weights(u, 1.0)
        assert abs(np.sum(wgt * (win - f.trend64[0, i]))) < 1e-12
    cst = np.full((1, 100), 2.5, np.float32)
    assert np.array_equal(orc.family(cst, 9, orc.SCALE_MAD, orc.WEIGHT_WELSCH).trend64, cst.astype(np.float64))


def test_mad_is_inflated_by_a_deep_dip_but_upper_rms_is_not():
    # "deep transits can inflate the [MAD] scale"; the upper-RMS never sees them
    rng = np.random.default_rng(21)
    x = (1.0 + 1e-3 * rng.standard_normal(201)).astype(np.float32)
    y = x.copy()
    lows = np.argsort(x)[:80]                      # 40 % of the window, all below the median
    y[lows] -= 0.05
    a0, a1 = (orc.family(v[None, :], 201, orc.SCALE_UPPER_RMS, 0, n_iter=0).scale[0, 100] for v in (x, y))
    m0, m1 = (orc.family(v[None, :], 201, orc.SCALE_MAD, 0, n_iter=0).scale[0, 100] for v in (x, y))
    assert a0 == a1
    assert m1 > 1.5 * m0


# ------------------------------------------------------------------ F2, second part: segments (reading R23)
def _segment_case(seed, S=2, N=700):
    from workloads import lightcurves as lc
    grid = lc.random_series(seed, S, N, nan_frac=0.03, inf_frac=0.0)
    rng = np.random.default_rng(seed)
    for b in range(S):                                     # a few wide gaps and one island of 5 samples
        for _ in range(3):
            a = int(rng.integers(50, N - 120))
            grid[b, a:a + int(rng.integers(15, 60))] = np.nan
        a = int(rng.integers(200, N - 200))
        grid[b, a - 30:a + 35] = np.nan
        grid[b, a:a + 5] = 1.0 + 1e-3 * rng.standard_normal(5).astype(np.float32)
    return lc.compact(grid, 0.02, t0=3.5, jitter=0.2, seed=seed) + (N,)


@pytest.mark.parametrize("W,brk,mseg,ecut", [(21, 10, 0, 0), (21, 10, 8, 0), (21, 12, 8, 3), (51, 25, 17, 0),
                                              (51, 40, 0, 7), (9, 0, 3, 1), (21, 3, 0, 0), (21, -1, 0, 4)])
def test_gapped_segments_brute_force(W, brk, mseg, ecut):
    # independent numpy brute force (np.split on the slot differences) incl. break_slots < h, where the
    # "own segment only" clause of R23 is what keeps a window from reaching across a short gap
    t, f, slot, N = _segment_case(100 + W + brk)
    got = orc.gapped_ex(t, f, 3.5, 0.02, N, W, break_slots=brk, min_segment=mseg, edge_cut=ecut)
    bt, bm = brute.detrend_gapped_ex(t, f, 3.5, 0.02, N, W, break_slots=brk, min_segment=mseg, edge_cut=ecut)
    assert np.array_equal(np.isnan(got.trend64), np.isnan(bt))
    ok = ~np.isnan(bt)
    assert np.array_equal(got.median[ok], bm[ok].astype(np.float32))
    assert np.allclose(got.trend64[ok], bt[ok], rtol=1e-12, atol=0.0)


def test_gapped_segments_reduce_to_plain_gap_handling():
    t, f, slot, N = _segment_case(7)
    base = orc.gapped(t, f, 3.5, 0.02, N, 21)
    off = orc.gapped_ex(t, f, 3.5, 0.02, N, 21)                       # nothing switched on
    assert np.array_equal(base.trend64, off.trend64, equal_nan=True)
    # breaks at least h slots wide cannot be crossed by a window anyway: only the bookkeeping differs
    wide = orc.gapped_ex(t, f, 3.5, 0.02, N, 21, break_slots=10)
    assert np.array_equal(base.trend64, wide.trend64, equal_nan=True)
    # a break narrower than h does change windows: with break_slots = 0 every missing slot ends a segment
    narrow = orc.gapped_ex(t, f, 3.5, 0.02, N, 21, break_slots=0, min_valid=1)
    both = ~np.isnan(base.trend64) & ~np.isnan(narrow.trend64)
    assert (base.trend64[both] != narrow.trend64[both]).any()


def test_gapped_segments_hand_example():
    # slots 0..9, a 4-slot hole, 14..16, another hole, 30..49: break at > 3 empty slots gives segments of
    # 10, 3 and 20 samples; min_segment = 4 drops the middle one; edge_cut = 2 blanks two slots at every end
    k = np.r_[0:10, 14:17, 30:50].astype(np.float64)
    t = (10.0 + 0.5 * k)[None, :]
    f = (1.0 + 0.01 * np.sin(k))[None, :].astype(np.float32)
    r = orc.gapped_ex(t, f, 10.0, 0.5, 50, 5, break_slots=3, min_segment=4, edge_cut=2, min_valid=1)
    nan = np.isnan(r.trend64[0])
    expect = np.ones(33, bool)
    expect[2:8] = False                      # slots 2..7 of the first segment
    expect[15:31] = False                    # slots 32..47 of the last one
    assert np.array_equal(nan, expect)
    # the first window that survives: slots 0..4 (the cut samples still count)
    assert r.n_valid[0, 2] == 5 and r.median[0, 2] == np.sort(f[0, 0:5])[2]
    # without the minimum length the island is a segment of its own and never sees its neighbours
    r2 = orc.gapped_ex(t, f, 10.0, 0.5, 50, 9, break_slots=3, min_valid=1)
    assert list(r2.n_valid[0, 10:13]) == [3, 3, 3]
