"""Seeded synthetic light curves: the five configurations of BASELINE.json.

Shared by the oracle-side tests and the CUDA-side tests/bench as INPUTS ONLY.
This module holds none of the method's arithmetic (no median, scale, weights or
window rule: W is a constant of each config) and imports neither `oracle` nor
`paper_2604_06602_b200`.

They stand in for the paper's real TESS / Kepler light curves (PAPER.md:91, 105,
141-147), which are not available; no item of any archive is reproduced.  The
recipe is DESIGN.md, "Input recipe":

  star b of config n draws from numpy Generator(PCG64(SeedSequence([seed_n, b])))
  so any subset of stars regenerates identically; t_j = j*dt (days); flux is
  built in fp64 and cast to fp32; log-U = uniform in log; sinusoid phases
  U[0, 2pi); transit centres U[0, span]; trapezoid ingress = egress = 10 % of the
  duration; flares rise instantly at U[0, span] and decay with tau U[5, 60] min.
"""
from collections import namedtuple
import concurrent.futures
import os

import numpy as np

Config = namedtuple("Config", "name seed n_stars n_cadences dt_days W alpha n_iter")

MIN = 1.0 / 1440.0
SEC = 1.0 / 86400.0

CONFIGS = {
    1: Config("tess_single", 0, 1, 19440, 2 * MIN, 361, 2.0, 5),
    2: Config("tess_batch", 1, 1000, 19440, 2 * MIN, 361, 2.0, 5),
    3: Config("kepler_lc", 2, 10000, 70000, 29.4 * MIN, 25, 2.0, 5),
    4: Config("tess_20s", 3, 200, 116640, 20 * SEC, 2161, 2.0, 5),
    5: Config("ffi_sweep", 4, 100000, 11664, 200 * SEC, 217, 2.0, 5),
}


def _logu(rng, lo, hi, size=None):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), size))


def _add_sinusoids(rng, t, flux, count, p_lo, p_hi, a_lo, a_hi, log_amp):
    for _ in range(count):
        period = rng.uniform(p_lo, p_hi)
        amp = _logu(rng, a_lo, a_hi) if log_amp else rng.uniform(a_lo, a_hi)
        phase = rng.uniform(0.0, 2.0 * np.pi)
        flux += amp * np.sin(2.0 * np.pi * t / period + phase)


def _trapezoid(t, centre, duration, depth):
    """1 at mid-transit, linear ingress/egress each 10 % of `duration`."""
    half = 0.5 * duration
    ramp = 0.1 * duration
    x = np.abs(t - centre)
    prof = np.clip((half - x) / ramp, 0.0, 1.0)
    return -depth * prof


def _box(t, centre, duration, depth):
    return np.where(np.abs(t - centre) <= 0.5 * duration, -depth, 0.0)


def _tess_like(rng, t, sigma_lo, sigma_hi):
    """Generator of configs 2, 4, 5: sinusoids + noise + trapezoid transits + flares."""
    span = t[-1]
    flux = np.ones_like(t)
    _add_sinusoids(rng, t, flux, int(rng.integers(1, 6)), 0.5, 10.0, 1e-4, 1e-2, True)
    sigma = _logu(rng, sigma_lo, sigma_hi)
    flux += rng.normal(0.0, sigma, t.size)
    for _ in range(int(rng.integers(0, 5))):
        depth = _logu(rng, 1e-4, 5e-2)
        duration = rng.uniform(1.0, 8.0) / 24.0
        flux += _trapezoid(t, rng.uniform(0.0, span), duration, depth)
    for _ in range(int(rng.integers(0, 4))):
        amp = rng.uniform(1e-3, 2e-2)
        t0 = rng.uniform(0.0, span)
        tau = rng.uniform(5.0, 60.0) * MIN
        dtf = t - t0
        flux += np.where(dtf >= 0.0, amp * np.exp(-np.maximum(dtf, 0.0) / tau), 0.0)
    return flux, sigma


def star(config_id, b):
    """fp32 flux of star `b` of config `config_id`, shape [n_cadences]."""
    cfg = CONFIGS[config_id]
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed, int(b)])))
    n = cfg.n_cadences
    t = np.arange(n, dtype=np.float64) * cfg.dt_days
    span = t[-1]
    if config_id == 1:
        flux = np.ones(n)
        _add_sinusoids(rng, t, flux, 3, 0.5, 10.0, 1e-4, 5e-3, False)
        flux += rng.normal(0.0, 1e-3, n)
        flux += _box(t, rng.uniform(2.0, 25.0), 3.0 / 24.0, 1e-3)
    elif config_id == 2:
        flux, _ = _tess_like(rng, t, 2e-4, 5e-3)
        flux[9360:10080] = np.nan
    elif config_id == 3:
        flux = np.ones(n)
        _add_sinusoids(rng, t, flux, int(rng.integers(1, 4)), 1.0, 30.0, 1e-5, 5e-3, True)
        flux += rng.normal(0.0, _logu(rng, 3e-5, 1e-3), n)
        n_ev = int(rng.integers(0, 21))
        if n_ev > 0:
            period = span / n_ev
            epoch = rng.uniform(0.0, period)
            depth = _logu(rng, 5e-5, 1e-2)
            duration = rng.uniform(1.0, 8.0) / 24.0
            phase = np.mod(t - epoch + 0.5 * period, period) - 0.5 * period
            flux += np.where(np.abs(phase) <= 0.5 * duration, -depth, 0.0)
        bad = np.zeros(n, dtype=bool)
        while bad.sum() < 0.01 * n:
            run = int(rng.integers(10, 101))
            start = int(rng.integers(0, n - run + 1))
            bad[start:start + run] = True
        flux[bad] = np.nan
    elif config_id == 4:
        flux, sigma = _tess_like(rng, t, 5e-4, 1e-2)
        hit = rng.random(n) < 0.05
        amp = rng.uniform(5.0, 50.0, n) * sigma * np.where(rng.random(n) < 0.5, -1.0, 1.0)
        flux += np.where(hit, amp, 0.0)
        flux[56160:60480] = np.nan
    elif config_id == 5:
        flux, _ = _tess_like(rng, t, 2e-4, 5e-3)
        start = int(rng.integers(217, n - 649 + 1))
        flux[start:start + 432] = np.nan
    else:
        raise KeyError(config_id)
    return flux.astype(np.float32)


def _stars_chunk(args):
    config_id, idx = args
    return np.stack([star(config_id, b) for b in idx])


def stars(config_id, indices, workers=None):
    """fp32 [len(indices), n_cadences] for the listed star indices (any subset, any order)."""
    indices = [int(b) for b in indices]
    cfg = CONFIGS[config_id]
    if not indices:
        return np.empty((0, cfg.n_cadences), np.float32)
    if workers is None:
        workers = min(os.cpu_count() or 1, 32)
    total = len(indices) * cfg.n_cadences
    if workers <= 1 or total < 4_000_000:
        return _stars_chunk((config_id, indices))
    chunks = [c for c in np.array_split(np.asarray(indices), min(len(indices), workers * 4)) if len(c)]
    import multiprocessing
    with concurrent.futures.ProcessPoolExecutor(max_workers=workers, mp_context=multiprocessing.get_context("spawn")) as ex:
        parts = list(ex.map(_stars_chunk, [(config_id, c.tolist()) for c in chunks]))
    return np.concatenate(parts, axis=0)


def make(config_id, n_stars=None, workers=None):
    """(Config, flux[n_stars, n_cadences] fp32) for the first n_stars stars (default: all)."""
    cfg = CONFIGS[config_id]
    n = cfg.n_stars if n_stars is None else int(n_stars)
    return cfg, stars(config_id, range(n), workers=workers)


def times(config_id, n_stars):
    """fp64 [n_stars, n_cadences] time stamps t_j = j*dt (uniform grid, identical rows)."""
    cfg = CONFIGS[config_id]
    t = np.arange(cfg.n_cadences, dtype=np.float64) * cfg.dt_days
    return np.broadcast_to(t, (int(n_stars), cfg.n_cadences)).copy()


def random_series(seed, n_stars, n_cadences, nan_frac=0.05, inf_frac=0.01, ties=False):
    """Small adversarial arrays for parity tests: noise around 1 with scattered NaN/Inf
    runs and, optionally, heavy ties (values quantised to a handful of levels)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([977, int(seed)])))
    x = 1.0 + 1e-3 * rng.standard_normal((n_stars, n_cadences))
    x += 2e-3 * np.sin(np.arange(n_cadences) / 37.0)[None, :]
    if ties:
        x = np.round(x * 400.0) / 400.0
    x = x.astype(np.float32)
    if nan_frac > 0:
        x[rng.random(x.shape) < nan_frac] = np.nan
        for b in range(n_stars):
            if n_cadences > 8:
                run = int(rng.integers(1, max(2, n_cadences // 3)))
                s = int(rng.integers(0, n_cadences - run + 1))
                x[b, s:s + run] = np.nan
    if inf_frac > 0:
        m = rng.random(x.shape) < inf_frac
        x[m] = np.where(rng.random(m.sum()) < 0.5, np.inf, -np.inf).astype(np.float32)
    return x


def compact(flux_grid, dt_days, t0=0.0, jitter=0.0, seed=0):
    """Compacted rows with real time stamps, as a mission pipeline delivers them after
    quality filtering: the non-finite slots of a uniform-grid array are
    REMOVED, so time jumps across gaps.  Returns (time[S, M] fp64, flux[S, M] fp32,
    slot[S, M] int64) with M = the longest row; shorter rows are padded at the end with
    NaN time / NaN flux / slot -1.  time = t0 + slot*dt + U(-jitter, jitter)*dt (inputs
    only: no method arithmetic here; `slot` is what the caller started from, for tests)."""
    flux_grid = np.atleast_2d(np.asarray(flux_grid, dtype=np.float32))
    S, N = flux_grid.shape
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([4242, int(seed)])))
    keep = [np.flatnonzero(np.isfinite(flux_grid[b])) for b in range(S)]
    M = max([k.size for k in keep] + [1])
    time = np.full((S, M), np.nan, np.float64)
    flux = np.full((S, M), np.nan, np.float32)
    slot = np.full((S, M), -1, np.int64)
    for b, k in enumerate(keep):
        slot[b, :k.size] = k
        flux[b, :k.size] = flux_grid[b, k]
        time[b, :k.size] = t0 + (k + rng.uniform(-jitter, jitter, k.size)) * dt_days
    return time, flux, slot
