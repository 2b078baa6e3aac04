"""Synthetic injection-recovery workload (Tables 1-2).

The paper injects box transits (period 3 d, duration 3 h, depths 5-1000 ppm) into 1,000 real
TESS sector-6 and 1,000 Kepler Q5 light curves, detrends, and reports the median over stars of
the absolute percentage error of the recovered depth.  Those light curves and the comparison
system (wotan) are not available; this module reproduces the SHAPE of the experiment on the
seeded generator stars of `workloads.lightcurves` (config 2 for TESS, config 3 for Kepler) with
the estimator settings of PAPER.md Table 4.  Inputs and the depth metric only: the detrending
itself is done by whoever calls `depth_errors` (the CUDA path in the CLI below and in the GPU
test; the fp64 oracle in the CPU cross-check of that test).

CLI (needs a GPU):  python -m workloads.injection_recovery [--config 2] [--stars 1000]
"""
import argparse
import json

import numpy as np

from workloads import lightcurves as lc

DEPTHS_PPM = (5.0, 50.0, 100.0, 200.0, 500.0, 1000.0)        # PAPER.md:121, 131 (table columns)
PERIOD_DAYS = 3.0
DURATION_DAYS = 3.0 / 24.0
SETTINGS = {                                                 # PAPER.md:202-209 (Table 4); scale/weight kinds: include/umi.h
    "UMI default (alpha=2, c=5)": dict(alpha=2.0, c=5.0, scale_kind=0, weight_kind=0),
    "UMI aggressive (alpha=10, c=2.5)": dict(alpha=10.0, c=2.5, scale_kind=0, weight_kind=0),
    "symmetric, upper-RMS scale (alpha=1, c=5)": dict(alpha=1.0, c=5.0, scale_kind=0, weight_kind=0),
    # the rows the paper takes from wotan, here as the sibling estimators of row F4
    "biweight, MAD scale (alpha=1, c=5)": dict(alpha=1.0, c=5.0, scale_kind=1, weight_kind=0),
    "Welsch, MAD scale (alpha=1, c=5)": dict(alpha=1.0, c=5.0, scale_kind=1, weight_kind=1),
    # the ablation of PAPER.md:91: UMI's asymmetric weights on the MAD instead of the upper-RMS
    "UMI weights on the MAD (alpha=2, c=5)": dict(alpha=2.0, c=5.0, scale_kind=1, weight_kind=0),
}


def transit_mask(n_stars, n_cadences, dt_days, seed=0):
    """Boolean [n_stars, n_cadences]: in-transit cadences of a box train with the paper's period
    and duration and a per-star random epoch."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([31337, int(seed)])))
    t = np.arange(n_cadences, dtype=np.float64) * dt_days
    epoch = rng.uniform(0.0, PERIOD_DAYS, n_stars)
    phase = np.mod(t[None, :] - epoch[:, None] + 0.5 * PERIOD_DAYS, PERIOD_DAYS) - 0.5 * PERIOD_DAYS
    return np.abs(phase) <= 0.5 * DURATION_DAYS


def inject(flux, mask, depth_ppm):
    """flux - depth inside the mask (fp32 in, fp32 out; NaN slots stay NaN)."""
    return (flux.astype(np.float64) - depth_ppm * 1e-6 * mask).astype(np.float32)


def recovered_depth(flat, mask):
    """Per star: mean out-of-transit level minus mean in-transit level of the flattened curve
    (so a constant offset of the trend, cancels).  NaN-aware.  [n_stars]."""
    flat = np.asarray(flat, dtype=np.float64)
    ok = np.isfinite(flat)
    n_in = np.maximum((ok & mask).sum(axis=1), 1)
    n_out = np.maximum((ok & ~mask).sum(axis=1), 1)
    s_in = np.where(ok & mask, flat, 0.0).sum(axis=1)
    s_out = np.where(ok & ~mask, flat, 0.0).sum(axis=1)
    return s_out / n_out - s_in / n_in


def depth_errors(flux, dt_days, flatten, depths_ppm=DEPTHS_PPM, seed=0, differential=True):
    """Median over stars of |recovered - injected| / injected * 100 for each depth.
    `flatten(flux_fp32) -> flat` is the detrender under test.
    differential=True: the depth the same detrender 'recovers' from the un-injected curve (noise
    and the star's own structure under the mask) is subtracted, which isolates what the
    detrender absorbs; False is the paper's raw metric, noise-limited at
    shallow depths."""
    mask = transit_mask(flux.shape[0], flux.shape[1], dt_days, seed)
    base = recovered_depth(flatten(flux), mask) if differential else 0.0
    out = []
    for d in depths_ppm:
        rec = recovered_depth(flatten(inject(flux, mask, d)), mask) - base
        out.append(float(np.median(np.abs(rec - d * 1e-6) / (d * 1e-6) * 100.0)))
    return out


def main():
    import torch
    import paper_2604_06602_b200 as umi
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2, choices=(2, 3))
    ap.add_argument("--stars", type=int, default=1000)
    ap.add_argument("--raw", action="store_true", help="the paper's raw metric (no differential baseline)")
    a = ap.parse_args()
    cfg, flux = lc.make(a.config, a.stars)
    rows = {}
    for name, kw in SETTINGS.items():
        def flatten(x, kw=kw):
            _, _, flat = umi.umi_detrend_family(None, torch.from_numpy(x).cuda(), cfg.W, n_iter=cfg.n_iter,
                                                flat=True, **kw)
            return flat.cpu().numpy()
        rows[name] = depth_errors(flux, cfg.dt_days, flatten, differential=not a.raw)
    print(json.dumps({"config": cfg.name, "stars": a.stars, "W": cfg.W, "depths_ppm": DEPTHS_PPM,
                      "metric": "raw" if a.raw else "differential", "median_abs_pct_error": rows}))


if __name__ == "__main__":
    main()
