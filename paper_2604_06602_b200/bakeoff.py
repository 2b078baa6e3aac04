"""Bake-off runner: the alternatives of csrc/bakeoff/umi_bakeoff.cu against the product kernels.

    python -m paper_2604_06602_b200.build --bakeoff      # libumi_bakeoff.so (never part of libumi_b200.so)
    python -m paper_2604_06602_b200.bakeoff [--out FILE]  # one B200; prints a markdown table

north_star asks for the Phase-1 selection scheme "picked by measurement" among a shared-memory
radix/bucket select, an incrementally maintained sorted window per warp, and the per-tile sort with
sliding walkers the product uses; and names warp-per-window + shuffle reductions for Phases 2-3, where
the product uses thread-per-4-positions without reductions.  Each candidate is first checked against
the product's output on the same input (medians bit for bit, trends to 2e-6 relative), then timed with
CUDA events (L2 flushed between iterations), per window bucket W = 217 / 361 / 2161 on the synthetic
stars of configs 5 / 2 / 4 (workloads/lightcurves.py).  Product code, not test code: no oracle here.
"""
import argparse
import ctypes
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

BAKEOFF_LIB = os.path.join(HERE, "libumi_bakeoff.so")
# (config id, stars): sizes that keep the slowest candidate under a second per run
CASES = ((5, 2000), (2, 1000), (4, 60))


def _lib():
    if not os.path.exists(BAKEOFF_LIB):
        raise ImportError("%s not found: python -m paper_2604_06602_b200.build --bakeoff" % BAKEOFF_LIB)
    L = ctypes.CDLL(BAKEOFF_LIB)
    vp, i64, ci, cf = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_float
    L.umi_bakeoff_median_radix.restype = ci
    L.umi_bakeoff_median_radix.argtypes = [vp, i64, i64, ci, vp, vp]
    L.umi_bakeoff_median_warp_sorted.restype = ci
    L.umi_bakeoff_median_warp_sorted.argtypes = [vp, i64, i64, ci, ci, vp, vp]
    L.umi_bakeoff_paper_design.restype = ci
    L.umi_bakeoff_paper_design.argtypes = [vp, i64, i64, ci, cf, cf, ci, vp, vp]
    L.umi_bakeoff_reweight_warp_window.restype = ci
    L.umi_bakeoff_reweight_warp_window.argtypes = [vp, vp, i64, i64, ci, cf, cf, ci, vp, vp]
    return L


def _timed(fn, flush, steps=5, warmup=2):
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ms = []
    for _ in range(steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    return float(np.median(ms))


def run(out=None):
    import torch
    import paper_2604_06602_b200 as umi
    from workloads import lightcurves as lc
    L = _lib()
    umi.lib()
    dev = torch.device("cuda", 0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    sptr = torch.cuda.current_stream(dev).cuda_stream
    rows = []
    for cid, n_stars in CASES:
        cfg = lc.CONFIGS[cid]
        W = cfg.W
        flux = torch.from_numpy(lc.stars(cid, range(n_stars))).to(dev)
        S, N = flux.shape
        med = umi.umi_detrend(None, flux, W, n_iter=0)
        trend = umi.umi_detrend(None, flux, W, alpha=cfg.alpha, n_iter=cfg.n_iter)
        cand = torch.empty_like(flux)

        def same_median(t):
            torch.cuda.synchronize()
            return bool(torch.equal(torch.isnan(t), torch.isnan(med)) and
                        torch.equal(torch.nan_to_num(t, nan=0.0), torch.nan_to_num(med, nan=0.0)))

        def check(st):
            if st != 0:
                raise RuntimeError("bake-off entry point returned %d" % st)

        # product: per-kernel times from the library's own events
        prof = [umi.umi_detrend_profile(None, flux, W, alpha=cfg.alpha, n_iter=cfg.n_iter)[1:] for _ in range(5)]
        prod_med, prod_rw = float(np.median([p[0] for p in prof])), float(np.median([p[1] for p in prof]))
        # (i) radix select
        f1 = lambda: check(L.umi_bakeoff_median_radix(flux.data_ptr(), S, N, W, cand.data_ptr(), sptr))
        f1()
        ok1 = same_median(cand)
        t1 = _timed(f1, flush)
        # (ii) sorted window per warp, runs of 256 and 1024 positions
        t2 = {}
        ok2 = True
        for run_len in (256, 1024):
            f2 = lambda: check(L.umi_bakeoff_median_warp_sorted(flux.data_ptr(), S, N, W, run_len, cand.data_ptr(), sptr))
            cand.zero_()
            f2()
            ok2 = ok2 and same_median(cand)
            t2[run_len] = _timed(f2, flush)
        # (iii) warp per window for Phases 2-3
        f3 = lambda: check(L.umi_bakeoff_reweight_warp_window(flux.data_ptr(), med.data_ptr(), S, N, W, float(cfg.alpha), 5.0,
                                                              int(cfg.n_iter), cand.data_ptr(), sptr))
        f3()
        torch.cuda.synchronize()
        fin = ~torch.isnan(trend)
        rel = ((cand[fin] - trend[fin]).abs() / trend[fin].abs()).max().item()
        ok3 = bool(torch.equal(torch.isnan(cand), torch.isnan(trend)) and rel <= 2e-6)
        t3 = _timed(f3, flush)
        # (0) the paper's design, whole path (W <= 385 only), against the product's whole step
        t0 = ok0 = None
        if W <= 385:
            f0 = lambda: check(L.umi_bakeoff_paper_design(flux.data_ptr(), S, N, W, float(cfg.alpha), 5.0, int(cfg.n_iter), cand.data_ptr(), sptr))
            f0()
            torch.cuda.synchronize()
            rel0 = ((cand[fin] - trend[fin]).abs() / trend[fin].abs()).max().item()
            ok0 = bool(torch.equal(torch.isnan(cand), torch.isnan(trend)) and rel0 <= 1e-5)
            t0 = _timed(f0, flush, steps=3, warmup=1)
        rows.append((cid, S, N, W, prod_med, t1, ok1, t2[256], t2[1024], ok2, prod_rw, t3, ok3, rel, t0, ok0))
        del flux, med, trend, cand
    lines = ["| config (stars x cadences) | W | Phase 1: product (sort + walkers) | (i) radix select, warp per position | "
             "(ii) sorted window per warp, runs of 256 / 1024 | Phases 2-3: product (thread per 4 positions) | "
             "(iii) warp per window + shuffles | whole path: product | (0) the paper's design, thread per position + quickselect in local memory |",
             "|---|---|---|---|---|---|---|---|---|"]
    for r in rows:
        cid, S, N, W, pm, t1, ok1, t2a, t2b, ok2, prw, t3, ok3, rel, t0, ok0 = r
        paper = "n/a (W > 385)" if t0 is None else "%.1f ms (%.0fx), %s" % (t0, t0 / (pm + prw), "agrees" if ok0 else "MISMATCH")
        lines.append("| %d (%d x %d) | %d | %.3f ms | %.3f ms (%.1fx), %s | %.3f / %.3f ms (%.1fx), %s | %.3f ms | "
                     "%.3f ms (%.2fx), %s (max rel diff %.1e) | %.3f ms | %s |"
                     % (cid, S, N, W, pm, t1, t1 / pm, "bit-exact" if ok1 else "MISMATCH", t2a, t2b, min(t2a, t2b) / pm,
                        "bit-exact" if ok2 else "MISMATCH", prw, t3, t3 / prw, "agrees" if ok3 else "MISMATCH", rel, pm + prw, paper))
    text = "\n".join(lines)
    print(text)
    if out:
        with open(out, "w") as f:
            f.write(text + "\n")
    return all(r[6] and r[9] and r[12] and r[15] is not False for r in rows)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None)
    sys.exit(0 if run(ap.parse_args().out) else 1)
