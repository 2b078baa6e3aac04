"""Parity comparison between the CUDA path and the fp64 oracle (SURVEY.md 8(c),
"Parity criteria").  Test helper: imports the oracle, so it lives under tests/.

  - NaN pattern identical;
  - n_iter = 0: output equals the oracle median as fp32 VALUES (-0.0 == +0.0, R18);
  - n_iter > 0: |gpu - orc| / max(|orc|, 1e-30) <= TOL at every position the oracle
    did not flag near_cutoff (some residual within 1e-5 relative of the bisquare
    cut-off); flagged positions are counted and bounded by a looser tolerance.
"""
from collections import namedtuple

import numpy as np

TOL = 1e-5            # north_star: trend within 1e-5 relative of local flux
TOL_FLAGGED = 1e-4    # near-cutoff positions: counted, reported, still bounded

Report = namedtuple("Report", "n n_nan max_rel n_flagged max_rel_flagged")


def compare_median(gpu, orc_median):
    gpu = np.asarray(gpu, dtype=np.float32).ravel()
    ref = np.asarray(orc_median, dtype=np.float32).ravel()
    assert gpu.shape == ref.shape
    nan_g, nan_r = np.isnan(gpu), np.isnan(ref)
    assert np.array_equal(nan_g, nan_r), "NaN pattern differs at %d positions" % int((nan_g != nan_r).sum())
    ok = ~nan_r
    bad = np.flatnonzero(gpu[ok] != ref[ok])
    assert bad.size == 0, "median not bit-exact at %d positions, first %r" % (bad.size, bad[:5])
    return Report(gpu.size, int(nan_r.sum()), 0.0, 0, 0.0)


def compare_trend(gpu, orc, tol=TOL, tol_flagged=TOL_FLAGGED):
    """`orc` is an oracle.OracleResult (trend64 + near_cutoff) for the same positions."""
    gpu = np.asarray(gpu, dtype=np.float32).ravel().astype(np.float64)
    ref = np.asarray(orc.trend64, dtype=np.float64).ravel()
    flag = np.asarray(orc.near_cutoff).ravel().astype(bool)
    assert gpu.shape == ref.shape
    nan_g, nan_r = np.isnan(gpu), np.isnan(ref)
    assert np.array_equal(nan_g, nan_r), "NaN pattern differs at %d positions" % int((nan_g != nan_r).sum())
    ok = ~nan_r
    rel = np.zeros_like(ref)
    rel[ok] = np.abs(gpu[ok] - ref[ok]) / np.maximum(np.abs(ref[ok]), 1e-30)
    plain = ok & ~flagged(flag)
    fl = ok & flagged(flag)
    max_rel = float(rel[plain].max()) if plain.any() else 0.0
    max_fl = float(rel[fl].max()) if fl.any() else 0.0
    assert max_rel <= tol, "max rel err %.3e > %.1e at %d" % (max_rel, tol, int(np.argmax(np.where(plain, rel, 0))))
    assert max_fl <= tol_flagged, "near-cutoff max rel err %.3e" % max_fl
    return Report(gpu.size, int(nan_r.sum()), max_rel, int(fl.sum()), max_fl)


def flagged(flag):
    return np.asarray(flag, dtype=bool)
