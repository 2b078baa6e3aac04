"""CPU checks of the input generators and of the injection-recovery bookkeeping (no method
arithmetic lives in `workloads/`; these tests only pin shapes, seeds and the depth metric)."""
import numpy as np

from workloads import injection_recovery as ir
from workloads import lightcurves as lc


def test_stars_regenerate_identically_and_have_the_config_shape():
    a = lc.stars(2, [7, 3])
    b = lc.stars(2, [3, 7])
    assert a.shape == (2, lc.CONFIGS[2].n_cadences) and a.dtype == np.float32
    assert np.array_equal(a[0], b[1], equal_nan=True) and np.array_equal(a[1], b[0], equal_nan=True)
    assert np.isnan(a[:, 9360:10080]).all() and np.isfinite(a[:, :9360]).all()
    k = lc.stars(3, [0])
    assert 0.01 <= np.isnan(k).mean() <= 0.03            # runs of 10-100 NaNs until >= 1 %


def test_compact_removes_invalid_slots_and_pads_with_nan_time():
    grid = lc.random_series(5, 3, 300, nan_frac=0.1, inf_frac=0.0)
    t, f, slot = lc.compact(grid, 0.5, t0=10.0, jitter=0.2, seed=1)
    assert t.shape == f.shape == slot.shape and t.shape[0] == 3
    for b in range(3):
        m = slot[b] >= 0
        assert m.sum() == np.isfinite(grid[b]).sum()
        assert np.array_equal(f[b, m], grid[b, slot[b, m]])
        assert np.all(np.diff(slot[b, m]) > 0)
        assert np.all(np.abs((t[b, m] - 10.0) / 0.5 - slot[b, m]) <= 0.2 + 1e-9)
        assert np.isnan(t[b, ~m]).all() and np.isnan(f[b, ~m]).all()


def test_injection_metric_with_a_perfect_and_a_transit_eating_detrender():
    cfg = lc.CONFIGS[2]
    rng = np.random.default_rng(0)
    flux = (1.0 + 1e-4 * rng.standard_normal((6, cfg.n_cadences))).astype(np.float32)
    mask = ir.transit_mask(6, cfg.n_cadences, cfg.dt_days, seed=0)
    # 3 h every 3 d at 2-min cadence: ~90 cadences per transit, ~9 transits
    assert 700 <= mask[0].sum() <= 1000
    inj = ir.inject(flux, mask, 1000.0)
    assert np.allclose(flux[mask] - inj[mask], 1e-3, atol=2e-7) and np.array_equal(inj[~mask], flux[~mask])
    perfect = lambda x: x / 1.0                           # trend == 1: nothing absorbed
    err = ir.depth_errors(flux, cfg.dt_days, perfect, depths_ppm=(1000.0,))
    assert err[0] < 0.1
    eater = lambda x: np.ones_like(x)                     # trend == flux: everything absorbed
    err = ir.depth_errors(flux, cfg.dt_days, eater, depths_ppm=(1000.0,))
    assert abs(err[0] - 100.0) < 1e-6


def test_bench_roofline_bookkeeping():
    # bench.py's host-side roofline arithmetic: executed FMA-pipe lane-operations per window-sample per kernel build,
    # the exact window-sample count, and the committed ncu record it quotes beside the live figure
    import bench
    assert bench.fma_ops_per_window_sample(361, 2.0, 5)[0] == 27        # 2 + 5 x 5: alpha = 2^m, integer-add form
    assert bench.fma_ops_per_window_sample(361, 3.0, 5)[0] == 32        # 2 + 6 x 5: general alpha
    assert bench.fma_ops_per_window_sample(25, 2.0, 5)[0] == 28         # fused short-window kernel, alpha = 2
    assert bench.fma_ops_per_window_sample(25, 3.0, 5)[0] == 33
    x = np.ones((2, 50), np.float32)
    x[0, 10:20] = np.nan
    # W = 5, min_valid = 1: every valid position counts its valid window members (brute force below)
    want = 0
    for b in range(2):
        for i in range(50):
            if np.isfinite(x[b, i]):
                want += int(np.isfinite(x[b, max(0, i - 2):i + 3]).sum())
    assert bench.exact_window_samples(x, 5, 1) == want
    rec = bench.ncu_record(2, 1000, "umi_reweight_kernel")
    assert rec is not None and rec["kernel"].startswith("umi_reweight_kernel<0, 1, 1>")
    assert 50.0 < rec["fma_pipe_pct"] <= 100.0 and rec["local_ld"] == 0 and rec["local_st"] == 0
    assert bench.ncu_record(2, 999, "umi_reweight_kernel") is None      # no capture of that size: no number
    assert bench.ncu_record(3, 10000, "umi_small_kernel")["registers"] <= 80


def test_bench_reference_arm_prints_the_contract_line():
    # `bench.py --impl reference` (the oracle on host cores) must print ONE JSON line with the contract's keys
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=300, cwd=root)
    assert res.returncode == 0, res.stderr[-500:]
    lines = [ln for ln in res.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "cadences/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["gpu_launches"] == 0 and d["dtype"] == "f64"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"]
