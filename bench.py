#!/usr/bin/env python
"""bench.py -- detrended cadences/s of the UMI hot path on B200 (BASELINE.json metric).

  python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
  python bench.py --impl reference ...                     # the fp64 oracle on host cores

A "step" is one pass of the whole hot path (median kernel + reweighting kernel,
SURVEY.md 8(a) rows a1-a5) over one synthetic batch.  Default workload = config 2,
the one the metric is quoted on: 1,000 stars x 19,440 cadences, W = 361, alpha = 2,
5 iterations (workloads/lightcurves.py, seeded; stands in for TESS sector data).
N > 1 (torchrun): stars are independent, each rank detrends its own 1,000
separately seeded stars, no collective on the data path -> "scaling": "weak".

Prints ONE JSON line ("Measurement", for every field).
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import lightcurves as lc  # noqa: E402

METRIC = "detrended cadences/sec on 1 B200 (TESS W=361 batch) + fraction of roofline"
UNIT = "cadences/s"

# DESIGN.md section 6, "Roofline".  The path is bound by the FMA pipe (148 SMs x 128 FP32 lanes, one lane-operation
# per lane per clock; a packed FFMA2/FMUL2/FADD2 is two lane-operations).  FMA-pipe lane-operations per
# window-sample the kernels EXECUTE (counted in the SASS of the inner loops, cross-checked against ncu's
# sm__pipe_fma_cycles_active in profiles/):
#   reweighting kernel (W > 49): Phase 2 = 2 (x - med, ss += d*d; n+ comes with the median); a pass = 5 when alpha
#     is 1, 2 or 4 (u' = x(-k) + mu k; n = e*e - 1; w = n*n; S += w; R += w x -- alpha*u is an integer add on the
#     ALU pipe), 6 for any other alpha (one more multiply)
#   fused short-window kernel (W <= 49): see FMA_OPS_SMALL below
# Beside it, as labelled side figures only: the survey's algorithmic FMA-pipe count (2 + 6 per pass) and its
# nominal 49 issue slots per window-sample (4 + 9 per pass), which packed fp32x2 and DPX instructions beat, so
# that figure is not a fraction of any hardware ceiling.
SM_COUNT = 148
LANES_PER_SM = 128          # FP32 lanes of the FMA pipe per SM (4 SMSPs x 32)
FMA_OPS_SMALL = (3, 6, 5)   # fused short-window kernel: Phase 2 (sub, fma, count), a pass (general alpha), a pass (alpha = 2)
NOMINAL_PHASE2, NOMINAL_PER_PASS = 4, 9
SURVEY_FMA_PHASE2, SURVEY_FMA_PER_PASS = 2, 6


def fma_ops_per_window_sample(W, alpha, n_iter):
    """(executed FMA-pipe lane-operations per window-sample, description) for the kernel that runs this W."""
    if W <= 49:
        p2, pp = FMA_OPS_SMALL[0], (FMA_OPS_SMALL[2] if alpha == 2.0 else FMA_OPS_SMALL[1])
        return p2 + pp * n_iter, "%d (Phase 2) + %d x %d passes, fused short-window kernel" % (p2, pp, n_iter)
    pp = 5 if alpha in (1.0, 2.0, 4.0) else 6
    return 2 + pp * n_iter, "2 (Phase 2) + %d x %d passes, alpha %s" % (pp, n_iter, "= 2^m: integer-add form" if pp == 5 else "general")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=sorted(lc.CONFIGS))
    ap.add_argument("--stars", type=int, default=None, help="override the star count (debug)")
    ap.add_argument("--row", default="base", choices=["base", "f1", "f2", "f2seg", "f4mad", "f4welsch"],
                    help="SURVEY.md 8(f) next rows on the same workload: f1 = umi_flatten, f2 = umi_detrend_gapped on the "
                         "compacted rows, f4mad / f4welsch = umi_detrend_family (symmetric biweight on the MAD / Welsch)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def exact_window_samples(flux, W, min_valid):
    """Sum over evaluated positions (own sample valid, >= min_valid valid samples in the
    window) of the number of valid samples in the window.  Host-side bookkeeping for the
    roofline numerator: a validity prefix sum, none of the method's arithmetic."""
    S, N = flux.shape
    h = W // 2
    lo = np.clip(np.arange(N) - h, 0, N)
    hi = np.clip(np.arange(N) + h + 1, 0, N)
    total = 0
    for s0 in range(0, S, 256):
        valid = np.isfinite(flux[s0:s0 + 256])
        csum = np.zeros((valid.shape[0], N + 1), np.int64)
        np.cumsum(valid, axis=1, out=csum[:, 1:])
        n = csum[:, hi] - csum[:, lo]
        ev = valid & (n >= min_valid)
        total += int(n[ev].sum())
    return total


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index, period=0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def shard_stars(rank, world, stars_per_rank):
    """Weak scaling: rank r owns the separately seeded stars [r*S, (r+1)*S); no data-path collective."""
    return range(rank * stars_per_rank, (rank + 1) * stars_per_rank)


def max_over_ranks(value, dist, device=None):
    """Max over ranks of a host scalar (timings); identity when not distributed."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def ncu_record(config_id, n_stars, kernel_prefix):
    """Counters of the dominant kernel for THIS workload from the committed ncu --set full capture
    (profiles/ncu_r02.json, written from the .ncu-rep by hand; the commands are in profiles/README.md):
    dram bytes per launch, FMA-pipe utilisation, executed warp instructions.  None if no capture of this
    configuration at this size is committed."""
    path = os.path.join(ROOT, "profiles", "ncu_r02.json")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        rec = json.load(f)
    cfgrec = rec.get("config%d" % config_id)
    if not cfgrec or cfgrec.get("n_stars") != n_stars:
        return None
    for name, v in cfgrec.get("kernels", {}).items():
        if name.startswith(kernel_prefix):
            return dict(v, kernel=name)
    return None


def oracle_sample(cfg, flux, n_stars):
    """Times the fp64 oracle, as it stands, on the first n_stars stars of the workload."""
    from oracle import umi_oracle as orc
    sub = np.ascontiguousarray(flux[:n_stars])
    orc.detrend(sub[:1, :2000], cfg.W)                       # load + thread pool warm-up
    t0 = time.perf_counter()
    orc.detrend(sub, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    dt = time.perf_counter() - t0
    return sub.size / dt, dt, orc.num_threads()


def run_reference(args, cfg, rank):
    """--impl reference: the oracle on the box's host cores, each step a bounded sample."""
    if rank != 0:
        return
    n_sample = min(cfg.n_stars if args.stars is None else args.stars,
                   max(1, int(600_000 // cfg.n_cadences) or 1))       # ~0.6 M cadences per step
    flux = lc.stars(args.config, range(n_sample))
    from oracle import umi_oracle as orc
    for _ in range(max(args.warmup, 1)):
        orc.detrend(flux[:1], cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.detrend(flux, cfg.W, alpha=cfg.alpha, n_iter=cfg.n_iter)
    dt = time.perf_counter() - t0
    value = flux.size * args.steps / dt
    sample = "first %d of %d stars per step, all cadences, fp64, OpenMP" % (n_sample, cfg.n_stars)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "gpu_launches": 0,
        "config": {"workload": "config%d %s: %d stars x %d cadences, W=%d, alpha=%g, n_iter=%d"
                   % (args.config, cfg.name, cfg.n_stars, cfg.n_cadences, cfg.W, cfg.alpha, cfg.n_iter)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def run_ours(args, cfg, rank, world, local_rank):
    import torch
    import paper_2604_06602_b200 as umi
    umi.lib()                                            # no fallback: raises if the .so is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --impl ours needs a CUDA device (no CPU fallback)")
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    S = cfg.n_stars if args.stars is None else args.stars
    N, W = cfg.n_cadences, cfg.W
    flux_np = lc.stars(args.config, shard_stars(rank, world, S))          # weak scaling: own stars
    min_valid = max(1, W // 3)
    ws_exact = exact_window_samples(flux_np, W, min_valid)
    h_flux = torch.from_numpy(flux_np).pin_memory()
    h_out = torch.empty_like(h_flux).pin_memory()
    d_flux = h_flux.to(dev, non_blocking=True)
    d_out = torch.empty_like(d_flux)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2
    stream = torch.cuda.Stream(dev)
    torch.cuda.synchronize()

    def step():
        umi.umi_detrend(None, d_flux, W, alpha=cfg.alpha, n_iter=cfg.n_iter, out=d_out, stream=stream)

    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            flush.zero_()
            step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()

    # ---- timed region: K steps, device time per step from CUDA events on the launch stream
    sampler = ClockSampler(local_rank, period=0.01)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        for a, b in ev:
            flush.zero_()                                # L2 flush between timed iterations (untimed)
            a.record(stream)
            step()
            b.record(stream)
    torch.cuda.synchronize()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    # ---- same steps again through umi_detrend_profile: per-kernel device times (events
    #      recorded by the library on the same stream), for the roofline of the dominant kernel
    k_ms = []
    with torch.cuda.stream(stream):
        for _ in range(args.steps):
            flush.zero_()
            _, m1, m2 = umi.umi_detrend_profile(None, d_flux, W, alpha=cfg.alpha, n_iter=cfg.n_iter,
                                                out=d_out, stream=stream)
            k_ms.append((m1, m2))
    clocks = sampler.stop()
    if dist is not None:
        dist.barrier()
    total_ms = max_over_ranks(sum(step_ms), dist, dev)

    # ---- end to end through the public host API: pinned host buffers in, pinned host out
    e2e = None
    if not args.no_e2e:
        for _ in range(2):
            umi.umi_detrend_host(None, h_flux, W, alpha=cfg.alpha, n_iter=cfg.n_iter, out=h_out)
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            umi.umi_detrend_host(None, h_flux, W, alpha=cfg.alpha, n_iter=cfg.n_iter, out=h_out)
        e2e_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
        e2e = {"value": world * S * N * args.steps / e2e_s, "unit": UNIT,
               "h2d_bytes_per_step": int(h_flux.numel() * 4), "d2h_bytes_per_step": int(h_out.numel() * 4),
               "ms_per_step": 1e3 * e2e_s / args.steps,
               "api": "umi_detrend_host (C ABI, pinned host buffers, 3 streams)"}
        # copy / compute overlap of the batch driver: the same bytes copied alone, one direction at a time (pinned
        # host <-> device, CUDA events), against the pipelined wall time above
        ca, cb, cc = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        d_tmp = torch.empty_like(d_flux)
        d_tmp.copy_(h_flux, non_blocking=True)
        h_out.copy_(d_tmp, non_blocking=True)
        torch.cuda.synchronize()
        ca.record()
        d_tmp.copy_(h_flux, non_blocking=True)
        cb.record()
        h_out.copy_(d_tmp, non_blocking=True)
        cc.record()
        torch.cuda.synchronize()
        h2d_ms, d2h_ms = ca.elapsed_time(cb), cb.elapsed_time(cc)
        del d_tmp
        kern_ms = sum(step_ms) / len(step_ms)
        serial = h2d_ms + kern_ms + d2h_ms
        e2e["pipeline"] = {"h2d_ms_alone": h2d_ms, "d2h_ms_alone": d2h_ms, "kernels_ms_alone": kern_ms,
                           "pcie_h2d_GBps": h_flux.numel() * 4 / h2d_ms / 1e6, "pcie_d2h_GBps": h_out.numel() * 4 / d2h_ms / 1e6,
                           "serial_sum_ms": serial, "longest_stage_ms": max(h2d_ms, kern_ms, d2h_ms),
                           "hidden_frac": (serial - e2e["ms_per_step"]) / max(serial - max(h2d_ms, kern_ms, d2h_ms), 1e-9)}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    pk, pk_kind = peaks()
    ms_per_step = total_ms / args.steps
    value = world * S * N / (ms_per_step * 1e-3)
    med_ms = float(np.mean([a for a, _ in k_ms]))
    rw_ms = float(np.mean([b for _, b in k_ms]))
    sm_max = float(clocks["sm_max_mhz"] or pk.get("sm_max_mhz", 1965.0))
    sm_now = float(clocks["sm_mhz"] or sm_max)
    peak = SM_COUNT * LANES_PER_SM * sm_max * 1e6 / 1e12                 # T FMA-pipe lane-op/s at max clock
    fma_ops, fma_def = fma_ops_per_window_sample(W, cfg.alpha, cfg.n_iter)
    kname = "umi_small_kernel" if W <= 49 else "umi_reweight_kernel"
    achieved = fma_ops * ws_exact / (rw_ms * 1e-3) / 1e12
    ncu = ncu_record(args.config, S, kname)
    nominal = NOMINAL_PHASE2 + NOMINAL_PER_PASS * cfg.n_iter
    survey_fma = SURVEY_FMA_PHASE2 + SURVEY_FMA_PER_PASS * cfg.n_iter
    roofline = {
        "bound": "alu", "pipe": "fma", "kernel": kname + (" (fused phases 1-3)" if W <= 49 else ""),
        "achieved": achieved, "peak": peak, "unit": "T FMA-pipe lane-op/s", "frac": achieved / peak,
        "peak_def": "148 SMs x 128 FP32 lanes x sm_max_mhz (%s clocks); achieved = executed FMA-pipe lane-ops per "
                    "window-sample [%s] x exact window-samples / kernel time" % (pk_kind, fma_def),
        "frac_at_measured_clock": achieved / (peak * sm_now / sm_max),
        "fma_pipe_lane_ops_per_window_sample": fma_ops,
        "window_samples_per_launch": ws_exact, "window_samples_nominal": S * N * W,
        "kernel_ms": rw_ms, "median_kernel_ms": med_ms, "kernel_share_of_step": rw_ms / (rw_ms + med_ms),
        "window_samples_per_s": ws_exact / (ms_per_step * 1e-3),
        # cross-check from the committed ncu capture of this same launch configuration (None: none committed)
        "ncu_fma_pipe_pct": None if ncu is None else ncu.get("fma_pipe_pct"),
        "ncu_issue_active_pct": None if ncu is None else ncu.get("issue_active_pct"),
        "ncu_kernel": None if ncu is None else ncu.get("kernel"),
        "traffic": None if ncu is None else ncu.get("dram_bytes_read", 0) + ncu.get("dram_bytes_write", 0),
        # side figures, NOT fractions of a hardware ceiling
        "frac_survey_fma_count": survey_fma * ws_exact / (rw_ms * 1e-3) / 1e12 / peak,
        "frac_nominal_issue": nominal * ws_exact / (rw_ms * 1e-3) / 1e12 / peak,
        "hbm_algorithmic_GBps": 8.0 * S * N / (ms_per_step * 1e-3) / 1e9, "hbm_peak_GBps": pk.get("hbm_gbs"),
        "hbm_frac": 8.0 * S * N / (ms_per_step * 1e-3) / 1e9 / float(pk.get("hbm_gbs") or 6549.4),
    }
    cpu = None
    if not args.no_cpu_baseline:
        rate, _, cores = oracle_sample(cfg, flux_np, min(S, 16))
        n_s = int(min(S, max(16, rate * 15.0 / N)))                      # ~15 s of host work
        rate, secs, cores = oracle_sample(cfg, flux_np, n_s)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "first %d of %d stars, all cadences, %.1f s" % (n_s, S, secs)}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "config%d %s: %d stars x %d cadences per GPU, W=%d, alpha=%g, n_iter=%d"
                   % (args.config, cfg.name, S, N, W, cfg.alpha, cfg.n_iter),
                   "l2": "256 MiB buffer written between timed iterations",
                   "timing": "CUDA events on the launch stream, per step, summed; max over ranks"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": (1 if W <= 49 else 2) * args.steps,
        "roofline": roofline, "cpu_baseline": cpu,
        "paper_context": "PAPER.md:147: 3.4 ms/star on AMD RX 9060 XT (~5.7e6 cadences/s at N=19440); not a target",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_row(args, cfg, local_rank):
    """Next rows on the configured workload, one GPU: device-resident step time with
    CUDA events, L2 flushed between iterations, next to the base path timed the same way."""
    import torch
    import paper_2604_06602_b200 as umi
    umi.lib()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    S = cfg.n_stars if args.stars is None else args.stars
    N, W = cfg.n_cadences, cfg.W
    flux_np = lc.stars(args.config, range(S))
    d_flux = torch.from_numpy(flux_np).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.Stream(dev)
    kw = dict(alpha=cfg.alpha, n_iter=cfg.n_iter)
    extra = {}
    if args.row == "f1":
        fn = lambda: umi.umi_flatten(None, d_flux, W, stream=stream, **kw)
        what = "umi_flatten: trend + flux/trend in the kernels' epilogue"
    elif args.row in ("f2", "f2seg"):
        t_np, f_np, _ = lc.compact(flux_np, cfg.dt_days, t0=1000.0, jitter=0.1, seed=args.config)
        d_t, d_f = torch.from_numpy(t_np).to(dev), torch.from_numpy(f_np).to(dev)
        seg = dict(break_slots=W - 1, min_segment=W // 3, edge_cut=W // 10) if args.row == "f2seg" else {}
        nbytes = umi.umi_gapped_ex_workspace_bytes(S, N) if seg else umi.umi_gapped_workspace_bytes(S, N)
        ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        fn = lambda: umi.umi_detrend_gapped(d_t, d_f, 1000.0, cfg.dt_days, N, W, flat=True, workspace=ws,
                                            stream=stream, **seg, **kw)
        what = "umi_detrend_gapped%s: compacted rows [%d x %d] + fp64 time -> grid [%d x %d] -> trend, flat" % (
            " with segments (break W-1 slots, min_segment W/3, edge_cut W/10)" if seg else "", S, f_np.shape[1], S, N)
        M = f_np.shape[1]
        # algorithmic bytes of the two regrid kernels + the NaN fill: scatter reads time (8) + flux (4) per
        # sample and writes 4 per valid sample; the fill writes 4 per slot; gather reads time (8) + flux (4)
        # + trend (4) and writes trend (4) + flat (4)
        if not seg:
            extra["regrid_bytes"] = int(S * M * (12 + 4) + S * N * 4 + S * M * (16 + 8))
    else:
        wk = 1 if args.row == "f4welsch" else 0
        fn = lambda: umi.umi_detrend_family(None, d_flux, W, 1, wk, alpha=1.0, n_iter=cfg.n_iter, stream=stream)
        what = "umi_detrend_family: MAD scale, %s weights, alpha=1" % ("Welsch" if wk else "bisquare")
    base = lambda: umi.umi_detrend(None, d_flux, W, stream=stream, **kw)

    def timed(f):
        with torch.cuda.stream(stream):
            for _ in range(max(args.warmup, 3)):
                flush.zero_()
                f()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        with torch.cuda.stream(stream):
            for a, b in ev:
                flush.zero_()
                a.record(stream)
                f()
                b.record(stream)
        torch.cuda.synchronize()
        return float(np.mean([a.elapsed_time(b) for a, b in ev]))

    sampler = ClockSampler(local_rank, period=0.01)
    sampler.start()
    base_ms = timed(base)
    row_ms = timed(fn)
    clocks = sampler.stop()
    n_cad = int(np.isfinite(flux_np).sum()) if args.row in ("f2", "f2seg") else S * N
    line = {"metric": METRIC, "row": args.row, "what": what, "value": n_cad / (row_ms * 1e-3), "unit": UNIT,
            "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": row_ms,
            "base_path_ms_per_step": base_ms, "overhead_ms": row_ms - base_ms, "higher_is_better": True,
            "dtype": "f32", "data": "synthetic", "clocks": clocks,
            "config": {"workload": "config%d %s: %d stars x %d cadences, W=%d" % (args.config, cfg.name, S, N, W),
                       "l2": "256 MiB buffer written between timed iterations"}}
    if "regrid_bytes" in extra and row_ms > base_ms:
        pk, _ = peaks()
        gbs = extra["regrid_bytes"] / ((row_ms - base_ms) * 1e-3) / 1e9
        line["roofline_regrid"] = {"bound": "hbm", "achieved": gbs, "peak": pk.get("hbm_gbs"), "unit": "GB/s",
                                   "frac": gbs / pk.get("hbm_gbs"), "bytes": extra["regrid_bytes"],
                                   "note": "fill + scatter + gather, time = row step - base step"}
    print(json.dumps(line))


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = lc.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg, rank)
    elif args.row != "base":
        if rank == 0:
            run_row(args, cfg, local_rank)
    else:
        run_ours(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
