"""umi_detrend_gapped_static (include/umi.h): the gap-handling path with its scratch in the library's static
device array instead of a caller workspace, for callers that cannot allocate.  Checked against the existing
path (umi_detrend_gapped with a workspace) on two calls in a row that share the array, against the oracle, and
for the size limit.  Collected last on purpose (pytest -x).
"""
import numpy as np
import pytest

from oracle import umi_oracle as orc
from tests import parity
from workloads import lightcurves as lc

pytestmark = pytest.mark.gpu

T0 = 2458000.25
DT = 2.0 / 1440


@pytest.fixture(scope="module")
def umi():
    import paper_2604_06602_b200 as m
    m.lib()
    return m


def _cuda(a, dtype):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def _rows(seed, S, N, W, jitter=0.3):
    grid = lc.random_series(seed, S, N, nan_frac=0.04, inf_frac=0.0)
    grid[S - 1, N // 3:N // 3 + W + 40] = np.nan            # a gap wider than the window
    t, f, _ = lc.compact(grid, DT, t0=T0, jitter=jitter, seed=seed)
    return t, f


def _same(got, want):
    # same kernels on the same inputs: the tests' tolerance (parity.TOL, 1e-5 relative) and the same NaN pattern
    got, want = got.cpu().numpy().astype(np.float64), want.cpu().numpy().astype(np.float64)
    assert np.array_equal(np.isnan(got), np.isnan(want))
    ok = ~np.isnan(want)
    assert ok.any()
    rel = np.abs(got[ok] - want[ok]) / np.maximum(np.abs(want[ok]), 1e-30)
    assert rel.max() <= parity.TOL, rel.max()


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row(umi):
    import torch
    assert umi.umi_static_scratch_bytes() == umi.UMI_STATIC_SCRATCH_BYTES == 16 << 20
    umi.umi_static_init()
    # call 1: W = 361 (two kernels), 6 stars x 6001 slots = 288 KB of the array, trend and flattened curve.
    # call 2: W = 25 (fused kernel), fewer and shorter rows, segments on (17 bytes per slot: another carve-up of
    # the same bytes), so what call 1 left behind lies under and beyond every region call 2 uses.
    cases = [(361, 6, 6001, {}), (25, 3, 2501, dict(break_slots=24, min_segment=12, edge_cut=3))]
    inputs = []
    for i, (W, S, N, seg) in enumerate(cases):
        t, f = _rows(7000 + i, S, N, W)
        inputs.append((_cuda(t, np.float64), _cuda(f, np.float32), t, f))
    want = []
    for (W, S, N, seg), (td, fd, _, _) in zip(cases, inputs):
        want.append(umi.umi_detrend_gapped(td, fd, T0, DT, N - 5, W, flat=True, **seg))
    outs = [(torch.empty_like(fd), torch.empty_like(fd)) for (_, fd, _, _) in inputs]
    torch.cuda.synchronize()
    # the two calls back to back on one stream, outputs preallocated: nothing is allocated in between
    for (W, S, N, seg), (td, fd, _, _), (o, of) in zip(cases, inputs, outs):
        got = umi.umi_detrend_gapped_static(td, fd, T0, DT, N - 5, W, out=o, out_flat=of, **seg)
        assert got[0] is o and got[1] is of
    torch.cuda.synchronize()
    for (o, of), (wt, wf) in zip(outs, want):
        _same(o, wt)
        _same(of, wf)
    # and against the oracle
    (W, S, N, seg), (_, _, t, f) = cases[0], inputs[0]
    parity.compare_trend(outs[0][0].cpu().numpy(), orc.gapped(t, f, T0, DT, N - 5, W))
    (W, S, N, seg), (_, _, t, f) = cases[1], inputs[1]
    parity.compare_trend(outs[1][0].cpu().numpy(), orc.gapped_ex(t, f, T0, DT, N - 5, W, **seg))
    # the first job once more after the second: the array's contents from call 2 change nothing
    (W, S, N, seg), (td, fd, _, _) = cases[0], inputs[0]
    again = umi.umi_detrend_gapped_static(td, fd, T0, DT, N - 5, W)
    torch.cuda.synchronize()
    _same(again, want[0][0])


def test_static_scratch_calls_allocate_no_device_memory(umi):
    import torch
    W, S, N = 217, 4, 5001
    t, f = _rows(7100, S, N, W)
    td, fd = _cuda(t, np.float64), _cuda(f, np.float32)
    o, of = torch.empty_like(fd), torch.empty_like(fd)
    umi.umi_detrend_gapped_static(td, fd, T0, DT, N, W, out=o, out_flat=of)      # loads the kernels (lazy module loading)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    reserved_before = torch.cuda.memory_reserved()
    for _ in range(3):
        umi.umi_detrend_gapped_static(td, fd, T0, DT, N, W, out=o, out_flat=of)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_reserved() == reserved_before                       # not through torch's allocator
    assert free_after >= free_before                                             # nor behind its back (cudaMalloc would lower it)
    _same(o, umi.umi_detrend_gapped(td, fd, T0, DT, N, W))


def test_static_scratch_refuses_jobs_beyond_the_array(umi):
    import torch
    limit = umi.umi_static_scratch_bytes()
    n_grid = 4096
    fits = limit // 8 // n_grid                               # 512 stars of 4096 slots: exactly the array
    t = np.tile(T0 + DT * np.arange(8), (fits + 1, 1))
    f = np.ones((fits + 1, 8), np.float32)
    td, fd = _cuda(t, np.float64), _cuda(f, np.float32)
    out = umi.umi_detrend_gapped_static(td[:fits], fd[:fits], T0, DT, n_grid, 5)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), f[:fits])        # constant rows: the trend is the constant
    with pytest.raises(umi.UmiError) as e:
        umi.umi_detrend_gapped_static(td, fd, T0, DT, n_grid, 5)
    assert e.value.status == umi.UMI_ERR_TOO_LARGE and "UMI_STATIC_SCRATCH_BYTES" in str(e.value)
    with pytest.raises(umi.UmiError) as e:                    # segments need 17 bytes per slot: the same job no longer fits
        umi.umi_detrend_gapped_static(td[:fits], fd[:fits], T0, DT, n_grid, 5, edge_cut=1)
    assert e.value.status == umi.UMI_ERR_TOO_LARGE
    with pytest.raises(umi.UmiError) as e:                    # sizes whose product overflows 64 bits are refused, not wrapped
        umi.umi_detrend_gapped_static(td, fd, T0, DT, 2 ** 62, 5)
    assert e.value.status == umi.UMI_ERR_TOO_LARGE
