"""CPU checks of the C-ABI boundary (include/umi.h): the library loads, exports every
declared symbol, and its host-only logic (window rule, validation, geometry) behaves
as the header says.  No kernel is launched here."""
import ctypes
import os
import re

import pytest

import paper_2604_06602_b200 as umi

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "umi.h")


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(umi_[a-z_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2604_06602_b200 import build
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert set(declared) == set(umi.EXPORTS), (declared, umi.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name
    assert umi.umi_version() >= 300
    assert L.umi_shutdown() == umi.UMI_OK          # nothing to release: no CUDA call is made


def test_window_len_paper_values_and_guard():
    # PAPER.md:35 (TESS 2 min -> 361), PAPER.md:192 (Kepler 30 min -> 25); BASELINE.json configs
    assert umi.umi_window_len(2.0 / 1440) == 361
    assert umi.umi_window_len(30.0 / 1440) == 25
    assert umi.umi_window_len(29.4 / 1440) == 25
    assert umi.umi_window_len(20.0 / 86400) == 2161
    assert umi.umi_window_len(200.0 / 86400) == 217
    # (R15) a cadence that went through fp32 must not lose the last sample
    import numpy as np
    assert umi.umi_window_len(float(np.float32(2.0 / 1440))) == 361
    assert umi.umi_window_len(float(np.float32(200.0 / 86400))) == 217
    for bad in (0.0, -1.0, float("nan"), float("inf"), 1e-300):
        assert umi.umi_window_len(bad) == 0
    assert umi.umi_window_len(10.0) == 1   # floor(0.05) | 1
    for dt in (0.001, 0.0137, 0.02, 0.3):
        W = umi.umi_window_len(dt)
        assert W % 2 == 1 and W >= 1


def test_validation_happens_on_the_host():
    L = umi.lib()
    one = ctypes.c_void_p(16)   # never dereferenced: validation fails first or sizes are 0
    call = lambda **k: L.umi_detrend(k.get("time"), k.get("flux", one), k.get("S", 1), k.get("N", 10),
                                     k.get("W", 5), k.get("alpha", 2.0), k.get("n_iter", 5),
                                     k.get("out", one), None)
    assert call(flux=None) == umi.UMI_ERR_INVALID_ARG
    assert call(out=None) == umi.UMI_ERR_INVALID_ARG
    assert call(S=-1) == umi.UMI_ERR_INVALID_ARG
    assert call(N=-1) == umi.UMI_ERR_INVALID_ARG
    assert call(W=4) == umi.UMI_ERR_INVALID_ARG
    assert call(W=0) == umi.UMI_ERR_INVALID_ARG
    assert call(W=-3) == umi.UMI_ERR_INVALID_ARG
    assert call(alpha=0.0) == umi.UMI_ERR_INVALID_ARG
    assert call(alpha=-2.0) == umi.UMI_ERR_INVALID_ARG
    assert call(alpha=float("nan")) == umi.UMI_ERR_INVALID_ARG
    assert call(alpha=float("inf")) == umi.UMI_ERR_INVALID_ARG
    assert call(n_iter=-1) == umi.UMI_ERR_INVALID_ARG
    assert call(W=umi.UMI_MAX_WINDOW + 2) == umi.UMI_ERR_UNSUPPORTED
    assert call(S=0) == umi.UMI_OK      # empty batch: nothing enqueued
    assert call(N=0) == umi.UMI_OK
    assert L.umi_detrend_ex(None, one, 1, 10, 5, 2.0, 0.0, 5, -1, one, None) == umi.UMI_ERR_INVALID_ARG
    assert L.umi_detrend_host(None, None, 1, 10, 5, 2.0, 5, one, 0, 0) == umi.UMI_ERR_INVALID_ARG
    assert L.umi_detrend_host(None, one, 0, 10, 5, 2.0, 5, one, 0, 0) == umi.UMI_OK
    # next rows: normalisation and time-stamped gap handling
    assert L.umi_flatten(None, one, 1, 10, 5, 2.0, 5.0, 5, -1, one, None, None) == umi.UMI_ERR_INVALID_ARG
    assert L.umi_flatten(None, one, 0, 10, 5, 2.0, 5.0, 5, -1, one, one, None) == umi.UMI_OK
    gap = lambda **k: L.umi_detrend_gapped(k.get("time", one), one, k.get("S", 1), 10, 0.0, k.get("dt", 0.5),
                                           k.get("n_grid", 12), 5, 2.0, 5.0, 5, -1, one, None,
                                           k.get("ws", one), k.get("wsb", 1 << 20), None)
    assert gap(time=None) == umi.UMI_ERR_INVALID_ARG
    assert gap(dt=0.0) == umi.UMI_ERR_INVALID_ARG
    assert gap(dt=float("nan")) == umi.UMI_ERR_INVALID_ARG
    assert gap(n_grid=-1) == umi.UMI_ERR_INVALID_ARG
    assert gap(ws=None) == umi.UMI_ERR_INVALID_ARG
    assert gap(wsb=95) == umi.UMI_ERR_INVALID_ARG      # 2 * 1 * 12 * 4 = 96 bytes needed
    assert gap(S=0) == umi.UMI_OK
    assert L.umi_flatten_host(None, one, 1, 10, 5, 2.0, 5.0, 5, -1, one, None, 0, 0) == umi.UMI_ERR_INVALID_ARG
    assert L.umi_flatten_host(None, one, 0, 10, 5, 2.0, 5.0, 5, -1, None, one, 0, 0) == umi.UMI_OK
    fam = lambda **k: L.umi_detrend_family(None, one, k.get("S", 1), 10, 5, k.get("sk", 0), k.get("wk", 0), 2.0, 5.0, 5, -1,
                                           one, k.get("scale", one), None, None)
    assert fam(sk=2) == umi.UMI_ERR_INVALID_ARG
    assert fam(wk=-1) == umi.UMI_ERR_INVALID_ARG
    assert fam(sk=1, scale=None) == umi.UMI_ERR_INVALID_ARG    # the MAD needs its buffer
    assert fam(S=0, scale=None) == umi.UMI_OK
    assert umi.umi_gapped_workspace_bytes(3, 100) == 2400     # two fp32 grids
    assert umi.umi_gapped_workspace_bytes(0, 100) == 0
    assert umi.umi_gapped_ex_workspace_bytes(3, 100) == 3 * 100 * 17
    gex = lambda **k: L.umi_detrend_gapped_ex(one, one, 1, 10, 0.0, 0.5, 12, k.get("W", 5), 2.0, 5.0, 5, -1, k.get("brk", -1), k.get("mseg", 0),
                                               k.get("ecut", 0), one, None, k.get("ws", one), k.get("wsb", 1 << 20), None)
    assert gex(W=51, brk=24) == umi.UMI_ERR_UNSUPPORTED       # a break a window could reach across
    assert gex(mseg=3, wsb=12 * 8) == umi.UMI_ERR_INVALID_ARG   # segments need the larger workspace
    for s in range(5):
        assert umi.umi_status_string(s)
    assert "UMI_OK" in umi.umi_status_string(0)


def test_launch_geometry():
    for W in (1, 3, 25, 217, 361, 513, 1081, 2161, 4097):
        T, NS, T2 = umi.umi_launch_geometry(W)
        assert NS & (NS - 1) == 0 and NS >= 1024
        assert T + W - 1 == NS
        assert T >= max(1, (W - 1) // 2)
        assert NS * 14 <= 227 * 1024  # sort entries + ranks + bitsets
        assert T2 == 128
    assert umi.umi_launch_geometry(361)[:2] == (664, 1024)
    with pytest.raises(umi.UmiError):
        umi.umi_launch_geometry(4)
    with pytest.raises(umi.UmiError):
        umi.umi_launch_geometry(5001)


def test_binding_rejects_host_tensors_on_the_device_path():
    import torch
    with pytest.raises(TypeError):
        umi.umi_detrend(None, torch.zeros(2, 8), 3)


def test_bakeoff_library_is_separate_and_exports_its_candidates():
    # the measured alternatives (csrc/bakeoff/) build into their own library and never into the product one
    from paper_2604_06602_b200 import build
    B = ctypes.CDLL(build.build_bakeoff())
    for name in ("umi_bakeoff_median_radix", "umi_bakeoff_median_warp_sorted", "umi_bakeoff_reweight_warp_window",
                 "umi_bakeoff_paper_design"):
        assert hasattr(B, name)
    L = ctypes.CDLL(build.build())
    assert not hasattr(L, "umi_bakeoff_median_radix")
    one = ctypes.c_void_p(16)
    B.umi_bakeoff_median_radix.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    assert B.umi_bakeoff_median_radix(one, 1, 10, 4, one, None) == 1        # even window: refused on the host
    assert B.umi_bakeoff_median_radix(one, 0, 10, 361, one, None) == 0      # empty batch: nothing enqueued


def test_static_scratch_size_and_limit_are_checked_without_a_gpu():
    # umi_detrend_gapped_static refuses a job beyond its static array before it touches CUDA
    L = umi.lib()
    assert umi.umi_static_scratch_bytes() == umi.UMI_STATIC_SCRATCH_BYTES == 16 << 20
    assert "UMI_STATIC_SCRATCH_BYTES" in umi.umi_status_string(umi.UMI_ERR_TOO_LARGE)
    dummy = ctypes.c_void_p(256)                     # never dereferenced: the size check comes first

    def call(n_stars, n_grid, edge_cut=0):
        return L.umi_detrend_gapped_static(dummy, dummy, n_stars, 8, 0.0, 0.01, n_grid, 5, 2.0, 5.0, 5, -1,
                                           -1, 0, edge_cut, dummy, None, None)

    assert call(513, 4096) == umi.UMI_ERR_TOO_LARGE              # 512 x 4096 slots x 8 bytes is exactly the array
    assert call(512, 4096, edge_cut=1) == umi.UMI_ERR_TOO_LARGE  # 17 bytes per slot with segments
    assert call(1, (16 << 20) // 8 + 1) == umi.UMI_ERR_TOO_LARGE
    assert call(2 ** 40, 2 ** 40) == umi.UMI_ERR_TOO_LARGE       # no 64-bit wrap-around
