"""ctypes loader for the fp64 CPU oracle (oracle/umi_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_2604_06602_b200 and holds no arithmetic of its own:
argument marshalling only.
"""
import ctypes
import importlib.util
import os
from collections import namedtuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def _load_build_module():
    spec = importlib.util.spec_from_file_location("_umi_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


_lib = None

OracleResult = namedtuple(
    "OracleResult", "trend64 trend32 median scale n_valid n_plus near_cutoff")

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_float_p = ctypes.POINTER(ctypes.c_float)
_c_i64_p = ctypes.POINTER(ctypes.c_int64)
_c_i32_p = ctypes.POINTER(ctypes.c_int32)
_c_u8_p = ctypes.POINTER(ctypes.c_uint8)


def lib():
    global _lib
    if _lib is None:
        path = _load_build_module().build()
        L = ctypes.CDLL(path)
        L.umi_oracle_window_len.restype = ctypes.c_int
        L.umi_oracle_window_len.argtypes = [ctypes.c_double]
        L.umi_oracle_weight.restype = ctypes.c_double
        L.umi_oracle_weight.argtypes = [ctypes.c_double, ctypes.c_double]
        L.umi_oracle_num_threads.restype = ctypes.c_int
        L.umi_oracle_num_threads.argtypes = []
        outs = [_c_double_p, _c_float_p, _c_float_p, _c_double_p, _c_i32_p, _c_i32_p, _c_u8_p]
        L.umi_oracle_detrend.restype = ctypes.c_int
        L.umi_oracle_detrend.argtypes = [
            _c_double_p, _c_float_p, ctypes.c_int64, ctypes.c_int64,
            ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            ctypes.c_double] + outs
        L.umi_oracle_positions.restype = ctypes.c_int
        L.umi_oracle_positions.argtypes = [
            _c_double_p, _c_float_p, ctypes.c_int64, ctypes.c_int64,
            _c_i64_p, _c_i64_p, ctypes.c_int64,
            ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            ctypes.c_double] + outs
        L.umi_oracle_family.restype = ctypes.c_int
        L.umi_oracle_family.argtypes = [
            _c_double_p, _c_float_p, ctypes.c_int64, ctypes.c_int64,
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int,
            ctypes.c_int, ctypes.c_double] + outs
        L.umi_oracle_normalize.restype = ctypes.c_int
        L.umi_oracle_normalize.argtypes = [_c_float_p, _c_double_p, ctypes.c_int64, _c_double_p]
        L.umi_oracle_gapped.restype = ctypes.c_int
        L.umi_oracle_gapped.argtypes = [
            _c_double_p, _c_float_p, ctypes.c_int64, ctypes.c_int64,
            ctypes.c_double, ctypes.c_double, ctypes.c_int64,
            ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            ctypes.c_double] + outs
        L.umi_oracle_gapped_ex.restype = ctypes.c_int
        L.umi_oracle_gapped_ex.argtypes = [
            _c_double_p, _c_float_p, ctypes.c_int64, ctypes.c_int64,
            ctypes.c_double, ctypes.c_double, ctypes.c_int64,
            ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_double] + outs
        _lib = L
    return _lib


def window_len(dt_days: float) -> int:
    return int(lib().umi_oracle_window_len(float(dt_days)))


def weight(u: float, alpha: float) -> float:
    return float(lib().umi_oracle_weight(float(u), float(alpha)))


def num_threads() -> int:
    return int(lib().umi_oracle_num_threads())


def _prep(flux, time):
    flux = np.ascontiguousarray(flux, dtype=np.float32)
    if flux.ndim == 1:
        flux = flux[None, :]
    if flux.ndim != 2:
        raise ValueError("flux must be [n_stars, n_cadences]")
    tp = None
    if time is not None:
        time = np.ascontiguousarray(time, dtype=np.float64)
        if time.ndim == 1:
            time = time[None, :]
        if time.shape != flux.shape:
            raise ValueError("time must have flux's shape")
        tp = time.ctypes.data_as(_c_double_p)
    return flux, time, tp


def _alloc(shape):
    return OracleResult(
        trend64=np.empty(shape, np.float64), trend32=np.empty(shape, np.float32),
        median=np.empty(shape, np.float32), scale=np.empty(shape, np.float64),
        n_valid=np.empty(shape, np.int32), n_plus=np.empty(shape, np.int32),
        near_cutoff=np.empty(shape, np.uint8))


def _out_ptrs(r):
    return [r.trend64.ctypes.data_as(_c_double_p), r.trend32.ctypes.data_as(_c_float_p),
            r.median.ctypes.data_as(_c_float_p), r.scale.ctypes.data_as(_c_double_p),
            r.n_valid.ctypes.data_as(_c_i32_p), r.n_plus.ctypes.data_as(_c_i32_p),
            r.near_cutoff.ctypes.data_as(_c_u8_p)]


def detrend(flux, W, alpha=2.0, n_iter=5, c=5.0, time=None, min_valid=-1,
            cutoff_tol=1e-5) -> OracleResult:
    """Every position of every star.  Returns arrays of flux's 2-D shape."""
    flux, time, tp = _prep(flux, time)
    S, N = flux.shape
    r = _alloc((S, N))
    rc = lib().umi_oracle_detrend(
        tp, flux.ctypes.data_as(_c_float_p), S, N, int(W), float(alpha), float(c),
        int(n_iter), int(min_valid), float(cutoff_tol), *_out_ptrs(r))
    if rc != 0:
        raise ValueError("umi_oracle_detrend: invalid arguments")
    return r


def positions(flux, star_idx, pos_idx, W, alpha=2.0, n_iter=5, c=5.0, time=None,
              min_valid=-1, cutoff_tol=1e-5) -> OracleResult:
    """Only the listed (star, position) pairs.  Returns 1-D arrays."""
    flux, time, tp = _prep(flux, time)
    S, N = flux.shape
    star_idx = np.ascontiguousarray(star_idx, dtype=np.int64)
    pos_idx = np.ascontiguousarray(pos_idx, dtype=np.int64)
    if star_idx.shape != pos_idx.shape or star_idx.ndim != 1:
        raise ValueError("star_idx and pos_idx must be 1-D and equal length")
    r = _alloc((star_idx.size,))
    rc = lib().umi_oracle_positions(
        tp, flux.ctypes.data_as(_c_float_p), S, N,
        star_idx.ctypes.data_as(_c_i64_p), pos_idx.ctypes.data_as(_c_i64_p), star_idx.size,
        int(W), float(alpha), float(c), int(n_iter), int(min_valid), float(cutoff_tol),
        *_out_ptrs(r))
    if rc != 0:
        raise ValueError("umi_oracle_positions: invalid arguments")
    return r


def normalize(flux, trend64):
    """PAPER.md:155 normalisation stage: flat = flux / trend in fp64, flux's shape."""
    flux = np.ascontiguousarray(flux, dtype=np.float32)
    trend64 = np.ascontiguousarray(trend64, dtype=np.float64)
    if flux.size != trend64.size:
        raise ValueError("flux and trend must have the same size")
    flat = np.empty(flux.shape, np.float64)
    rc = lib().umi_oracle_normalize(flux.ctypes.data_as(_c_float_p), trend64.ctypes.data_as(_c_double_p),
                                    flux.size, flat.ctypes.data_as(_c_double_p))
    if rc != 0:
        raise ValueError("umi_oracle_normalize: invalid arguments")
    return flat


def gapped(time, flux, t0, dt, n_grid, W, alpha=2.0, n_iter=5, c=5.0, min_valid=-1,
           cutoff_tol=1e-5) -> OracleResult:
    """Compacted rows with real time stamps (gap handling; reading R20):
    the window of a sample is the valid samples within +-h grid slots of its own slot."""
    flux, time, tp = _prep(flux, time)
    if tp is None:
        raise ValueError("time is required")
    S, M = flux.shape
    r = _alloc((S, M))
    rc = lib().umi_oracle_gapped(
        tp, flux.ctypes.data_as(_c_float_p), S, M, float(t0), float(dt), int(n_grid),
        int(W), float(alpha), float(c), int(n_iter), int(min_valid), float(cutoff_tol), *_out_ptrs(r))
    if rc != 0:
        raise ValueError("umi_oracle_gapped: invalid arguments")
    return r


def gapped_ex(time, flux, t0, dt, n_grid, W, alpha=2.0, n_iter=5, c=5.0, min_valid=-1,
              break_slots=-1, min_segment=0, edge_cut=0, cutoff_tol=1e-5) -> OracleResult:
    """gapped() with segments (reading R23): rows are cut where more than break_slots empty slots lie between
    valid samples, segments shorter than min_segment are dropped, windows stay inside a segment, and samples
    closer than edge_cut slots to a segment end get NaN."""
    flux, time, tp = _prep(flux, time)
    if tp is None:
        raise ValueError("time is required")
    S, M = flux.shape
    r = _alloc((S, M))
    rc = lib().umi_oracle_gapped_ex(
        tp, flux.ctypes.data_as(_c_float_p), S, M, float(t0), float(dt), int(n_grid),
        int(W), float(alpha), float(c), int(n_iter), int(min_valid),
        int(break_slots), int(min_segment), int(edge_cut), float(cutoff_tol), *_out_ptrs(r))
    if rc != 0:
        raise ValueError("umi_oracle_gapped_ex: invalid arguments")
    return r


SCALE_UPPER_RMS, SCALE_MAD = 0, 1
WEIGHT_BISQUARE, WEIGHT_WELSCH = 0, 1


def family(flux, W, scale_kind=0, weight_kind=0, alpha=2.0, n_iter=5, c=5.0, time=None, min_valid=-1,
           cutoff_tol=1e-5) -> OracleResult:
    """Sibling estimators: MAD scale and/or Welsch weights on the same windows."""
    flux, time, tp = _prep(flux, time)
    S, N = flux.shape
    r = _alloc((S, N))
    r.n_plus[...] = 0
    rc = lib().umi_oracle_family(
        tp, flux.ctypes.data_as(_c_float_p), S, N, int(W), int(scale_kind), int(weight_kind),
        float(alpha), float(c), int(n_iter), int(min_valid), float(cutoff_tol), *_out_ptrs(r))
    if rc != 0:
        raise ValueError("umi_oracle_family: invalid arguments")
    return r
