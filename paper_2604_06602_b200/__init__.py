"""paper_2604_06602_b200 -- B200 (sm_100a) UMI sliding-window detrender.

Thin Python binding over the C-ABI library declared in include/umi.h
(libumi_b200.so, built by paper_2604_06602_b200/build.py).  Argument
marshalling only: every step of the path runs in the CUDA kernels.  There is no
CPU fallback: if the library is missing the import of any entry point raises.

    W = umi_window_len(dt_days)
    trend = umi_detrend(None, flux_cuda, W)             # PAPER.md:37-63, [S, N] fp32 CUDA tensor
    trend = umi_detrend_host(None, flux_numpy, W)       # host buffers, streamed batches
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# UMI_B200_LIB selects another build of the same library (kernel experiments); default: in-tree.
LIB_PATH = os.environ.get("UMI_B200_LIB") or os.path.join(_HERE, "libumi_b200.so")

UMI_OK, UMI_ERR_INVALID_ARG, UMI_ERR_UNSUPPORTED, UMI_ERR_CUDA, UMI_ERR_TOO_LARGE = 0, 1, 2, 3, 4
UMI_STATIC_SCRATCH_BYTES = 16 << 20
UMI_MAX_WINDOW = 4097
UMI_SCALE_UPPER_RMS, UMI_SCALE_MAD = 0, 1
UMI_WEIGHT_BISQUARE, UMI_WEIGHT_WELSCH = 0, 1

EXPORTS = ("umi_window_len", "umi_detrend", "umi_detrend_ex", "umi_detrend_host", "umi_detrend_profile",
           "umi_flatten", "umi_flatten_host", "umi_detrend_family", "umi_detrend_gapped", "umi_gapped_workspace_bytes",
           "umi_launch_geometry", "umi_status_string", "umi_version", "umi_shutdown",
           "umi_detrend_gapped_ex", "umi_gapped_ex_workspace_bytes",
           "umi_detrend_gapped_static", "umi_static_scratch_bytes", "umi_static_init")

_lib = None


class UmiError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(message)
        self.status = status


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s not found: build it with `python -m paper_2604_06602_b200.build` "
            "(nvcc, sm_100a).  There is no CPU fallback." % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, ci, cf = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_float
    L.umi_window_len.restype = ci
    L.umi_window_len.argtypes = [ctypes.c_double]
    L.umi_detrend.restype = ci
    L.umi_detrend.argtypes = [vp, vp, i64, i64, ci, cf, ci, vp, vp]
    L.umi_detrend_ex.restype = ci
    L.umi_detrend_ex.argtypes = [vp, vp, i64, i64, ci, cf, cf, ci, ci, vp, vp]
    L.umi_detrend_profile.restype = ci
    L.umi_detrend_profile.argtypes = [vp, vp, i64, i64, ci, cf, cf, ci, ci, vp, vp, ctypes.POINTER(cf)]
    L.umi_detrend_host.restype = ci
    L.umi_detrend_host.argtypes = [vp, vp, i64, i64, ci, cf, ci, vp, i64, ci]
    L.umi_flatten.restype = ci
    L.umi_flatten.argtypes = [vp, vp, i64, i64, ci, cf, cf, ci, ci, vp, vp, vp]
    L.umi_flatten_host.restype = ci
    L.umi_flatten_host.argtypes = [vp, vp, i64, i64, ci, cf, cf, ci, ci, vp, vp, i64, ci]
    L.umi_detrend_family.restype = ci
    L.umi_detrend_family.argtypes = [vp, vp, i64, i64, ci, ci, ci, cf, cf, ci, ci, vp, vp, vp, vp]
    L.umi_gapped_workspace_bytes.restype = ctypes.c_size_t
    L.umi_gapped_workspace_bytes.argtypes = [i64, i64]
    L.umi_detrend_gapped.restype = ci
    L.umi_detrend_gapped.argtypes = [vp, vp, i64, i64, ctypes.c_double, ctypes.c_double, i64,
                                     ci, cf, cf, ci, ci, vp, vp, vp, ctypes.c_size_t, vp]
    L.umi_gapped_ex_workspace_bytes.restype = ctypes.c_size_t
    L.umi_gapped_ex_workspace_bytes.argtypes = [i64, i64]
    L.umi_detrend_gapped_ex.restype = ci
    L.umi_detrend_gapped_ex.argtypes = [vp, vp, i64, i64, ctypes.c_double, ctypes.c_double, i64,
                                        ci, cf, cf, ci, ci, i64, i64, i64, vp, vp, vp, ctypes.c_size_t, vp]
    L.umi_static_scratch_bytes.restype = ctypes.c_size_t
    L.umi_static_scratch_bytes.argtypes = []
    L.umi_static_init.restype = ci
    L.umi_static_init.argtypes = []
    L.umi_detrend_gapped_static.restype = ci
    L.umi_detrend_gapped_static.argtypes = [vp, vp, i64, i64, ctypes.c_double, ctypes.c_double, i64,
                                            ci, cf, cf, ci, ci, i64, i64, i64, vp, vp, vp]
    L.umi_launch_geometry.restype = ci
    L.umi_launch_geometry.argtypes = [ci] + [ctypes.POINTER(ci)] * 3
    L.umi_status_string.restype = ctypes.c_char_p
    L.umi_status_string.argtypes = [ci]
    L.umi_version.restype = ci
    L.umi_version.argtypes = []
    L.umi_shutdown.restype = ci
    L.umi_shutdown.argtypes = []
    _lib = L
    return L


def _check(status):
    if status != UMI_OK:
        raise UmiError(status, lib().umi_status_string(status).decode())


def umi_status_string(status):
    return lib().umi_status_string(int(status)).decode()


def umi_version():
    return int(lib().umi_version())


def umi_shutdown():
    """Release the host batch driver's memory pools and idle streams (include/umi.h)."""
    _check(lib().umi_shutdown())


def umi_window_len(dt_days):
    """W = floor(0.5/dt) | 1; 0 for a bad dt."""
    return int(lib().umi_window_len(float(dt_days)))


def umi_launch_geometry(W):
    """(median_tile, median_sort_n, weight_tile) the library uses for this W."""
    a, b, c = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(lib().umi_launch_geometry(int(W), ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
    return a.value, b.value, c.value


def _cuda_2d(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA torch.Tensor" % name)
    if t.dtype != dtype:
        raise TypeError("%s must be %s" % (name, dtype))
    if t.dim() == 1:
        t = t.unsqueeze(0)
    if t.dim() != 2 or not t.is_contiguous():
        raise ValueError("%s must be contiguous [n_stars, n_cadences]" % name)
    return t


def _time_like(time, f):
    import torch
    if time is None:
        return None
    tt = _cuda_2d(time, torch.float64, "time")
    if tt.shape != f.shape or tt.device != f.device:
        raise ValueError("time must have flux's shape and device")
    return tt


def umi_detrend(time, flux, W, alpha=2.0, n_iter=5, out=None, stream=None, c=None, min_valid=None):
    """Device path.  `flux`: CUDA fp32 [S, N] (or [N]); `time`: None or CUDA fp64 of the
    same shape.  Enqueues on `stream` (default: torch's current stream) and returns the
    CUDA fp32 trend tensor without synchronising.  `c` / `min_valid` route through
    umi_detrend_ex (Table 4)."""
    import torch
    f = _cuda_2d(flux, torch.float32, "flux")
    tt = _time_like(time, f)
    if out is not None:
        out = _cuda_2d(out, torch.float32, "out")
        if out.shape != f.shape or out.device != f.device:
            raise ValueError("out must have flux's shape and device")
    S, N = f.shape
    with _OnStream(stream, f.device) as on:
        if out is None:
            out = torch.empty_like(f)
        on.uses(f, tt, out)
        if S == 0 or N == 0:
            return out.view(flux.shape)
        tptr = None if tt is None else tt.data_ptr()
        if c is None and min_valid is None:
            st = lib().umi_detrend(tptr, f.data_ptr(), S, N, int(W), float(alpha), int(n_iter), out.data_ptr(), on.ptr)
        else:
            st = lib().umi_detrend_ex(tptr, f.data_ptr(), S, N, int(W), float(alpha),
                                      5.0 if c is None else float(c), int(n_iter),
                                      -1 if min_valid is None else int(min_valid), out.data_ptr(), on.ptr)
    _check(st)
    return out.view(flux.shape)


class _OnStream:
    """Allocations made inside the block belong to `stream` (torch's caching allocator hands memory
    out per stream, so a tensor allocated on another stream could still be in use there), and tensors
    the caller allocated elsewhere are recorded as used on it.  `stream`: None (torch's current
    stream), a torch.cuda.Stream / ExternalStream, or a raw cudaStream_t as int."""

    def __init__(self, stream, device):
        import torch
        if stream is None:
            stream = torch.cuda.current_stream(device)
        elif not hasattr(stream, "cuda_stream"):
            stream = torch.cuda.ExternalStream(int(stream), device=device)
        self.stream = stream
        self.ptr = stream.cuda_stream
        self._dev = torch.cuda.device(device)
        self._ctx = torch.cuda.stream(stream)

    def __enter__(self):
        self._dev.__enter__()
        self._ctx.__enter__()
        return self

    def __exit__(self, *exc):
        self._ctx.__exit__(*exc)
        self._dev.__exit__(*exc)
        return False

    def uses(self, *tensors):
        for t in tensors:
            if t is not None and t.numel():
                t.record_stream(self.stream)


def umi_flatten(time, flux, W, alpha=2.0, n_iter=5, c=5.0, min_valid=-1, stream=None):
    """Detrend + normalise: returns (trend, flat) with flat = flux / trend
    computed in the kernels' epilogue.  Same argument rules as umi_detrend."""
    import torch
    f = _cuda_2d(flux, torch.float32, "flux")
    tt = _time_like(time, f)
    S, N = f.shape
    with _OnStream(stream, f.device) as on:
        trend, flat = torch.empty_like(f), torch.empty_like(f)
        on.uses(f, tt)
        if S and N:
            _check(lib().umi_flatten(None if tt is None else tt.data_ptr(), f.data_ptr(), S, N, int(W), float(alpha),
                                     float(c), int(n_iter), int(min_valid), trend.data_ptr(), flat.data_ptr(), on.ptr))
    return trend.view(flux.shape), flat.view(flux.shape)


def umi_detrend_family(time, flux, W, scale_kind=0, weight_kind=0, alpha=2.0, n_iter=5, c=5.0, min_valid=-1,
                       flat=False, stream=None):
    """Sibling estimators (include/umi.h): MAD or upper-RMS scale, bisquare or Welsch weights.
    Returns (trend, scale) or (trend, scale, flat)."""
    import torch
    f = _cuda_2d(flux, torch.float32, "flux")
    tt = _time_like(time, f)
    S, N = f.shape
    with _OnStream(stream, f.device) as on:
        trend, scale = torch.empty_like(f), torch.empty_like(f)
        fl = torch.empty_like(f) if flat else None
        on.uses(f, tt)
        if S and N:
            _check(lib().umi_detrend_family(None if tt is None else tt.data_ptr(), f.data_ptr(), S, N, int(W),
                                            int(scale_kind), int(weight_kind), float(alpha), float(c), int(n_iter),
                                            int(min_valid), trend.data_ptr(), scale.data_ptr(),
                                            fl.data_ptr() if flat else None, on.ptr))
    out = (trend.view(flux.shape), scale.view(flux.shape))
    return out + (fl.view(flux.shape),) if flat else out


def umi_gapped_workspace_bytes(n_stars, n_grid):
    return int(lib().umi_gapped_workspace_bytes(int(n_stars), int(n_grid)))


def umi_gapped_ex_workspace_bytes(n_stars, n_grid):
    return int(lib().umi_gapped_ex_workspace_bytes(int(n_stars), int(n_grid)))


def umi_detrend_gapped(time, flux, t0, dt, n_grid, W, alpha=2.0, n_iter=5, c=5.0, min_valid=-1,
                       flat=False, workspace=None, stream=None, break_slots=-1, min_segment=0, edge_cut=0):
    """Compacted rows with real time stamps (gap handling; include/umi.h).
    `time` CUDA fp64 [S, M], `flux` CUDA fp32 [S, M].  Returns trend, or (trend, flat).
    break_slots / min_segment / edge_cut: segments (umi_detrend_gapped_ex; all off by default).
    `workspace`: optional CUDA uint8 tensor of at least umi_gapped[_ex]_workspace_bytes bytes; when it is
    not given, one is allocated on `stream`, so its release is ordered after the kernels that use it."""
    import torch
    f = _cuda_2d(flux, torch.float32, "flux")
    tt = _cuda_2d(time, torch.float64, "time")
    if tt.shape != f.shape or tt.device != f.device:
        raise ValueError("time must have flux's shape and device")
    S, M = f.shape
    segments = break_slots >= 0 or min_segment > 0 or edge_cut > 0
    need = umi_gapped_ex_workspace_bytes(S, n_grid) if segments else umi_gapped_workspace_bytes(S, n_grid)
    if workspace is not None and not (isinstance(workspace, torch.Tensor) and workspace.is_cuda and workspace.is_contiguous()):
        raise TypeError("workspace must be a contiguous CUDA tensor")
    with _OnStream(stream, f.device) as on:
        if workspace is None:
            workspace = torch.empty(max(need, 1), dtype=torch.uint8, device=f.device)
        wbytes = workspace.numel() * workspace.element_size()
        trend = torch.empty_like(f)
        fl = torch.empty_like(f) if flat else None
        on.uses(f, tt, workspace)
        if S and M:
            _check(lib().umi_detrend_gapped_ex(tt.data_ptr(), f.data_ptr(), S, M, float(t0), float(dt), int(n_grid),
                                               int(W), float(alpha), float(c), int(n_iter), int(min_valid),
                                               int(break_slots), int(min_segment), int(edge_cut),
                                               trend.data_ptr(), fl.data_ptr() if flat else None,
                                               workspace.data_ptr(), wbytes, on.ptr))
    return (trend.view(flux.shape), fl.view(flux.shape)) if flat else trend.view(flux.shape)


def umi_static_scratch_bytes():
    return int(lib().umi_static_scratch_bytes())


def umi_static_init():
    """Look up the static scratch array's address on the current device now (include/umi.h)."""
    _check(lib().umi_static_init())


def umi_detrend_gapped_static(time, flux, t0, dt, n_grid, W, alpha=2.0, n_iter=5, c=5.0, min_valid=-1,
                              out=None, out_flat=None, stream=None, break_slots=-1, min_segment=0, edge_cut=0):
    """umi_detrend_gapped without a workspace: the scratch is the library's static device array of
    UMI_STATIC_SCRATCH_BYTES (include/umi.h: limit, and calls that overlap on the GPU race on it).
    With `out` (and `out_flat`, when the flattened curve is wanted) given, nothing is allocated at all;
    otherwise the trend tensor is. Returns trend, or (trend, flat) when `out_flat` is given.
    A job beyond the array raises UmiError with status UMI_ERR_TOO_LARGE."""
    import torch
    f = _cuda_2d(flux, torch.float32, "flux")
    tt = _cuda_2d(time, torch.float64, "time")
    if tt.shape != f.shape or tt.device != f.device:
        raise ValueError("time must have flux's shape and device")
    S, M = f.shape
    for name, o in (("out", out), ("out_flat", out_flat)):
        if o is not None and not (isinstance(o, torch.Tensor) and o.is_cuda and o.dtype == torch.float32 and
                                  o.is_contiguous() and o.numel() == f.numel() and o.device == f.device):
            raise TypeError("%s must be a contiguous CUDA float32 tensor of flux's size" % name)
    with _OnStream(stream, f.device) as on:
        trend = out if out is not None else torch.empty_like(f)
        on.uses(f, tt, trend, out_flat)
        if S and M:
            _check(lib().umi_detrend_gapped_static(tt.data_ptr(), f.data_ptr(), S, M, float(t0), float(dt), int(n_grid),
                                                   int(W), float(alpha), float(c), int(n_iter), int(min_valid),
                                                   int(break_slots), int(min_segment), int(edge_cut),
                                                   trend.data_ptr(), None if out_flat is None else out_flat.data_ptr(),
                                                   on.ptr))
    return trend if out_flat is None else (trend, out_flat)


def umi_detrend_profile(time, flux, W, alpha=2.0, n_iter=5, out=None, stream=None, c=5.0, min_valid=-1):
    """umi_detrend plus per-kernel device times: returns (trend, median_ms, reweight_ms).
    Synchronises the stream (measurement aid)."""
    import torch
    f = _cuda_2d(flux, torch.float32, "flux")
    tt = _time_like(time, f)
    S, N = f.shape
    ms = (ctypes.c_float * 2)()
    with _OnStream(stream, f.device) as on:
        if out is None:
            out = torch.empty_like(f)
        o = _cuda_2d(out, torch.float32, "out")
        on.uses(f, tt, o)
        _check(lib().umi_detrend_profile(None if tt is None else tt.data_ptr(), f.data_ptr(), S, N, int(W), float(alpha),
                                         float(c), int(n_iter), int(min_valid), o.data_ptr(), on.ptr, ms))
    return out.view(flux.shape), float(ms[0]), float(ms[1])


_np = None
_torch = None


def _host_modules():
    global _np, _torch
    if _np is None:
        import numpy
        _np = numpy
        try:
            import torch
            _torch = torch
        except ImportError:  # pragma: no cover
            _torch = False
    return _np, (_torch or None)


def _host_array(a, want, name):
    """(address, shape, element count) of a C-contiguous host array: numpy array or CPU tensor of dtype `want`
    ("float32" / "float64").  No copy, no conversion: anything else is a TypeError."""
    np, torch = _host_modules()
    if torch is not None and isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != getattr(torch, want) or not a.is_contiguous():
            raise TypeError("%s must be a C-contiguous %s host array" % (name, want))
        return a.data_ptr(), tuple(a.shape), a.numel()
    if not isinstance(a, np.ndarray) or a.dtype != want or not a.flags.c_contiguous:
        raise TypeError("%s must be a C-contiguous %s host array" % (name, want))
    return a.ctypes.data, a.shape, a.size


def _rows(shape):
    if len(shape) == 1:
        return 1, shape[0]
    if len(shape) != 2:
        raise ValueError("flux must be [n_stars, n_cadences]")
    return shape


def umi_detrend_host(time, flux, W, alpha=2.0, n_iter=5, out=None, stars_per_batch=0, n_streams=0):
    """Host path (batch driver).  `flux`: C-contiguous fp32 numpy array or CPU tensor
    [S, N]; `time`: None or fp64 of the same shape; pinned memory makes the copies
    overlap.
    Returns `out` (same kind as `flux`) after all batches are back."""
    np, torch = _host_modules()
    fptr, shape, size = _host_array(flux, "float32", "flux")
    S, N = _rows(shape)
    tptr = None
    if time is not None:
        tptr, _, tsize = _host_array(time, "float64", "time")
        if tsize != size:
            raise ValueError("time must have flux's shape")
    if out is None:
        out = torch.empty_like(flux) if (torch is not None and isinstance(flux, torch.Tensor)) else np.empty_like(flux)
    optr, _, osize = _host_array(out, "float32", "out")
    if osize != size:
        raise ValueError("out must have flux's shape")
    if S and N:
        _check(lib().umi_detrend_host(tptr, fptr, S, N, int(W), float(alpha), int(n_iter),
                                      optr, int(stars_per_batch), int(n_streams)))
    return out


def umi_flatten_host(time, flux, W, alpha=2.0, n_iter=5, c=5.0, min_valid=-1, want_trend=True,
                     stars_per_batch=0, n_streams=0, out_trend=None, out_flat=None):
    """Host path with the normalisation fused in: returns (trend or None, flat), of flux's shape.
    `flux`: C-contiguous fp32 numpy array or CPU tensor; `out_trend` / `out_flat`: optional
    buffers of the same shape to fill (default: new numpy arrays); pinned memory overlaps copies."""
    np, torch = _host_modules()
    fptr, shape, size = _host_array(flux, "float32", "flux")
    S, N = _rows(shape)
    tptr = None
    if time is not None:
        tptr, _, tsize = _host_array(time, "float64", "time")
        if tsize != size:
            raise TypeError("time must be a C-contiguous float64 host array of flux's shape")
    trend = None
    trptr = None
    if want_trend:
        trend = out_trend if out_trend is not None else np.empty(shape, dtype=np.float32)
        trptr, _, n = _host_array(trend, "float32", "out_trend")
        if n != size:
            raise ValueError("out_trend must have flux's shape")
    flat = out_flat if out_flat is not None else np.empty(shape, dtype=np.float32)
    flptr, _, n = _host_array(flat, "float32", "out_flat")
    if n != size:
        raise ValueError("out_flat must have flux's shape")
    if S and N:
        _check(lib().umi_flatten_host(tptr, fptr, S, N, int(W), float(alpha), float(c), int(n_iter),
                                      int(min_valid), trptr, flptr, int(stars_per_batch), int(n_streams)))
    return trend, flat
