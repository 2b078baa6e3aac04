"""Brute-force checker for the C oracle: numpy, one window at a time.

TEST INFRASTRUCTURE, NOT PRODUCT.  Written separately from umi_oracle.c (it
does not load it) so that the two can be compared: full `np.sort` for the
median, boolean masks for the one-sided scale, and direct weighted means with
`np.average`.  Pure-Python loops over positions: only for small cases.

Follows PAPER.md section 2 (lines 35-63) and the readings R1..R18 in DESIGN.md.
"""
import numpy as np

SCALE_CONST = 0.6745


def bisquare_weights(u, alpha):
    """PAPER.md:56-58 (Eq. 2-3) on an array of standardized residuals."""
    u = np.asarray(u, dtype=np.float64)
    u_eff = np.where(u < 0.0, alpha * u, u)
    inside = np.abs(u_eff) < 1.0
    return np.where(inside, (1.0 - u_eff ** 2) ** 2, 0.0)


def window_samples(flux_row, i, W, time_row=None):
    """Valid samples of the centred window [i-h, i+h] clipped to the series (R1-R3)."""
    N = len(flux_row)
    h = (W - 1) // 2
    lo, hi = max(0, i - h), min(N, i + h + 1)
    x = np.asarray(flux_row[lo:hi], dtype=np.float64)
    ok = np.isfinite(x)
    if time_row is not None:
        ok &= np.isfinite(np.asarray(time_row[lo:hi], dtype=np.float64))
    return x[ok]


def location(x, alpha=2.0, c=5.0, n_iter=5, history=False):
    """UMI location of the 1-D sample x (all valid).  Returns (mu, median, s)."""
    x = np.asarray(x, dtype=np.float64)
    n = x.size
    med = np.sort(x)[(n - 1) // 2]                      # PAPER.md:39; lower median (R6)
    upper = x[x > med]                                  # Eq. 1, strict (R7)
    if upper.size == 0:
        return (med, med, 0.0) if not history else (med, med, 0.0, [])
    s = SCALE_CONST * np.sqrt(np.mean((upper - med) ** 2))
    if not s > 0.0:
        return (med, med, s) if not history else (med, med, s, [])
    mu = med
    trace = []
    for _ in range(n_iter):
        w = bisquare_weights((x - mu) / (c * s), alpha)
        if not w.sum() > 0.0:
            break
        mu = np.average(x, weights=w)                   # Eq. 4
        trace.append(mu)
    return (mu, med, s) if not history else (mu, med, s, trace)


def detrend(flux, W, alpha=2.0, n_iter=5, c=5.0, time=None, min_valid=None):
    """Brute-force trend, median and scale for a [S, N] (or [N]) array."""
    flux = np.atleast_2d(np.asarray(flux, dtype=np.float32))
    if time is not None:
        time = np.atleast_2d(np.asarray(time, dtype=np.float64))
    S, N = flux.shape
    if min_valid is None:
        min_valid = max(1, W // 3)                      # PAPER.md:192 (R4)
    trend = np.full((S, N), np.nan)
    median = np.full((S, N), np.nan)
    scale = np.full((S, N), np.nan)
    for b in range(S):
        trow = None if time is None else time[b]
        for i in range(N):
            own_ok = np.isfinite(flux[b, i]) and (trow is None or np.isfinite(trow[i]))
            x = window_samples(flux[b], i, W, trow)
            if not own_ok or x.size < min_valid:        # (R4, R5)
                continue
            trend[b, i], median[b, i], scale[b, i] = location(x, alpha, c, n_iter)
    return trend, median, scale


def detrend_gapped(time, flux, t0, dt, n_grid, W, alpha=2.0, n_iter=5, c=5.0, min_valid=None):
    """Brute force for compacted rows with time stamps (PAPER.md:155 gap handling, reading
    R20): slot = rint((t - t0)/dt); a sample is valid iff time and flux are finite, its slot is
    inside [0, n_grid) and the next sample of the row has a different slot; its window is the
    valid samples whose slot differs from its own by at most h.  Whole-row boolean masks."""
    time = np.atleast_2d(np.asarray(time, dtype=np.float64))
    flux = np.atleast_2d(np.asarray(flux, dtype=np.float32))
    S, M = flux.shape
    h = (W - 1) // 2
    if min_valid is None:
        min_valid = max(1, W // 3)
    trend = np.full((S, M), np.nan)
    median = np.full((S, M), np.nan)
    for b in range(S):
        with np.errstate(invalid="ignore"):
            k = np.rint((time[b] - t0) / dt)
        ok = np.isfinite(time[b]) & (k >= 0) & (k < n_grid)
        same_as_next = np.zeros(M, dtype=bool)
        same_as_next[:-1] = np.isfinite(time[b, :-1]) & np.isfinite(time[b, 1:]) & (k[:-1] == k[1:])
        ok &= ~same_as_next
        ok &= np.isfinite(flux[b])
        for i in range(M):
            if not ok[i]:
                continue
            x = flux[b][ok & (np.abs(k - k[i]) <= h)].astype(np.float64)
            if x.size < min_valid:
                continue
            trend[b, i], median[b, i], _ = location(x, alpha, c, n_iter)
    return trend, median


def detrend_gapped_ex(time, flux, t0, dt, n_grid, W, alpha=2.0, n_iter=5, c=5.0, min_valid=None,
                      break_slots=-1, min_segment=0, edge_cut=0):
    """Brute force for the segmented gap handling (reading R23), written with whole-row masks and
    np.split instead of the oracle's running counters: valid samples (as in detrend_gapped) are cut
    where np.diff(slot) - 1 > break_slots, pieces shorter than min_segment are thrown away, a window
    is the piece's samples within h slots, samples closer than edge_cut slots to a piece's end get NaN."""
    time = np.atleast_2d(np.asarray(time, dtype=np.float64))
    flux = np.atleast_2d(np.asarray(flux, dtype=np.float32))
    S, M = flux.shape
    h = (W - 1) // 2
    if min_valid is None:
        min_valid = max(1, W // 3)
    trend = np.full((S, M), np.nan)
    median = np.full((S, M), np.nan)
    for b in range(S):
        with np.errstate(invalid="ignore"):
            k = np.rint((time[b] - t0) / dt)
        ok = np.isfinite(time[b]) & (k >= 0) & (k < n_grid)
        same_as_next = np.zeros(M, dtype=bool)
        same_as_next[:-1] = np.isfinite(time[b, :-1]) & np.isfinite(time[b, 1:]) & (k[:-1] == k[1:])
        ok &= ~same_as_next & np.isfinite(flux[b])
        idx = np.flatnonzero(ok)
        if idx.size == 0:
            continue
        ks = k[idx].astype(np.int64)
        cuts = np.flatnonzero(np.diff(ks) - 1 > break_slots) + 1 if break_slots >= 0 else np.array([], dtype=np.int64)
        for piece_idx, piece_k in zip(np.split(idx, cuts), np.split(ks, cuts)):
            if piece_idx.size < min_segment:
                continue
            x_all = flux[b][piece_idx].astype(np.float64)
            for i, ki in zip(piece_idx, piece_k):
                if ki - piece_k[0] < edge_cut or piece_k[-1] - ki < edge_cut:
                    continue
                x = x_all[np.abs(piece_k - ki) <= h]
                if x.size < min_valid:
                    continue
                trend[b, i], median[b, i], _ = location(x, alpha, c, n_iter)
    return trend, median


def location_family(x, scale_kind="upper_rms", weight_kind="bisquare", alpha=2.0, c=5.0, n_iter=5):
    """Sibling estimators (F4): scale_kind "mad" = np.median-style MAD (lower middle, R21),
    weight_kind "welsch" = exp(-u_eff^2) (R22).  Returns (mu, median, s)."""
    x = np.asarray(x, dtype=np.float64)
    n = x.size
    med = np.sort(x)[(n - 1) // 2]
    if scale_kind == "mad":
        s = np.sort(np.abs(x - med))[(n - 1) // 2]
    else:
        upper = x[x > med]
        if upper.size == 0:
            return med, med, 0.0
        s = SCALE_CONST * np.sqrt(np.mean((upper - med) ** 2))
    if not s > 0.0:
        return med, med, s
    mu = med
    for _ in range(n_iter):
        u = (x - mu) / (c * s)
        if weight_kind == "welsch":
            u_eff = np.where(u < 0.0, alpha * u, u)
            w = np.exp(-u_eff ** 2)
        else:
            w = bisquare_weights(u, alpha)
        if not w.sum() > 0.0:
            break
        mu = np.average(x, weights=w)
    return mu, med, s
