"""CPU oracle for baseline removal + boxcar matched filtering -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs may import
this module; the product (``paper_1112_0065_b200``) never does, and nothing here
imports the product.  It shares no code with the CUDA path.

What it computes (Sec. 2.3), following
the paper's algorithm step by step:

  1. "compute a running mean for the data with a given window size (equivalent to
     convolving with a wide boxcar) and then subtracting this off the original
     data ... exploit a parallel prefix sum ... the running mean may be calculated
     by subtracting the points at plus and minus the window radius":

         S[k]  = sum_{t<k} x[t]                          (exclusive prefix sum)
         a(t)  = min(max(t - R, 0), n - N),   N = 2R + 1 (readings R21, R22)
         m[t]  = (S[a(t)+N] - S[a(t)]) / N
         y[t]  = x[t] - m[t]

  2. "convolving the time series with boxcar functions of increasing sizes (e.g.,
     2, 4, 8 etc. samples) ... implemented in the same manner using the parallel
     prefix sum":

         P[k]   = sum_{t<k} y[t]
         z_w[t] = (P[t+w] - P[t]) / sqrt(w)   for 0 <= t <= n - w,   0 otherwise
                                               (readings R24, R25)

The paper gives no window radius, no edge rule, no boxcar alignment and no
normalisation; the readings are listed in DESIGN.md ("Readings", R21-R26).

Arithmetic: x is an array of non-negative integers (dedispersed sums < 2**24).
N*y[t] = N*x[t] - (S[a+N] - S[a]) and its prefix sums are exact in int64, so the
only rounding is the final division by N*sqrt(w) in float64.

Pins (tests/test_matched_filter_pins.py, tests/golden/matched_filter_hand.txt):
hand-worked example, brute force from the definition with exact fractions,
numpy.convolve (a library routine that does not use prefix sums) on the interior,
constant input, linear ramp, impulse response closed form, width-1 identity,
white-noise variance.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def _as_rows(x) -> np.ndarray:
    x = np.asarray(x)
    if x.ndim == 1:
        x = x[None, :]
    if x.ndim != 2:
        raise ValueError("x must be [n] or [nrows, n]")
    if np.issubdtype(x.dtype, np.floating):
        xi = x.astype(np.int64)
        if not np.array_equal(xi, x):
            raise ValueError("float input must hold exact integers")
        x = xi
    return x.astype(np.int64)


def window_start(n: int, radius: int) -> np.ndarray:
    """a(t): first sample of the running-mean window of sample t (readings R21, R22)."""
    N = 2 * radius + 1
    if radius < 0 or N > n:
        raise ValueError("need 0 <= radius and 2*radius+1 <= n")
    return np.clip(np.arange(n) - radius, 0, n - N)


def baseline_numerator(x, radius: int) -> np.ndarray:
    """N*y[t] = N*x[t] - sum of the window of t, exact int64 (step 1 above)."""
    x = _as_rows(x)
    n = x.shape[1]
    N = 2 * radius + 1
    a = window_start(n, radius)
    S = np.zeros((x.shape[0], n + 1), dtype=np.int64)
    np.cumsum(x, axis=1, out=S[:, 1:])            # prefix sum
    W = S[:, a + N] - S[:, a]                     # points at plus and minus the radius
    return N * x - W


def running_mean(x, radius: int) -> np.ndarray:
    """m[t] in float64."""
    x = _as_rows(x)
    N = 2 * radius + 1
    return (N * x - baseline_numerator(x, radius)) / float(N)


def baseline_removed(x, radius: int) -> np.ndarray:
    """y[t] = x[t] - m[t] in float64 (one rounding: exact numerator / N)."""
    return baseline_numerator(x, radius) / float(2 * radius + 1)


def matched_filter(x, radius: int, widths) -> np.ndarray:
    """z[w_index][row][t] in float64 (steps 1 and 2 above)."""
    x = _as_rows(x)
    nrows, n = x.shape
    N = 2 * radius + 1
    Y = baseline_numerator(x, radius)
    P = np.zeros((nrows, n + 1), dtype=np.int64)
    np.cumsum(Y, axis=1, out=P[:, 1:])
    out = np.zeros((len(widths), nrows, n), dtype=np.float64)
    for i, w in enumerate(widths):
        w = int(w)
        if w < 1 or w > n:
            raise ValueError("need 1 <= width <= n")
        Z = P[:, w:] - P[:, : n + 1 - w]          # t = 0 .. n-w
        out[i, :, : n + 1 - w] = Z / (float(N) * np.sqrt(float(w)))
    return out
