"""CPU oracle for peak finding (sigma-cut + grouping of contiguous regions) -- TEST
INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU
legs may import this module; the product never does and nothing here imports the product.

What it computes (Sec. 2.3: "detect peaks in the
reduced time series ... by first performing a sigma-cut and then gathering contiguous
regions together into individual events.  These algorithms map to the 'transform' and
'reduce_by_key' functions"), in the paper's order:

  1. transform (sigma-cut):  m[s][t] = z[s][t] > nsigma * sigma[s]
     -- strict '>', the product taken in float32 (the type of z), NaN is never above
     (readings R27, R28: sigma[s] is an input; ``series_rms`` is the estimate offered);
  2. reduce by key: every maximal run of consecutive samples of ONE series with m true is
     one event (runs never join across series; reading R29), reduced to
         (series, t_start, length, t_peak, peak)
     with peak = max of z over the run and t_peak its FIRST position (reading R30);
     events are listed in ascending (series, t_start) order (reading R31).

The paper gives no threshold, no sigma estimator and no event record; the readings are
listed in DESIGN.md (R27-R31).  Everything here is comparisons of float32 values and
integer bookkeeping: exactly one result is correct, parity is exact.

Pins (tests/test_peak_finding_pins.py, tests/golden/peak_finding_hand.txt): hand-worked
example, a literal sample-by-sample state machine, run-length identities against
numpy, edge cases (run at either end, whole series, equal maxima, NaN, value equal to
the threshold, adjacent series).  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

EVENT_DTYPE = np.dtype([("series", np.int32), ("t_start", np.int32), ("length", np.int32),
                        ("t_peak", np.int32), ("peak", np.float32)])


def sigma_cut(z, sigma, nsigma) -> np.ndarray:
    """Step 1: boolean mask [nseries, n]."""
    z = np.asarray(z, dtype=np.float32)
    thr = np.float32(nsigma) * np.asarray(sigma, dtype=np.float32)       # float32 product
    with np.errstate(invalid="ignore"):
        return z > thr[:, None]


def find_events(z, sigma, nsigma) -> np.ndarray:
    """Steps 1 and 2: structured array of events in (series, t_start) order."""
    z = np.asarray(z, dtype=np.float32)
    m = sigma_cut(z, sigma, nsigma)
    out = []
    for s in range(z.shape[0]):
        # run boundaries: +1 where a run starts, -1 one past where it ends
        edge = np.diff(np.concatenate(([0], m[s].astype(np.int8), [0])))
        starts = np.flatnonzero(edge == 1)
        ends = np.flatnonzero(edge == -1)
        for a, b in zip(starts, ends):
            k = int(np.argmax(z[s, a:b]))                                 # first maximum
            out.append((s, a, b - a, a + k, z[s, a + k]))
    return np.array(out, dtype=EVENT_DTYPE)


def series_rms(z) -> np.ndarray:
    """sqrt(mean(z^2)) per series in float64 (the sigma estimate of reading R28)."""
    z = np.asarray(z, dtype=np.float64)
    return np.sqrt(np.mean(z * z, axis=1))
