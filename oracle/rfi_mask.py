"""CPU oracle for the multibeam coincidence RFI mask -- TEST INFRASTRUCTURE ONLY.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs may import this module;
the product never does and nothing here imports the product.

What it computes (Sec. 2.1: "apply signal-to-noise
and coincidence thresholds ... 'a signal exceeding 3 sigma in 4 or more beams' ... a transform
of the multibeam time series, where for each sample the 13 beams are checked against the
thresholds and the result is written as a boolean RFI mask"):

    above[b][s][t] = x[b][s][t] > fl32( mean[b][s] + fl32( nsigma * sigma[b][s] ) )
    mask[s][t]     = ( number of beams b with above[b][s][t] )  >=  min_beams

x holds nseries time series per beam (e.g. the DM-0 trial of every beam, or one series per
channel); mean and sigma are inputs per (beam, series) -- the paper leaves their estimate
unspecified (readings R32-R35 in DESIGN.md).  The threshold is formed in float32 (the type
of x), the comparison is strict, NaN is never above.  Everything is comparisons and a
count: exactly one result is correct, parity is exact.

Pins (tests/test_rfi_mask_pins.py, tests/golden/rfi_mask_hand.txt): hand-worked example, a
literal per-sample loop, the paper's printed false-positive bound C(13,4) x 0.01^4 =
7.15e-6 against the exact binomial tail and against the oracle run on seeded uniform
noise, monotonicity in min_beams.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def thresholds(mean, sigma, nsigma) -> np.ndarray:
    """fl32(mean + fl32(nsigma * sigma)), shape [nbeams, nseries]."""
    mean = np.asarray(mean, dtype=np.float32)
    sigma = np.asarray(sigma, dtype=np.float32)
    return (mean + (np.float32(nsigma) * sigma).astype(np.float32)).astype(np.float32)


def beam_count(x, mean, sigma, nsigma) -> np.ndarray:
    """Number of beams above threshold, int32 [nseries, n]."""
    x = np.asarray(x, dtype=np.float32)
    if x.ndim != 3:
        raise ValueError("x must be [nbeams, nseries, n]")
    thr = thresholds(mean, sigma, nsigma)
    if thr.shape != x.shape[:2]:
        raise ValueError("mean/sigma must be [nbeams, nseries]")
    with np.errstate(invalid="ignore"):
        return (x > thr[:, :, None]).sum(axis=0).astype(np.int32)


def coincidence_mask(x, mean, sigma, nsigma, min_beams) -> np.ndarray:
    """uint8 [nseries, n]: 1 where at least min_beams beams exceed their threshold."""
    return (beam_count(x, mean, sigma, nsigma) >= int(min_beams)).astype(np.uint8)


def veto_events(events: np.ndarray, mask_row: np.ndarray) -> tuple[np.ndarray, int]:
    """A consumer of the mask (reading R39): an event whose PEAK sample is flagged in ``mask_row``
    (uint8 [n], one series of the mask) is vetoed -- its ``series`` becomes ``-1 - series`` (order kept).
    Returns (events with vetoes marked, number of events kept).  Events already vetoed stay so and are not counted."""
    out = events.copy()
    kept = 0
    for i in range(len(out)):
        s = int(out["series"][i])
        if s < 0:
            continue
        if mask_row[int(out["t_peak"][i])]:
            out["series"][i] = -1 - s
        else:
            kept += 1
    return out, kept
