"""CPU oracle for dedispersion at reduced time resolution ("time scrunching") -- TEST
INFRASTRUCTURE ONLY (same import rules as the rest of ``oracle/``).

What it computes (SURVEY.md Sec. 8(f) row f4 "per-DM-range time scrunching"; DESIGN.md reading
R38).  The paper does not describe the step (PAPER.md:44 only says that ~1200 trial DMs are
searched); the reading taken is the usual one: for a range of trial DMs whose dispersion smearing
inside one channel exceeds the sampling time, every channel's series is first summed in
non-overlapping blocks of k samples, block 0 starting at sample 0, and the trials of that range are
dedispersed on the coarser grid dt' = k*dt with delays computed from dt' by the rule of reading R3:

    s[c][u]   = sum_{j<k} in[c][k*u + j]                              (raw sums, no division: R13)
    out[d][t] = sum_c s[c][t + delay'[c][d]],   delay' = oracle.delay_table(nchans, k*dt, ...)

Exact unsigned integers; exactly one output is correct; parity is ``array_equal``.

``dedisperse_tscrunch`` is that definition written out (numpy unpack, reshape-sum, a plain
``for d: for c:`` slice sum).  ``dedisperse_tscrunch_bytes`` is the same thing for larger parity
cases: the scrunched rows (values <= 255) handed to the pinned C oracle as 8-bit samples.

Pins (tests/test_tscrunch_pins.py): a hand-worked example, a literal quadruple loop on the packed
bytes, k = 1 == plain dedispersion, "k adjacent full-resolution outputs add up" when the
full-resolution delays are k times the scrunched ones, constant input, both functions equal.
"""
from __future__ import annotations

import numpy as np

import oracle


def unpack_row(row: np.ndarray, nbits: int, nsamps: int) -> np.ndarray:
    """Samples 0..nsamps-1 of a tight LSB-first row (readings R10, R36) as uint8."""
    if nbits == 8:
        return np.asarray(row[:nsamps], dtype=np.uint8)
    bits = np.unpackbits(np.asarray(row, dtype=np.uint8), bitorder="little")[: nsamps * nbits]
    weights = (1 << np.arange(nbits)).astype(np.uint8)
    return (bits.reshape(nsamps, nbits) * weights).sum(axis=1).astype(np.uint8)


def scrunch_rows(packed: np.ndarray, nbits: int, k: int, nsamps_scr: int) -> np.ndarray:
    """s[c][u] = sum of samples k*u .. k*u+k-1 of row c, u < nsamps_scr; uint32 [nchans, nsamps_scr]."""
    if nbits not in (1, 2, 4, 8) or k < 1 or nsamps_scr < 1:
        raise ValueError("bad nbits / k / nsamps")
    packed = np.asarray(packed, dtype=np.uint8)
    if packed.ndim != 2 or packed.shape[1] * 8 < nsamps_scr * k * nbits:
        raise ValueError("packed rows too short")
    out = np.empty((packed.shape[0], nsamps_scr), dtype=np.uint32)
    for c in range(packed.shape[0]):
        out[c] = unpack_row(packed[c], nbits, nsamps_scr * k).reshape(nsamps_scr, k).sum(axis=1, dtype=np.uint32)
    return out


def dedisperse_tscrunch(delay_scr: np.ndarray, packed: np.ndarray, nbits: int, k: int,
                        nsamps_out: int) -> np.ndarray:
    """out[d][t] = sum_c s[c][t + delay_scr[c][d]]; uint32 [ndm, nsamps_out].

    ``delay_scr`` is the delay table of the coarse grid (in scrunched samples); ``packed`` holds
    nchans tight rows of k*(nsamps_out + max(delay_scr)) samples of ``nbits`` bits."""
    delay_scr = np.asarray(delay_scr, dtype=np.int64)
    nchans, ndm = delay_scr.shape
    if delay_scr.min() < 0:
        raise ValueError("negative delay")
    n_scr = nsamps_out + int(delay_scr.max())
    s = scrunch_rows(packed, nbits, k, n_scr)
    if s.shape[0] != nchans:
        raise ValueError("row count != nchans")
    out = np.zeros((ndm, nsamps_out), dtype=np.uint32)
    for d in range(ndm):
        for c in range(nchans):
            o = int(delay_scr[c, d])
            out[d] += s[c, o:o + nsamps_out]
    return out


def dedisperse_tscrunch_bytes(delay_scr: np.ndarray, packed: np.ndarray, nbits: int, k: int,
                              nsamps_out: int, **kw) -> np.ndarray:
    """Same result through the C oracle: the scrunched rows are 8-bit samples (needs k*(2^nbits-1) <= 255)."""
    if k * ((1 << nbits) - 1) > 255:
        raise ValueError("scrunched samples do not fit a byte")
    delay_scr = np.ascontiguousarray(delay_scr, dtype=np.int32)
    n_scr = nsamps_out + int(delay_scr.max())
    s = np.ascontiguousarray(scrunch_rows(packed, nbits, k, n_scr).astype(np.uint8))
    return oracle.dedisperse(delay_scr, s, 8, nsamps_out, **kw)
