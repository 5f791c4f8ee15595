"""CPU oracle for the time-major -> channel-major input transpose -- TEST INFRASTRUCTURE ONLY
(same import rules as the rest of ``oracle/``).

What it computes ("filterbank" data as the telescope
writes it; reading R37): telescope-order filterbank data holds, for every time
sample, all channels next to each other,

    sample (t, c) = bits [ (t*nchans + c)*nbits , +nbits ) of the stream, LSB-first,

while dedisp_execute wants one tight row per channel (readings R9, R10),

    sample (c, t) = bits [ t*nbits , +nbits ) of row c,  rows of ceil(nsamps*nbits/8) bytes,
    unused high bits of the last byte zero.

A pure re-layout: exactly one output is correct, parity is exact.  Steps: numpy.unpackbits
(little bit order) -> reshape [nsamps, nchans, nbits] -> transpose -> numpy.packbits per row.

Pins (tests/test_time_major_pins.py): hand-typed bytes, a literal bit-by-bit loop, and
dedispersing the transposed data == dedispersing the channel-major original.
"""
from __future__ import annotations

import numpy as np


def to_channel_major(stream: np.ndarray, nchans: int, nsamps: int, nbits: int) -> np.ndarray:
    """uint8 [nchans, ceil(nsamps*nbits/8)] from the time-major byte stream."""
    if nbits not in (1, 2, 4, 8) or (nchans * nbits) % 8:
        raise ValueError("need nbits in 1/2/4/8 and whole bytes per time sample")
    stream = np.ascontiguousarray(stream, dtype=np.uint8).reshape(-1)
    need = nsamps * nchans * nbits // 8
    if stream.size < need:
        raise ValueError("stream too short")
    bits = np.unpackbits(stream[:need], bitorder="little").reshape(nsamps, nchans, nbits)
    rows = bits.transpose(1, 0, 2).reshape(nchans, nsamps * nbits)
    return np.ascontiguousarray(np.packbits(rows, axis=1, bitorder="little"))   # zero-pads the last byte
