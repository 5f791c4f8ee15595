"""Pins for the time-major -> channel-major oracle (no GPU)."""
import numpy as np
import pytest

import oracle
from oracle import time_major as TM
import workloads as W


def test_hand_typed_bytes():
    # 2-bit, 4 channels, 3 time samples: one byte per time sample, channel 0 in the low bits.
    #   t0: c0=1 c1=2 c2=3 c3=0 -> 0b00_11_10_01 = 0x39;  t1: 3,0,1,2 -> 0b10_01_00_11 = 0x93
    #   t2: 2,2,0,1 -> 0b01_00_10_10 = 0x4a
    got = TM.to_channel_major(np.array([0x39, 0x93, 0x4A], np.uint8), 4, 3, 2)
    # rows: c0 = 1,3,2 -> 0b10_11_01 = 0x2d; c1 = 2,0,2 -> 0b10_00_10 = 0x22; c2 = 3,1,0 -> 0x07; c3 = 0,2,1 -> 0x18
    assert got.tolist() == [[0x2D], [0x22], [0x07], [0x18]]
    # 1-bit, 8 channels, 2 time samples: t0 = 0xb1 (c0,c4,c5,c7 set), t1 = 0x03 (c0,c1 set)
    got = TM.to_channel_major(np.array([0xB1, 0x03], np.uint8), 8, 2, 1)
    assert got[:, 0].tolist() == [3, 2, 0, 0, 1, 1, 0, 1]


@pytest.mark.parametrize("nbits,nchans,nsamps", [(1, 8, 13), (2, 12, 9), (4, 6, 7), (8, 3, 5), (2, 64, 131)])
def test_literal_bit_loop(nbits, nchans, nsamps):
    rng = np.random.default_rng(nbits * 100 + nchans)
    stream = rng.integers(0, 256, nsamps * nchans * nbits // 8, dtype=np.uint8)
    got = TM.to_channel_major(stream, nchans, nsamps, nbits)
    stride = (nsamps * nbits + 7) // 8
    want = np.zeros((nchans, stride), np.uint8)
    for t in range(nsamps):
        for c in range(nchans):
            for k in range(nbits):
                src = (t * nchans + c) * nbits + k
                bit = (stream[src >> 3] >> (src & 7)) & 1
                dst = t * nbits + k
                want[c, dst >> 3] |= bit << (dst & 7)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("nbits", [1, 2, 4, 8])
def test_dedispersing_the_transposed_stream_equals_the_channel_major_original(nbits):
    nchans, nsamps = 16, 300
    cm = W.random_small(5 + nbits, nchans, nsamps, nbits)
    lev = np.stack([W.unpack_bits(cm[c], nbits, nsamps) for c in range(nchans)])       # [c][t]
    stream = W.pack_bits(lev.T.reshape(-1), nbits)                                       # [t][c]
    back = TM.to_channel_major(stream, nchans, nsamps, nbits)
    assert np.array_equal(back, cm)
    delay = np.sort(np.random.default_rng(1).integers(0, 40, (nchans, 5)), axis=1).astype(np.int32)
    assert np.array_equal(oracle.dedisperse(delay, back, nbits, 200), oracle.dedisperse(delay, cm, nbits, 200))
