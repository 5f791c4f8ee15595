"""Pins for the time-scrunch oracle (row f4, reading R38; no GPU)."""
import numpy as np
import pytest

import oracle
from oracle import tscrunch as TS
import workloads as W

# the hand-worked example of SURVEY.md Sec. 8(c) (4 channels, f_top 1500, df -100, DMs 0/10/25),
# rows of 32 two-bit samples, digits = samples t = 0..31
HAND_ROWS = ["00123112210323301010313010001232", "03223323011210301101113222230111",
             "30021003222332100112130230003221", "00120122033202211333122202230022"]


def _hand_packed():
    return np.stack([W.pack_bits(np.array([int(ch) for ch in r], np.uint8), 2) for r in HAND_ROWS])


def test_hand_worked_example():
    # dt' = 2 * 1 ms: x' = x / 2 -> ch1 {0, 1.364.., 3.410..}, ch2 {0, 3.055.., 7.637..}, ch3 {0, 5.18601, 12.965025}
    delay, md = oracle.delay_table(4, 2e-3, 1500.0, -100.0, [0.0, 10.0, 25.0])
    assert delay.tolist() == [[0, 0, 0], [0, 1, 3], [0, 3, 8], [0, 5, 13]] and md == 13
    packed = _hand_packed()
    # pairs summed by hand: ch0 "00 12 31 12 21 03 23 30 10 10 31 30 10 00 12 32" -> 0 3 4 3 3 3 5 3 1 1 4 3 1 0 3 5
    s = TS.scrunch_rows(packed, 2, 2, 16)
    assert s.tolist() == [[0, 3, 4, 3, 3, 3, 5, 3, 1, 1, 4, 3, 1, 0, 3, 5], [3, 4, 6, 5, 1, 3, 1, 3, 2, 1, 2, 5, 4, 5, 1, 2],
                          [3, 2, 1, 3, 4, 5, 5, 1, 1, 3, 4, 2, 3, 0, 5, 3], [0, 3, 1, 4, 3, 5, 2, 3, 4, 6, 3, 4, 2, 5, 0, 4]]
    # out[1][0] = s0[0] + s1[1] + s2[3] + s3[5] = 0 + 4 + 3 + 5; out[2][1] = s0[1] + s1[4] + s2[9] + s3[14] = 3 + 1 + 3 + 0
    want = [[6, 12, 12], [12, 15, 17], [11, 7, 15]]
    assert TS.dedisperse_tscrunch(delay, packed, 2, 2, 3).tolist() == want
    assert TS.dedisperse_tscrunch_bytes(delay, packed, 2, 2, 3).tolist() == want


@pytest.mark.parametrize("nbits,k", [(1, 2), (1, 16), (2, 2), (2, 4), (2, 3), (4, 2), (4, 8), (8, 2)])
def test_literal_loop_on_the_packed_bytes(nbits, k):
    nchans, ndm, nout = 5, 4, 11
    rng = np.random.default_rng(10 * nbits + k)
    delay = np.sort(rng.integers(0, 9, (nchans, ndm)), axis=1).astype(np.int32)
    n_scr = nout + int(delay.max())
    packed = W.random_small(77 + k, nchans, n_scr * k, nbits)
    want = np.zeros((ndm, nout), np.uint32)
    for d in range(ndm):
        for t in range(nout):
            for c in range(nchans):
                for j in range(k):
                    bit = (k * (t + int(delay[c, d])) + j) * nbits
                    want[d, t] += (int(packed[c, bit >> 3]) >> (bit & 7)) & ((1 << nbits) - 1)
    assert np.array_equal(TS.dedisperse_tscrunch(delay, packed, nbits, k, nout), want)
    if k * ((1 << nbits) - 1) <= 255:
        assert np.array_equal(TS.dedisperse_tscrunch_bytes(delay, packed, nbits, k, nout), want)


@pytest.mark.parametrize("nbits", [1, 2, 4, 8])
def test_factor_one_is_plain_dedispersion(nbits):
    nchans, nout = 12, 90
    delay = np.sort(np.random.default_rng(3).integers(0, 30, (nchans, 6)), axis=1).astype(np.int32)
    packed = W.random_small(9 + nbits, nchans, nout + int(delay.max()), nbits)
    assert np.array_equal(TS.dedisperse_tscrunch(delay, packed, nbits, 1, nout),
                          oracle.dedisperse_literal(delay, packed, nbits, nout))


@pytest.mark.parametrize("nbits,k", [(2, 2), (2, 8), (1, 4), (4, 4)])
def test_adjacent_full_resolution_outputs_add_up(nbits, k):
    # if every full-resolution delay is exactly k times the coarse one, a coarse output sample is
    # the sum of the k full-resolution output samples it covers (pinned C oracle on the fine grid)
    nchans, nout = 10, 40
    delay = np.sort(np.random.default_rng(k).integers(0, 12, (nchans, 5)), axis=1).astype(np.int32)
    packed = W.random_small(31 + k, nchans, k * (nout + int(delay.max())), nbits)
    fine = oracle.dedisperse(delay * k, packed, nbits, k * nout)
    want = fine.reshape(5, nout, k).sum(axis=2)
    assert np.array_equal(TS.dedisperse_tscrunch(delay, packed, nbits, k, nout), want)


def test_constant_input_and_zero_dm():
    nchans, nout, k = 7, 20, 4
    delay = np.sort(np.random.default_rng(2).integers(0, 6, (nchans, 3)), axis=1).astype(np.int32)
    delay[:, 0] = 0
    n = k * (nout + int(delay.max()))
    packed = np.stack([W.pack_bits(np.full(n, 3, np.uint8), 2)] * nchans)
    assert (TS.dedisperse_tscrunch(delay, packed, 2, k, nout) == 3 * k * nchans).all()
    packed = W.random_small(5, nchans, n, 2)
    lev = np.stack([W.unpack_bits(packed[c], 2, n) for c in range(nchans)]).astype(np.int64)
    # DM 0: the channel sum, summed in blocks of k
    assert np.array_equal(TS.dedisperse_tscrunch(delay, packed, 2, k, nout)[0],
                          lev.sum(axis=0)[: k * nout].reshape(nout, k).sum(axis=1))


def test_coarse_delays_track_the_fine_ones():
    # delay' = round(x / k) with x the unrounded fine delay: |k delay' - delay| <= (k + 1) / 2
    dms = np.linspace(0, 1000, 50)
    fine, _ = oracle.delay_table(1024, 64e-6, 1581.8, -0.390625, dms)
    for k in (2, 4, 16):
        coarse, _ = oracle.delay_table(1024, k * 64e-6, 1581.8, -0.390625, dms)
        assert np.abs(k * coarse.astype(np.int64) - fine).max() <= (k + 1) / 2
