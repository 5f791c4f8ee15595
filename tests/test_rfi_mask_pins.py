"""Pins for the coincidence-RFI-mask oracle (no GPU): hand-worked numbers, a literal loop,
and the paper's printed false-positive bound (Sec. 2.1)."""
from math import comb
from pathlib import Path

import numpy as np

from oracle import rfi_mask as RM

GOLDEN = Path(__file__).resolve().parent / "golden"


def _read():
    d, xs = {}, []
    for line in (GOLDEN / "rfi_mask_hand.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        if p[0] == "x":
            xs.append([float(v) for v in p[1:]])
        else:
            d[p[0]] = [float(v) for v in p[1:]]
    d["x"] = np.array(xs, dtype=np.float32)[:, None, :]
    return d


def test_hand_worked_example():
    d = _read()
    nb = d["x"].shape[0]
    mean = np.full((nb, 1), d["mean"][0], np.float32)
    sigma = np.full((nb, 1), d["sigma"][0], np.float32)
    assert RM.beam_count(d["x"], mean, sigma, d["nsigma"][0])[0].tolist() == [int(v) for v in d["count"]]
    got = RM.coincidence_mask(d["x"], mean, sigma, d["nsigma"][0], int(d["min_beams"][0]))
    assert got.dtype == np.uint8 and got[0].tolist() == [int(v) for v in d["mask"]]


def test_literal_loop():
    rng = np.random.default_rng(4)
    x = rng.standard_normal((5, 3, 400)).astype(np.float32)
    x[2, 1, 7] = np.nan
    mean = (0.1 * rng.standard_normal((5, 3))).astype(np.float32)
    sigma = (0.5 + rng.random((5, 3))).astype(np.float32)
    got = RM.coincidence_mask(x, mean, sigma, 1.0, 2)
    for s in range(3):
        for t in range(400):
            k = 0
            for b in range(5):
                thr = np.float32(mean[b, s] + np.float32(np.float32(1.0) * sigma[b, s]))
                if x[b, s, t] > thr:
                    k += 1
            assert got[s, t] == (1 if k >= 2 else 0)


def test_paper_false_positive_bound():
    """PAPER.md:40 prints p <= C(13,4) x 0.01^4 = 7.15e-6: the union bound on the exact binomial
    tail; the oracle's mask rate on noise with a 1 % single-beam exceedance must obey both."""
    d = _read()
    nb, k, p = int(d["paper_nbeams"][0]), int(d["paper_min_beams"][0]), d["paper_p_single"][0]
    bound = comb(nb, k) * p ** k
    assert abs(bound - d["paper_bound"][0]) < 5e-9                     # 715e-8 = 7.15e-6 as printed
    tail = sum(comb(nb, i) * p ** i * (1 - p) ** (nb - i) for i in range(k, nb + 1))
    assert tail <= bound and abs(tail - 6.652e-6) < 0.001e-6     # 6.5316e-6 + 1.188e-7 + 1.6e-9 by hand
    # uniform noise on [0,1): x > 0.8 has probability exactly 0.2 (rates large enough to measure)
    rng = np.random.default_rng(12)
    n = 200_000
    x = rng.random((nb, 1, n)).astype(np.float32)
    zero, one = np.zeros((nb, 1), np.float32), np.ones((nb, 1), np.float32)
    rate = RM.coincidence_mask(x, zero, one, 0.8, k).mean()
    q = 0.2
    tail_q = sum(comb(nb, i) * q ** i * (1 - q) ** (nb - i) for i in range(k, nb + 1))
    assert abs(rate - tail_q) < 4 * np.sqrt(tail_q * (1 - tail_q) / n)
    assert rate <= comb(nb, k) * q ** k


def test_monotone_in_min_beams_and_limits():
    rng = np.random.default_rng(2)
    x = rng.standard_normal((13, 2, 1000)).astype(np.float32)
    z, o = np.zeros((13, 2), np.float32), np.ones((13, 2), np.float32)
    prev = None
    for k in range(0, 15):
        m = RM.coincidence_mask(x, z, o, 0.5, k)
        if prev is not None:
            assert np.all(m <= prev)
        prev = m
    assert np.all(RM.coincidence_mask(x, z, o, 0.5, 0) == 1)
    assert np.all(RM.coincidence_mask(x, z, o, 0.5, 14) == 0)
    np.testing.assert_array_equal(RM.coincidence_mask(x, z, o, 0.5, 1), (x > 0.5).any(axis=0))
    np.testing.assert_array_equal(RM.coincidence_mask(x, z, o, 0.5, 13), (x > 0.5).all(axis=0))


def test_veto_events_hand_worked():
    # reading R39: an event is vetoed when its PEAK sample is masked; series -> -1 - series, order kept
    from oracle import peak_finding as PF
    ev = np.zeros(4, dtype=PF.EVENT_DTYPE)
    ev["series"] = [0, 0, 3, 5]
    ev["t_start"] = [2, 10, 4, 7]
    ev["length"] = [3, 1, 4, 2]
    ev["t_peak"] = [3, 10, 7, 8]
    mask = np.zeros(12, np.uint8)
    mask[[2, 7, 10]] = 1                     # t_start of event 0 is masked, its peak (3) is not
    out, kept = RM.veto_events(ev, mask)
    assert kept == 2 and out["series"].tolist() == [0, -1, -4, 5]
    assert np.array_equal(out["t_peak"], ev["t_peak"]) and ev["series"].tolist() == [0, 0, 3, 5]
    out2, kept2 = RM.veto_events(out, np.ones(12, np.uint8))      # vetoed events stay vetoed, are not counted
    assert kept2 == 0 and out2["series"].tolist() == [-1, -1, -4, -6]


def test_counts_of_beam_subsets_add_up_to_the_coincidence_mask():
    # the multi-GPU form: counts of disjoint beam subsets summed, then thresholded == the mask over all beams
    rng = np.random.default_rng(11)
    x = rng.standard_normal((13, 2, 500)).astype(np.float32)
    mean, sigma = rng.normal(0, 0.1, (13, 2)).astype(np.float32), rng.uniform(0.8, 1.2, (13, 2)).astype(np.float32)
    total = sum(RM.beam_count(x[a:b], mean[a:b], sigma[a:b], 1.0) for a, b in ((0, 4), (4, 9), (9, 13)))
    assert np.array_equal(total, RM.beam_count(x, mean, sigma, 1.0))
    assert np.array_equal((total >= 4).astype(np.uint8), RM.coincidence_mask(x, mean, sigma, 1.0, 4))
