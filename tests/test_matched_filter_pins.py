"""Pins for the baseline-removal + boxcar oracle (no GPU).  Each test fixes
``oracle.matched_filter`` to something other than itself: hand-worked numbers,
brute force from the definition in exact fractions, numpy.convolve (no prefix
sums), closed forms (constant, ramp, impulse) and a white-noise variance check.

Definition under test (Sec. 2.3; readings R21-R26):
    y[t]   = x[t] - mean(x[a(t) : a(t)+N]),  N = 2R+1,  a(t) = clip(t-R, 0, n-N)
    z_w[t] = sum(y[t : t+w]) / sqrt(w)  for t <= n-w,  0 beyond
"""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

from oracle import matched_filter as MF

GOLDEN = Path(__file__).resolve().parent / "golden"


def _brute(x, R, widths):
    """The definition, literally, in exact fractions (tiny inputs only)."""
    n, N = len(x), 2 * R + 1
    y = []
    for t in range(n):
        a = min(max(t - R, 0), n - N)
        y.append(Fraction(int(x[t])) - Fraction(sum(int(v) for v in x[a:a + N]), N))
    out = []
    for w in widths:
        row = [float(sum(y[t:t + w], Fraction(0))) / np.sqrt(float(w)) if t + w <= n else 0.0
               for t in range(n)]
        out.append(row)
    return np.array(y, dtype=object), np.array(out)


def _read_hand():
    d = {"widths": {}}
    for line in (GOLDEN / "matched_filter_hand.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        if p[0] == "width":
            d["widths"][int(p[1])] = [int(v) for v in p[3:]]
        elif p[0] == "radius":
            d["radius"] = int(p[1])
        else:
            d[p[0]] = [int(v) for v in p[1:]]
    return d


def test_hand_worked_example():
    h = _read_hand()
    x, R = np.array(h["x"]), h["radius"]
    N = 2 * R + 1
    assert list(MF.window_start(len(x), R)) == h["window_start"]
    num = MF.baseline_numerator(x, R)[0]
    assert list(num) == h["num_y"]
    assert list(N * x - num) == h["window_sum"]
    ws = sorted(h["widths"])
    z = MF.matched_filter(x, R, ws)
    for i, w in enumerate(ws):
        want = np.zeros(len(x))
        want[: len(h["widths"][w])] = np.array(h["widths"][w]) / (N * np.sqrt(w))
        np.testing.assert_allclose(z[i, 0], want, rtol=1e-15, atol=0)
        assert np.all(z[i, 0, len(x) - w + 1:] == 0.0)


@pytest.mark.parametrize("n,R,widths,seed", [(16, 0, [1, 2, 3], 1), (23, 3, [1, 2, 4, 8, 23], 2),
                                             (40, 19, [1, 5, 16], 3), (9, 4, [9], 4)])
def test_brute_force_fractions(n, R, widths, seed):
    x = np.random.default_rng(seed).integers(0, 3073, size=n)
    y, z = _brute(x, R, widths)
    got_y = MF.baseline_removed(x, R)[0]
    np.testing.assert_allclose(got_y, np.array([float(v) for v in y]), rtol=1e-15, atol=1e-300)
    np.testing.assert_allclose(MF.matched_filter(x, R, widths)[:, 0, :], z, rtol=4e-16, atol=1e-300)


def test_numpy_convolve_interior():
    """A library routine with no prefix sums: np.convolve with a box of ones."""
    rng = np.random.default_rng(7)
    x = rng.integers(0, 1_044_481, size=(3, 700))           # 8-bit x 4096-channel range
    R, N = 37, 75
    m = MF.running_mean(x, R)
    for r in range(3):
        valid = np.convolve(x[r].astype(np.float64), np.ones(N), mode="valid") / N
        np.testing.assert_allclose(m[r, R:700 - R], valid, rtol=1e-13)
        # clamped windows at the ends repeat the first / last full window
        np.testing.assert_allclose(m[r, :R], valid[0], rtol=1e-13)
        np.testing.assert_allclose(m[r, 700 - R:], valid[-1], rtol=1e-13)
    y = MF.baseline_removed(x, R)
    for i, w in enumerate([1, 2, 4, 8, 16, 33]):
        z = MF.matched_filter(x, R, [w])[0]
        for r in range(3):
            box = np.convolve(y[r], np.ones(w), mode="valid") / np.sqrt(w)
            np.testing.assert_allclose(z[r, :700 - w + 1], box, rtol=1e-9, atol=1e-6)
            assert np.all(z[r, 700 - w + 1:] == 0)


def test_constant_input_is_removed():
    z = MF.matched_filter(np.full((2, 300), 1536), 20, [1, 2, 64])
    assert np.all(z == 0.0)


def test_linear_ramp():
    """A symmetric window removes a ramp exactly; at the ends the window centre lags."""
    n, R, beta = 200, 15, 7
    t = np.arange(n)
    y = MF.baseline_removed(100 + beta * t, R)[0]
    centre = np.clip(t, R, n - 1 - R)
    np.testing.assert_allclose(y, beta * (t - centre), rtol=0, atol=1e-12)


def test_impulse_response():
    n, R, t0, v = 400, 25, 180, 1000
    N = 2 * R + 1
    x = np.zeros(n, dtype=np.int64)
    x[t0] = v
    y = MF.baseline_removed(x, R)[0]
    want = np.where(np.abs(np.arange(n) - t0) <= R, -v / N, 0.0)
    want[t0] += v
    np.testing.assert_allclose(y, want, rtol=1e-15, atol=0)
    for w in (1, 4, 16):
        z = MF.matched_filter(x, R, [w])[0, 0]
        # a boxcar that covers the impulse and lies inside the window: v - w*v/N, over sqrt(w)
        np.testing.assert_allclose(z[t0 - w + 1:t0 + 1], (v - w * v / N) / np.sqrt(w), rtol=1e-14)
        # the best-matching width-1 boxcar sits on the impulse
        assert np.argmax(z) in range(t0 - w + 1, t0 + 1)


def test_width_one_is_identity_and_rows_independent():
    rng = np.random.default_rng(11)
    x = rng.integers(0, 3073, size=(4, 257))
    z = MF.matched_filter(x, 10, [1])[0]
    np.testing.assert_array_equal(z, MF.baseline_removed(x, 10))
    for r in range(4):
        np.testing.assert_array_equal(z[r], MF.matched_filter(x[r], 10, [1])[0, 0])


def test_white_noise_variance_is_width_independent():
    """1/sqrt(w) keeps the noise variance (reading R25): var(z_w) ~ sigma^2 (1 - w/N) for w << N."""
    rng = np.random.default_rng(5)
    x = np.rint(rng.normal(1536, 30.1, size=(8, 20000))).astype(np.int64)
    R = 500
    N = 2 * R + 1
    for i, w in enumerate([1, 4, 16, 64]):
        z = MF.matched_filter(x, R, [w])[0][:, R:20000 - R - w]
        assert abs(z.var() / (30.1 ** 2 * (1 - w / N)) - 1) < 0.05


def test_argument_checks():
    with pytest.raises(ValueError):
        MF.matched_filter(np.zeros(10, dtype=np.int64), 5, [1])     # N = 11 > n
    with pytest.raises(ValueError):
        MF.matched_filter(np.zeros(10, dtype=np.int64), 1, [11])    # width > n
    with pytest.raises(ValueError):
        MF.matched_filter(np.zeros(10) + 0.5, 1, [1])               # not integers
