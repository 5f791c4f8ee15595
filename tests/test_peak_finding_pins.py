"""Pins for the peak-finding oracle (no GPU): hand-worked numbers, a literal
sample-by-sample state machine, run-length identities, and the edge cases of the
definition (Sec. 2.3; readings R27-R31)."""
from pathlib import Path

import numpy as np
import pytest

from oracle import peak_finding as PF

GOLDEN = Path(__file__).resolve().parent / "golden"


def _state_machine(z, sigma, nsigma):
    """The definition, one sample at a time, no numpy tricks."""
    ev = []
    for s in range(len(z)):
        thr = np.float32(nsigma) * np.float32(sigma[s])
        run = None
        for t in range(len(z[s])):
            v = np.float32(z[s][t])
            if v > thr:
                if run is None:
                    run = [s, t, 1, t, v]
                else:
                    run[2] += 1
                    if v > run[4]:
                        run[3], run[4] = t, v
            elif run is not None:
                ev.append(tuple(run))
                run = None
        if run is not None:
            ev.append(tuple(run))
    return np.array(ev, dtype=PF.EVENT_DTYPE)


def _read_hand():
    z, ev, sigma, nsigma = [], [], None, None
    for line in (GOLDEN / "peak_finding_hand.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        if p[0] == "z":
            z.append([float(v) for v in p[1:]])
        elif p[0] == "sigma":
            sigma = [float(v) for v in p[1:]]
        elif p[0] == "nsigma":
            nsigma = float(p[1])
        elif p[0] == "event":
            ev.append((int(p[1]), int(p[2]), int(p[3]), int(p[4]), float(p[5])))
    return np.array(z, dtype=np.float32), sigma, nsigma, np.array(ev, dtype=PF.EVENT_DTYPE)


def test_hand_worked_example():
    z, sigma, nsigma, want = _read_hand()
    got = PF.find_events(z, sigma, nsigma)
    assert got.tolist() == want.tolist()
    assert PF.sigma_cut(z, sigma, nsigma)[0].tolist() == [True, True, False, False, True, False, False,
                                                         True, True, True]


@pytest.mark.parametrize("seed,nseries,n,nsigma", [(1, 4, 200, 1.0), (2, 3, 1000, 2.5), (3, 6, 77, 0.0),
                                                   (4, 2, 5000, 3.5)])
def test_state_machine(seed, nseries, n, nsigma):
    rng = np.random.default_rng(seed)
    z = rng.standard_normal((nseries, n)).astype(np.float32)
    z[0, :5] = 9.0                      # run at the start
    z[-1, -3:] = 9.0                    # run at the end
    sigma = (0.5 + rng.random(nseries)).astype(np.float32)
    got = PF.find_events(z, sigma, nsigma)
    want = _state_machine(z, sigma, nsigma)
    assert got.tolist() == want.tolist() and len(got) > 0


def test_run_length_identities():
    rng = np.random.default_rng(9)
    z = rng.standard_normal((5, 3000)).astype(np.float32)
    sigma = np.ones(5, dtype=np.float32)
    ev = PF.find_events(z, sigma, 1.2)
    m = PF.sigma_cut(z, sigma, 1.2)
    assert ev["length"].sum() == m.sum()                                  # runs tile the mask
    starts = (m & ~np.concatenate((np.zeros((5, 1), bool), m[:, :-1]), axis=1)).sum()
    assert len(ev) == starts                                              # one event per rising edge
    assert np.all(np.diff(ev["series"].astype(np.int64) * 3000 + ev["t_start"]) > 0)   # sorted, disjoint
    for e in ev:
        seg = z[e["series"], e["t_start"]:e["t_start"] + e["length"]]
        assert e["peak"] == seg.max() and e["t_peak"] == e["t_start"] + int(np.argmax(seg))
        assert np.all(seg > np.float32(1.2))


def test_edge_cases():
    one = np.float32(1.0)
    # whole series above; nothing above; value equal to threshold; NaN; equal maxima
    z = np.array([[2, 2, 2, 2], [0, 0, 0, 0], [1, 1, 1, 1], [np.nan, 5, np.nan, 5], [3, 7, 7, 3]],
                 dtype=np.float32)
    ev = PF.find_events(z, np.full(5, one), 1.0)
    assert ev.tolist() == [(0, 0, 4, 0, 2.0), (3, 1, 1, 1, 5.0), (3, 3, 1, 3, 5.0), (4, 0, 4, 1, 7.0)]
    assert len(PF.find_events(np.zeros((1, 1), np.float32), [1.0], 1.0)) == 0
    # the threshold product is taken in float32
    s, k = np.float32(0.1), np.float32(3.0)
    thr32 = s * k
    z = np.array([[thr32, np.nextafter(thr32, np.float32(np.inf))]], dtype=np.float32)
    assert PF.find_events(z, [s], k).tolist() == [(0, 1, 1, 1, float(z[0, 1]))]


def test_series_rms_closed_forms():
    assert PF.series_rms(np.full((2, 100), 3.0, np.float32)).tolist() == [3.0, 3.0]
    z = np.tile(np.array([1.0, -1.0, 2.0, -2.0], np.float32), (1, 25))
    np.testing.assert_allclose(PF.series_rms(z), [np.sqrt(2.5)], rtol=1e-15)
    g = np.random.default_rng(3).standard_normal((1, 200000)).astype(np.float32) * 30.1
    assert abs(PF.series_rms(g)[0] / 30.1 - 1) < 0.01
