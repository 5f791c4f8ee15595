"""Pins for the CPU oracle (no GPU).  Each test fixes the oracle to something
other than itself: hand-worked numbers, exact rational arithmetic, the textbook
closed form, invariants of the definition, or an independent NumPy slice-sum.

Definition under test (BASELINE.json:north_star; Sec. 2.2):
    out[d][t] = sum_c in[c][t + delay[c][d]]
    delay[c][d] = round_half_away(4148.808 * DM_d * (f_c^-2 - f_top^-2) / dt)
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import workloads as W


# ----------------------------------------------------------------- helpers
def _exact_delay(c, dm, dt, f_top, df):
    """Exact-rational evaluation of the formula on the double inputs, rounded
    half away from zero (all values are >= 0 here)."""
    fc = Fraction(f_top) + c * Fraction(df)
    a = 1 / (fc * fc) - 1 / (Fraction(f_top) ** 2)
    x = Fraction(4148.808) * Fraction(dm) * a / Fraction(dt)
    assert x >= 0
    return int(x + Fraction(1, 2))  # floor(x + 1/2) == round half away for x >= 0


def _slice_sum(delay, u8, nsamps_out):
    """Independent NumPy restatement: one shifted row slice per channel."""
    nchans, ndm = delay.shape
    out = np.zeros((ndm, nsamps_out), dtype=np.uint32)
    for d in range(ndm):
        for c in range(nchans):
            s = int(delay[c, d])
            out[d] += u8[c, s:s + nsamps_out]
    return out


def _unpack(packed, nbits, nsamps):
    if nbits == 8:
        return packed[:, :nsamps]
    if nbits == 2:
        return np.stack([W.unpack2(r, nsamps) for r in packed])
    return np.stack([W.unpack_bits(r, nbits, nsamps) for r in packed])


def _read_delay_pins(golden_dir):
    rows = []
    for line in (golden_dir / "delay_pins.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        rows.append(dict(name=p[0], nchans=int(p[1]), f_top=float(p[2]), df=float(p[3]),
                         dt=float(p[4]), ndm=int(p[5]), dm_lo=float(p[6]), dm_hi=float(p[7]),
                         max_delay=int(p[8]), total=int(p[9]), checksum=int(p[10]),
                         corners=[int(v) for v in p[11:16]], lastchan=int(p[16]),
                         lastdm=int(p[17])))
    return rows


def _read_hand(golden_dir):
    kv = {"delay": [], "row": [], "packed": [], "out": []}
    for line in (golden_dir / "hand_worked.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        if k in kv:
            kv[k].append(v)
        else:
            kv[k] = v
    return kv


# ------------------------------------------------------------- delay table
def test_delay_table_pins(golden_dir):
    for p in _read_delay_pins(golden_dir):
        dms = np.linspace(p["dm_lo"], p["dm_hi"], p["ndm"])
        d, md = oracle.delay_table(p["nchans"], p["dt"], p["f_top"], p["df"], dms)
        nch, ndm = d.shape
        assert md == p["max_delay"] == int(d.max())
        d64 = d.astype(np.int64)
        assert int(d64.sum()) == p["total"]
        wgt = (1000003 * np.arange(nch, dtype=np.uint64)[:, None]
               + 7919 * np.arange(ndm, dtype=np.uint64)[None, :] + np.uint64(1))
        with np.errstate(over="ignore"):
            cs = int((d.astype(np.uint64) * wgt).sum(dtype=np.uint64))
        assert cs == p["checksum"]
        assert [int(d[1, 1]), int(d[-1, 1]), int(d[1, -1]), int(d[-1, -1]),
                int(d[nch // 2, ndm // 2])] == p["corners"]
        assert int(d64[-1].sum()) == p["lastchan"]
        assert int(d64[:, -1].sum()) == p["lastdm"]
        # invariants: reference channel and DM 0 have zero delay; monotone in c and d
        assert not d[0].any() and not d[:, 0].any()
        assert (np.diff(d64, axis=0) >= 0).all() and (np.diff(d64, axis=1) >= 0).all()


def test_delay_exact_rational_tiny_full_and_htru_sample():
    w = W.CONFIGS["tiny"]
    d, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    for c in range(w.nchans):
        for k, dm in enumerate(w.dms()):
            assert d[c, k] == _exact_delay(c, dm, w.dt, w.f_top, w.df), (c, k)
    for name in ("htru_gulp", "wide8"):
        w = W.CONFIGS[name]
        dms = w.dms()
        d, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, dms)
        rng = np.random.default_rng(5)
        cs = rng.integers(0, w.nchans, 1500)
        ks = rng.integers(0, w.ndm, 1500)
        # plus the entry SURVEY.md Sec. 8(c) R4 names as closest to a tie
        extra = [(983, 932)] if name == "htru_gulp" else [(2807, 460)]
        for c, k in list(zip(cs, ks)) + extra:
            assert d[c, k] == _exact_delay(int(c), dms[k], w.dt, w.f_top, w.df), (c, k)


def test_delay_rounding_is_half_away_not_half_even():
    # f_top=2, df=-1, one channel below: a = 1 - 1/4 = 3/4 exactly.
    # x = 4148.808*DM*0.75/dt ; choose dt = 4148.808*0.75 => x == DM (up to fp rounding),
    # so use dyadic DMs where the product chain is exact: K*DM exact is not guaranteed,
    # hence verify against exact rationals *and* require a .5 case to round up.
    K = 4148.808
    dt = K * 0.75
    dms = np.array([0.5, 1.5, 2.5, 3.5, 4.5])
    d, _ = oracle.delay_table(2, dt, 2.0, -1.0, dms)
    for k, dm in enumerate(dms):
        x = ((K * dm) * 0.75) / dt
        if x == dm:  # chain happened to be exact: an exact tie
            assert d[1, k] == int(dm + 0.5), "ties must round away from zero"
    # at least these exact ties exist (0.5, 1.5, 2.5 ... multiply exactly by powers of 2 / small ints)
    assert d[1, 0] == 1 and d[1, 2] == 3  # 0.5 -> 1, 2.5 -> 3 (half-even would give 0 and 2)


def test_delay_textbook_closed_form():
    # Continuous sweep: 4.148808 ms * DM * ((f/GHz)^-2 - (f_top/GHz)^-2); HTRU DM 1000,
    # lowest channel 1182.190625 MHz vs 1581.8 MHz: 1.31044 s = 20475.6 samples of 64 us.
    w = W.CONFIGS["htru_gulp"]
    f_lo = w.f_top + (w.nchans - 1) * w.df
    assert f_lo == 1182.190625
    sec = 4.148808e-3 * 1000.0 * ((f_lo / 1e3) ** -2 - (w.f_top / 1e3) ** -2)
    assert abs(sec - 1.310441) < 1e-6
    d, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    assert md == d[-1, -1] == 20476 == int(np.floor(sec / w.dt + 0.5))


def test_delay_table_argument_errors():
    with pytest.raises(ValueError):
        oracle.delay_table(4, -1.0, 1500.0, -1.0, [0.0])
    with pytest.raises(ValueError):
        oracle.delay_table(0, 1e-3, 1500.0, -1.0, [0.0])


# ------------------------------------------------------- hand-worked example
def test_hand_worked_example(golden_dir):
    h = _read_hand(golden_dir)
    nchans = int(h["nchans"][0])
    dms = np.array([float(v) for v in h["dms"]])
    d, md = oracle.delay_table(nchans, float(h["dt"][0]), float(h["f_top"][0]),
                               float(h["df"][0]), dms)
    assert d.tolist() == [[int(v) for v in r] for r in h["delay"]]
    assert md == int(h["max_delay"][0])
    rows = np.array([[int(ch) for ch in r[0]] for r in h["row"]], dtype=np.uint8)
    packed = np.array([[int(b, 16) for b in r] for r in h["packed"]], dtype=np.uint8)
    # fixture self-consistency: the packed bytes are the digit rows, LSB first
    assert np.array_equal(np.stack([W.pack2(r) for r in rows]), packed)
    nso = int(h["nsamps_out"][0])
    want = np.array([[int(v) for v in r] for r in h["out"]], dtype=np.uint32)
    assert np.array_equal(oracle.dedisperse_literal(d, packed, 2, nso), want)
    assert np.array_equal(oracle.dedisperse(d, packed, 2, nso), want)
    # one entry by hand: out[1][0] = in0[0] + in1[3] + in2[6] + in3[10]
    assert rows[0, 0] + rows[1, 3] + rows[2, 6] + rows[3, 10] == want[1, 0] == 5


# ------------------------------------------------------------- invariants
@pytest.fixture(scope="module")
def tiny():
    w = W.CONFIGS["tiny"]
    d, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    return w, d, md, x


def test_tiny_literal_equals_fast_equals_slice_sum(tiny):
    w, d, md, x = tiny
    o1 = oracle.dedisperse_literal(d, x, 2, w.nsamps_out)
    o2 = oracle.dedisperse(d, x, 2, w.nsamps_out)
    o3 = _slice_sum(d, _unpack(x, 2, w.nsamps_out + md), w.nsamps_out)
    assert np.array_equal(o1, o2) and np.array_equal(o1, o3)
    # statistics of a uniform {0..3} sum over 64 channels: mean 96, var 80
    assert abs(o1.mean() - 96.0) < 0.2 and abs(o1.var() - 80.0) < 2.0
    assert o1.max() <= 3 * w.nchans


def test_dm0_is_plain_channel_sum(tiny):
    w, d, md, x = tiny
    assert w.dms()[0] == 0.0
    o = oracle.dedisperse(d, x, 2, w.nsamps_out)
    u8 = _unpack(x, 2, w.nsamps_out + md)
    assert np.array_equal(o[0], u8[:, :w.nsamps_out].sum(axis=0, dtype=np.uint32))


@pytest.mark.parametrize("nbits,v", [(2, 3), (8, 201)])
def test_impulse_peaks_at_its_trial(tiny, nbits, v):
    w, d, md, _ = tiny
    k, t0 = 16, 1000
    nin = w.nsamps_out + md
    u8 = np.zeros((w.nchans, nin), dtype=np.uint8)
    for c in range(w.nchans):
        u8[c, t0 + d[c, k]] = v
    packed = u8 if nbits == 8 else np.stack([W.pack2(r) for r in u8])
    o = oracle.dedisperse(d, packed, nbits, w.nsamps_out)
    assert o[k, t0] == w.nchans * v
    assert (o == w.nchans * v).sum() == 1          # unique global maximum
    assert o.max() == w.nchans * v
    assert int(o.astype(np.int64).sum()) >= w.nchans * v
    # largest off-trial response for tiny, k=16 is 2*v
    o[k, t0] = 0
    assert o.max() == 2 * v
    assert np.array_equal(oracle.dedisperse_literal(d, packed, nbits, w.nsamps_out)[k, t0],
                          w.nchans * v)


def test_linearity(tiny):
    w, d, md, _ = tiny
    nin = w.nsamps_out + md
    g = np.random.default_rng(11)
    a = g.integers(0, 2, (w.nchans, nin), dtype=np.uint8)
    b = g.integers(0, 3, (w.nchans, nin), dtype=np.uint8)   # a+b <= 3
    pk = lambda m: np.stack([W.pack2(r) for r in m])
    oa = oracle.dedisperse(d, pk(a), 2, w.nsamps_out)
    ob = oracle.dedisperse(d, pk(b), 2, w.nsamps_out)
    oab = oracle.dedisperse(d, pk(a + b), 2, w.nsamps_out)
    assert np.array_equal(oa + ob, oab)
    a8 = g.integers(0, 128, (w.nchans, nin), dtype=np.uint8)
    b8 = g.integers(0, 128, (w.nchans, nin), dtype=np.uint8)
    assert np.array_equal(oracle.dedisperse(d, a8, 8, w.nsamps_out)
                          + oracle.dedisperse(d, b8, 8, w.nsamps_out),
                          oracle.dedisperse(d, a8 + b8, 8, w.nsamps_out))


def test_constant_and_per_channel_constant(tiny):
    w, d, md, _ = tiny
    nin = w.nsamps_out + md
    x = np.full((w.nchans, W.row_stride_bytes(nin, 2)), 0xFF, dtype=np.uint8)
    assert (oracle.dedisperse(d, x, 2, w.nsamps_out) == 3 * w.nchans).all()
    gc = (np.arange(w.nchans) * 7 % 256).astype(np.uint8)
    x8 = np.repeat(gc[:, None], nin, axis=1)
    assert (oracle.dedisperse(d, x8, 8, w.nsamps_out) == int(gc.astype(np.int64).sum())).all()


def test_time_shift(tiny):
    w, d, md, x = tiny
    s = 37
    nso = w.nsamps_out - s
    u8 = _unpack(x, 2, w.nsamps_out + md)
    shifted = np.stack([W.pack2(r[s:]) for r in u8])
    o = oracle.dedisperse(d, x, 2, w.nsamps_out)
    os_ = oracle.dedisperse(d, shifted, 2, nso)
    assert np.array_equal(o[:, s:], os_)


def test_prefix_sum_conservation(tiny):
    w, d, md, x = tiny
    u8 = _unpack(x, 2, w.nsamps_out + md).astype(np.int64)
    S = np.concatenate([np.zeros((w.nchans, 1), np.int64), np.cumsum(u8, axis=1)], axis=1)
    o = oracle.dedisperse(d, x, 2, w.nsamps_out).astype(np.int64)
    T = w.nsamps_out
    for k in range(w.ndm):
        want = sum(S[c, T + d[c, k]] - S[c, d[c, k]] for c in range(w.nchans))
        assert o[k].sum() == want


def test_sub_byte_layouts_against_unpackbits():
    """Row f4 (reading R36): 1-, 2- and 4-bit samples are LSB-first; numpy.unpackbits
    (bitorder='little') is the independent statement of that layout."""
    for nbits, hexrow, want in ((1, "b1 03", [1, 0, 0, 0, 1, 1, 0, 1, 1, 1, 0, 0, 0, 0, 0, 0]),
                                (4, "a3 0f 70", [3, 10, 15, 0, 0, 7]),
                                (2, "e4", [0, 1, 2, 3])):
        row = np.frombuffer(bytes.fromhex(hexrow.replace(" ", "")), dtype=np.uint8)
        assert W.unpack_bits(row, nbits, len(want)).tolist() == want
        assert W.pack_bits(np.array(want, np.uint8), nbits).tolist() == row.tolist()
        delay = np.zeros((1, 1), np.int32)
        out = oracle.dedisperse_literal(delay, row[None].copy(), nbits, len(want))
        assert out[0].tolist() == want          # one channel, DM 0: the output is the samples


@pytest.mark.parametrize("nbits", [1, 2, 4, 8])
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_brute_force_random_small_shapes(seed, nbits):
    g = np.random.default_rng(seed)
    nchans = int(g.integers(1, 17))
    ndm = int(g.integers(1, 9))
    nso = int(g.integers(1, 65))
    delay = np.sort(g.integers(0, 50, (nchans, ndm)), axis=1).astype(np.int32)
    delay[0] = 0
    md = int(delay.max())
    x = W.random_small(seed, nchans, nso + md, nbits)
    u8 = _unpack(x, nbits, nso + md)
    want = _slice_sum(delay, u8, nso)
    assert np.array_equal(oracle.dedisperse_literal(delay, x, nbits, nso), want)
    assert np.array_equal(oracle.dedisperse(delay, x, nbits, nso), want)
    # pure-Python triple loop straight from the definition
    for d_ in range(ndm):
        for t in range(min(nso, 5)):
            assert want[d_, t] == sum(int(u8[c, t + delay[c, d_]]) for c in range(nchans))


def test_partial_dm_range_and_threads(tiny):
    w, d, md, x = tiny
    full = oracle.dedisperse(d, x, 2, w.nsamps_out)
    part, used = oracle.dedisperse(d, x, 2, w.nsamps_out, d_begin=5, d_end=9, nthreads=2,
                                   return_threads=True)
    assert used == 2
    assert np.array_equal(part[5:9], full[5:9]) and not part[:5].any() and not part[9:].any()


def test_f32_view_is_exact(tiny):
    w, d, md, x = tiny
    o = oracle.dedisperse(d, x, 2, w.nsamps_out)
    f = oracle.to_f32(o)
    assert f.dtype == np.float32 and np.array_equal(f.astype(np.uint32), o)
    big = np.array([4096 * 255, 2 ** 24 - 1], dtype=np.uint32)
    assert np.array_equal(oracle.to_f32(big).astype(np.uint32), big)


def test_short_rows_rejected(tiny):
    w, d, md, x = tiny
    with pytest.raises(ValueError):
        oracle.dedisperse(d, x[:, :-8].copy(), 2, w.nsamps_out)
