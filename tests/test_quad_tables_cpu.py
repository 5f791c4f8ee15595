"""-m "not gpu": the host half of the quad-row path (dedisp_debug_quad_tables = the code dedisp_set_dm_list runs for
DEDISP_KERNEL_QUADS, on host arrays) against the addressing contract the tiled kernel relies on:

    out[d][t] = sum_q Q_{q, D_q(d)}[t + delay[4q][d]],   D_q(d) = (delay[4q+k][d] - delay[4q][d])_{k=1..3}
    (the re-association of out[d][t] = sum_c in[c][t + delay[c][d]], BASELINE.json:north_star; DESIGN.md Sec. 6 C)

i.e. for every (DM group, quad, lane): the row the lane's variant points at is the row of the lane's own triple of
delay differences, and the word the lane reads first -- box start of the variant + the lane's word in the box -- is
word delay[4q][d] >> 5 of that row, shifted by delay[4q][d] & 31; every word a lane reads lies inside its box; box
starts are multiples of 4 words (16-byte aligned TMA source).  The delay table comes from the oracle (test
infrastructure); no GPU is involved."""
import numpy as np
import pytest

import oracle
import paper_1112_0065_b200 as dd
import workloads as W

WIDE8 = W.CONFIGS["wide8"]
STEP8 = 2000.0 / 2047


def _tables(nchans, dm_lo, ndm, step=STEP8, shuffle=False):
    w = WIDE8.scaled(nchans=nchans, ndm=ndm, dm_lo=dm_lo, dm_hi=dm_lo + step * (ndm - 1))
    dms = np.asarray(w.dms())
    if shuffle:         # the caller's list in any order: the plan sorts the trials, a lane holds the caller's index
        dms = np.random.default_rng(5).permutation(dms)
    delay, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, dms)
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    ngroups = (ndm + 31) // 32
    lanes = np.full(ngroups * 32, -1, dtype=np.int32)
    lanes[:ndm] = np.argsort(dms, kind="stable")
    lanes = lanes.reshape(ngroups, 32)
    return delay, lanes, dd.dedisp_debug_quad_tables(delay, lanes)


def _lane_trials(lanes):
    """trial each lane serves: padding lanes repeat the last trial before them"""
    t = lanes.copy()
    for l in range(1, 32):
        t[:, l] = np.where(t[:, l] < 0, t[:, l - 1], t[:, l])
    return t


def _diffs(delay, nchans, q):
    """(ndm, 3) delay differences of quad q to its first channel; channels beyond nchans count as difference 0"""
    d0 = delay[4 * q]
    return np.stack([delay[4 * q + k] - d0 if 4 * q + k < nchans else np.zeros_like(d0) for k in (1, 2, 3)], axis=1)


@pytest.mark.parametrize("nchans,dm_lo,ndm,shuffle", [
    (4096, 0.0, 256, False),        # bottom of the DM range: few triples
    (4096, 1744.0, 262, False),     # top of the range: up to 7 variants per (group, quad); ragged last group
    (1001, 900.0, 288, False),      # last quad has one channel
    (514, 1200.0, 257, False),      # last quad has two channels; one trial in the last group
    (2048, 1500.0, 300, True),      # the caller's DM list in random order
])
def test_addressing_contract(nchans, dm_lo, ndm, shuffle):
    delay, lanes, (info, row0, trip, vlist, rel) = _tables(nchans, dm_lo, ndm, shuffle=shuffle)
    assert info["usable"] == 1
    nv, vslot, plw, tw, nq = (info[k] for k in ("nv", "vslot_bytes", "plane_words", "tile_words", "nquads_pad"))
    assert nv == 7 and vslot % 128 == 0 and plw * 10 * 4 <= vslot and tw % 4 == 0
    assert nq % 32 == 0 and nq >= (nchans + 3) // 4 and row0[0] == 0 and row0[nq] == info["nrows"] == len(trip)
    assert np.all(np.diff(row0) >= 1)
    trials = _lane_trials(lanes)                              # [ngroups][32]
    for q in range(nq):
        rows = trip[row0[q]:row0[q + 1]]
        assert np.all(rows[:, 3] == 0)
        if 4 * q >= nchans:                                   # padding quad: one all-zero row, every group on it
            assert len(rows) == 1 and not rows.any()
            assert np.all(vlist[:, q, 0, 0] == row0[q]) and np.all(vlist[:, q, 1:, 0] == -1)
            continue
        dq = _diffs(delay, nchans, q)
        # the rows of the quad are exactly the distinct triples of the list, in ascending (d1, d2, d3) order
        want = np.unique(dq, axis=0)
        assert np.array_equal(rows[:, :3], want)
        r = rel[:, q, :]                                      # [ngroups][32]
        off = (r >> 16).astype(np.int64)
        v, pos = off // vslot, (off % vslot) // 4
        assert np.all(off % 4 == 0) and np.all(v < nv)
        g = np.arange(lanes.shape[0])[:, None]
        row, xs = vlist[g, q, v, 0], vlist[g, q, v, 1]
        assert np.all(row >= row0[q]) and np.all(row < row0[q + 1])
        d0 = delay[4 * q][trials]                             # [ngroups][32]
        assert np.array_equal(trip[row][:, :, :3], dq[trials])      # the variant's row is the lane's own triple
        assert np.array_equal(xs + pos, d0 >> 5)                    # first word the lane reads
        assert np.array_equal(r & 0xFFFF, d0 & 31)                  # ... and its shift
        assert np.all(xs % 4 == 0)                                  # 16-byte aligned TMA source
        assert np.all(pos >= 0) and np.all(pos + tw + 1 <= plw)     # W + 1 words of every warp stay in the plane line
        # variants: used ones are distinct rows, listed first; the rest is -1
        for gi in range(lanes.shape[0]):
            used = vlist[gi, q, :, 0]
            n = int((used >= 0).sum())
            assert np.all(used[:n] >= 0) and np.all(used[n:] == -1) and len(set(used[:n])) == n
            assert set(used[:n]) == set(row[gi])


def _wavefronts(addr_words):
    """shared-memory wavefronts of one 32-lane load: lanes on the same word broadcast, a bank serves one word per
    wavefront"""
    a = np.unique(addr_words)
    return np.bincount(a % 32, minlength=32).max()


def test_box_placement_spreads_the_lanes_over_the_banks():
    # top of the wideband DM range: the triples of neighbouring trials alternate, the variants' windows interleave
    delay, lanes, (info, row0, trip, vlist, rel) = _tables(4096, 1744.0, 256)
    vslot, nq = info["vslot_bytes"], 1024
    fixed_skew = np.array([0, 16, 8, 24, 4, 20, 12])         # the first version: one skew per variant
    trials = _lane_trials(lanes)
    placed = fixed = n = 0
    for q in range(0, nq, 4):
        off = (rel[:, q, :] >> 16).astype(np.int64)
        v = off // vslot
        w0 = delay[4 * q][trials] >> 5
        for gi in range(lanes.shape[0]):
            placed += _wavefronts(off[gi] // 4)               # slots start at bank 0: word address = off / 4
            fixed += _wavefronts(v[gi] * (vslot // 4) + (w0[gi] - (w0[gi].min() & ~3)) + fixed_skew[v[gi]])
            n += 1
    assert placed / n < 1.40 and placed < 0.85 * fixed, (placed / n, fixed / n)


def test_lists_that_cannot_take_quad_rows_and_bad_arguments():
    # DM steps 40 x coarser: more than 7 distinct triples inside a group of 32 trials -> not usable, not an error
    _, _, (info, *rest) = _tables(4096, 0.0, 256, step=40 * STEP8)
    assert info["usable"] == 0 and info["nrows"] == 0 and all(a is None for a in rest)
    delay = np.zeros((8, 32), dtype=np.int32)
    lanes = np.arange(32, dtype=np.int32).reshape(1, 32)
    info, row0, trip, vlist, rel = dd.dedisp_debug_quad_tables(delay, lanes)       # all delays 0: one row per quad
    assert info["usable"] == 1 and info["nrows"] == info["nquads_pad"] and not trip.any()
    for bad_delay, bad_lanes in ((np.zeros((3, 32), np.int32), lanes),            # fewer than 4 channels
                                 (delay, np.full((1, 32), 32, np.int32)),         # lane beyond the table
                                 (delay, np.full((1, 32), -1, np.int32))):        # lane 0 is padding
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_debug_quad_tables(bad_delay, bad_lanes)
        assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    # a negative difference (delays must not decrease along the channels of a quad) -> not usable
    delay2 = delay.copy()
    delay2[0] = 5
    assert dd.dedisp_debug_quad_tables(delay2, lanes)[0]["usable"] == 0


def test_walking_the_tables_on_the_cpu_reproduces_the_oracle_sums():
    """The data flow of the quad path replayed in numpy from the PRODUCT's tables (rows from trip/row0, every lane
    gathering from the row, box start, word and shift its tables name) against oracle.dedisperse: the tables alone
    decide which samples are summed, so this pins them end to end without a GPU."""
    nchans, ndm, nso = 70, 256, 200                 # 70 channels: the last quad has two
    w = WIDE8.scaled(nchans=nchans, ndm=ndm, df=-4.0, dm_lo=100.0, dm_hi=100.0 + 0.02 * (ndm - 1), nsamps_out=nso)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    x = W.generate(w, md)                            # uint8 [nchans][nsamps_in]: 8-bit samples are the bytes
    lanes = np.arange(ndm, dtype=np.int32).reshape(ndm // 32, 32)
    info, row0, trip, vlist, rel = dd.dedisp_debug_quad_tables(delay, lanes)
    assert info["usable"] == 1 and info["nrows"] > 5 * info["nquads_pad"]    # many triples per quad (232 rows, 18 quads)
    vslot = info["vslot_bytes"]
    nin = nso + md
    xs8 = np.zeros((4 * info["nquads_pad"], nin + 64), dtype=np.int64)       # channels / samples beyond the input: zero
    xs8[:nchans, :nin] = x[:, :nin]
    t = np.arange(nso)
    got = np.zeros((ndm, nso), dtype=np.int64)
    for g in range(lanes.shape[0]):
        for l in range(32):
            d = lanes[g, l]
            for q in range(info["nquads_pad"]):
                r = int(rel[g, q, l])
                off = r >> 16
                v, pos = off // vslot, (off % vslot) // 4
                row, box = vlist[g, q, v]
                assert row0[q] <= row < row0[q + 1]
                first = (box + pos) * 32 + (r & 0xFFFF)          # sample of the row the lane's output t = 0 reads
                d1, d2, d3, _ = trip[row]
                for k, dk in enumerate((0, d1, d2, d3)):         # the row: sum of the quad's channels at its triple
                    got[d] += xs8[4 * q + k, first + dk + t]
    want = oracle.dedisperse(delay, x, 8, nso)
    assert np.array_equal(got, want.astype(np.int64))


def test_the_wideband_config_takes_quad_rows_with_the_documented_table_sizes():
    # BASELINE.json:configs[3] in full (4096 channels x 2048 trials): the numbers DESIGN.md Sec. 6 C and
    # profiles/r2_wide8.md quote for the quad path come from these tables
    w = WIDE8
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    lanes = np.arange(w.ndm, dtype=np.int32).reshape(w.ndm // 32, 32)
    info, row0, trip, vlist, rel = dd.dedisp_debug_quad_tables(np.ascontiguousarray(delay, dtype=np.int32), lanes)
    assert info["usable"] == 1 and info["nquads_pad"] == 1024 and info["nrows"] == 88042
    nvar = (vlist[:, :, :, 0] >= 0).sum(axis=2)              # variants per (DM group, quad)
    assert nvar.min() >= 1 and nvar.max() == 7 and abs(nvar.mean() - 4.256) < 0.001
    # AUTO's rule (bitslice_kernel.cu): at most 3 rows to build per (group, quad) slot served, rows within 24 GB
    assert info["nrows"] <= 3 * lanes.shape[0] * info["nquads_pad"]
    ntiles = -(-w.nsamps_out // (32 * info["tile_words"]))
    pitch = ((md >> 5) + ntiles * info["tile_words"] + 72 + 4 + 3) & ~3
    assert pitch == 5760 and abs(info["nrows"] * 10 * pitch * 4 / 1e9 - 20.28) < 0.01 and info["nrows"] * 10 * pitch * 4 < 24 << 30
    # shared-memory wavefronts per window load with the placement of the tables: 1.313 (with the one conflict-free rel
    # load per 50 window loads: 1.307; ncu measured 4.520 G wavefronts for 3.456 G loads = 1.308, profiles/r2_wide8.md)
    words = (rel >> 16).astype(np.int64) // 4
    wf = np.mean([_wavefronts(words[g, q]) for g in range(0, lanes.shape[0], 2) for q in range(0, 1024, 2)])
    assert abs(wf - 1.313) < 0.01
