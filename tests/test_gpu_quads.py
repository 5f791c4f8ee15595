"""-m gpu parity tests of the quad-row variant of the tiled kernel (DEDISP_KERNEL_QUADS, 8-bit samples; DESIGN.md
"Kernel C, quad rows"): the sum of four adjacent channels is formed once per triple of delay differences of the DM
list and the tiles add nchans/4 ten-plane rows.  It is the same integer sum as
out[d][t] = sum_c in[c][t + delay[c][d]] (BASELINE.json:north_star), so every case is bit-exact against the oracle."""
import numpy as np
import pytest
import torch

import oracle
import paper_1112_0065_b200 as dd
import workloads as W
from gpu_helpers import gpu_dedisperse, make_plan

pytestmark = pytest.mark.gpu

WIDE8 = W.CONFIGS["wide8"]
STEP8 = 2000.0 / 2047         # DM step of the wideband list


def _workload(nchans, dm_lo, ndm, nsamps, od="u32", nbeams=1):
    return WIDE8.scaled(nchans=nchans, ndm=ndm, dm_lo=dm_lo, dm_hi=dm_lo + STEP8 * (ndm - 1), nsamps_out=nsamps,
                        out_dtype=od, nbeams=nbeams)


@pytest.mark.parametrize("nchans,dm_lo,ndm,nsamps,od", [
    (4096, 0.0, 256, 1500, "u32"),       # bottom of the DM range: few distinct triples
    (4096, 1744.0, 262, 1409, "f32"),    # top of the range: up to 7 triples per (group, quad); ragged last group
    (1001, 900.0, 288, 3000, "u32"),     # channel count not a multiple of 4: the last quad has one channel
    (514, 1200.0, 257, 2817, "f32"),     # ... two channels; one trial in the last group
    (6, 0.0, 256, 50, "u32"),            # fewer channels than a stage of four quads
])
def test_eight_bit_quad_rows(nchans, dm_lo, ndm, nsamps, od):
    w = _workload(nchans, dm_lo, ndm, nsamps, od)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_QUADS)
    got = gpu_dedisperse(p, x[None], 8, w.nsamps_out, od)[0]
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_QUADS
    want = oracle.dedisperse(delay, x, 8, w.nsamps_out)
    assert np.array_equal(got, want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


def test_delay_differences_beyond_one_word_and_unsorted_list():
    # DM 4000 .. 4250 on the wideband channelisation: differences to the first channel of a quad beyond 64 samples
    w = _workload(4096, 4000.0, 256, 1500)
    dms = np.random.default_rng(3).permutation(w.dms())
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, dms)
    d3 = delay[3::4] - delay[0::4]
    assert d3.max() >= 64
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, dms, dd.DEDISP_KERNEL_QUADS)
    got = gpu_dedisperse(p, x[None], 8, w.nsamps_out)[0]
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_QUADS
    assert np.array_equal(got, oracle.dedisperse(delay, x, 8, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_extreme_values_and_beams():
    # all samples 255: every quad sum is 1020 (all ten planes, every carry), every output 255 * nchans
    w = _workload(4096, 0.0, 256, 1000, nbeams=2)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = np.full((2, w.nchans, w.nsamps_out + md), 0xFF, dtype=np.uint8)
    x[1, ::3] = 0x80
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_QUADS)
    got = gpu_dedisperse(p, x, 8, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_QUADS
    assert np.all(got[0] == 255 * w.nchans)
    assert np.array_equal(got[1], oracle.dedisperse(delay, x[1], 8, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_quads_equal_pairs_and_planes_on_one_plan_and_refusals():
    w = _workload(1024, 600.0, 320, 3000)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_QUADS)
    res = {}
    for k in (dd.DEDISP_KERNEL_QUADS, dd.DEDISP_KERNEL_PAIRS, dd.DEDISP_KERNEL_BITSLICE, dd.DEDISP_KERNEL_QUADS):
        dd.dedisp_set_kernel(p, k)
        res[k] = gpu_dedisperse(p, x[None], 8, w.nsamps_out)[0]
        assert dd.dedisp_get_last_kernel(p) == k
        assert np.array_equal(res[k], res[dd.DEDISP_KERNEL_QUADS])
    assert np.array_equal(res[dd.DEDISP_KERNEL_QUADS], oracle.dedisperse(delay, x, 8, w.nsamps_out))
    dd.dedisp_destroy(p)
    # 2-bit data and short DM lists (fewer than 8 groups) have no quad rows: forced QUADS is refused, AUTO serves
    w2 = W.CONFIGS["htru_gulp"].scaled(ndm=64, dm_hi=50.0, nsamps_out=500)
    _, md2 = oracle.delay_table(w2.nchans, w2.dt, w2.f_top, w2.df, w2.dms())
    x2 = W.generate(w2, md2)
    p = make_plan(w2.nchans, w2.dt, w2.f_top, w2.df, w2.dms(), dd.DEDISP_KERNEL_QUADS)
    with pytest.raises(dd.DedispError) as e:
        gpu_dedisperse(p, x2[None], 2, w2.nsamps_out)
    assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    dd.dedisp_destroy(p)
    w3 = _workload(256, 0.0, 64, 500)
    _, md3 = oracle.delay_table(w3.nchans, w3.dt, w3.f_top, w3.df, w3.dms())
    p = make_plan(w3.nchans, w3.dt, w3.f_top, w3.df, w3.dms(), dd.DEDISP_KERNEL_QUADS)
    with pytest.raises(dd.DedispError):
        gpu_dedisperse(p, W.generate(w3, md3)[None], 8, w3.nsamps_out)
    dd.dedisp_destroy(p)
    # more than 4096 channels would need two channel blocks: such plans have no quad rows either
    w4 = _workload(4100, 0.0, 256, 100)
    _, md4 = oracle.delay_table(w4.nchans, w4.dt, w4.f_top, w4.df, w4.dms())
    p = make_plan(w4.nchans, w4.dt, w4.f_top, w4.df, w4.dms(), dd.DEDISP_KERNEL_QUADS)
    with pytest.raises(dd.DedispError) as e:
        gpu_dedisperse(p, W.generate(w4, md4)[None], 8, w4.nsamps_out)
    assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    dd.dedisp_destroy(p)
