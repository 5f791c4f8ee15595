"""-m gpu parity tests of the pair-row variant of the tiled kernel (DEDISP_KERNEL_PAIRS, DESIGN.md
"Kernel C, pair rows"): the sum of two adjacent channels is formed once per delay difference of the DM
list and the tiles add nchans/2 three-plane rows.  It is the same integer sum as
out[d][t] = sum_c in[c][t + delay[c][d]] (BASELINE.json:north_star), so every case is bit-exact against
the oracle's literal loop."""
import numpy as np
import pytest
import torch

import oracle
import paper_1112_0065_b200 as dd
import workloads as W
from gpu_helpers import gpu_dedisperse, make_plan, oracle_inputs

pytestmark = pytest.mark.gpu

HTRU = W.CONFIGS["htru_gulp"]
STEP = 1000.0 / 1199          # DM step of the HTRU list


def _check(w, dms=None, od="u32"):
    dms = w.dms() if dms is None else dms
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, dms)
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, dms, dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x[None], 2, w.nsamps_out, od)[0]
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    want = oracle.dedisperse(delay, x, 2, w.nsamps_out)
    assert np.array_equal(got, want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("od", ["u32", "f32"])
@pytest.mark.parametrize("dm_lo,ndm", [(0.0, 70), (930.0, 84), (480.0, 33)])
def test_htru_shape_low_mid_and_top_of_the_dm_range(dm_lo, ndm, od):
    # 1024 channels, HTRU DM step; the top of the range has the largest delay differences (30 samples
    # between the two lowest channels) and groups whose trials use three differences of a pair
    w = HTRU.scaled(ndm=ndm, dm_lo=dm_lo, dm_hi=dm_lo + STEP * (ndm - 1), nsamps_out=4100, out_dtype=od)
    _check(w, od=od)


@pytest.mark.parametrize("od", ["u32", "f32"])
def test_delay_differences_beyond_one_word(od):
    # DM 2050 .. 2156 on the HTRU channelisation: pair delay differences reach 66 samples, so the rows of a pair
    # cross the 32- and 64-sample word boundaries (the row pre-pass re-reads the odd channel at a new word
    # offset in the middle of a pair's row list) and the lowest pairs start beyond one word
    w = HTRU.scaled(ndm=128, dm_lo=2050.0, dm_hi=2050.0 + STEP * 127, nsamps_out=4100, out_dtype=od)
    delay, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    delta = delay[1::2] - delay[0::2]
    assert delta.max() >= 64 and np.any((delta.min(axis=1) < 32) & (delta.max(axis=1) >= 32))
    _check(w, od=od)


@pytest.mark.parametrize("nchans,df,dm_hi,ndm,nsamps", [
    (2, -100.0, 0.4, 5, 100), (3, -50.0, 0.5, 33, 700), (37, -7.0, 3.0, 40, 1921), (1023, -0.39, 50.0, 64, 1920),
    (130, -2.5, 15.0, 97, 3841), (64, -6.25, 1.8, 32, 4096),
])
def test_odd_channel_counts_ragged_tiles_and_padding_lanes(nchans, df, dm_hi, ndm, nsamps):
    # (DM ranges chosen so that the 32 trials of a group span less than one sample of pair delay difference)
    w = HTRU.scaled(nchans=nchans, df=df, ndm=ndm, dm_hi=dm_hi, nsamps_out=nsamps, kind="uniform2")
    _check(w)


def test_extreme_values_all_threes():
    # every pair sum is 6, every output 3 * nchans: all three planes of a row and the carries are exercised
    w = HTRU.scaled(ndm=40, dm_hi=STEP * 39, nsamps_out=2000)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    stride = (w.nsamps_out + md + 3) // 4
    x = np.full((1, w.nchans, stride), 0xFF, dtype=np.uint8)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x, 2, w.nsamps_out)[0]
    assert np.all(got == 3 * w.nchans)
    dd.dedisp_destroy(p)


def test_unsorted_dm_list_with_duplicates():
    w = HTRU.scaled(nchans=256, ndm=90, dm_hi=STEP * 89, nsamps_out=2500)
    dms = np.random.default_rng(5).permutation(np.concatenate([w.dms()[:80], w.dms()[10:20]]))
    _check(w, dms=dms)


def test_batch_of_beams_equals_oracle_per_beam():
    w = HTRU.scaled(nchans=128, ndm=48, dm_hi=STEP * 47, nsamps_out=2100, nbeams=3)
    delay, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    for b in range(3):
        assert np.array_equal(got[b], oracle.dedisperse(delay, x[b], 2, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_many_channels_run_in_channel_blocks():
    # 2050 pairs x 6 > 8191: two blocks of pairs, the second adds to the partial sums in out
    w = HTRU.scaled(nchans=4100, df=-400.0 / 4100, ndm=40, dm_hi=30.0, nsamps_out=1500, kind="uniform2",
                    out_dtype="f32")
    _check(w, od="f32")


def test_pairs_equal_the_plain_tiled_kernel_and_repeat_calls():
    # same plan, kernel switched between calls: scratch buffers of both variants coexist
    w = HTRU.scaled(ndm=64, dm_lo=600.0, dm_hi=600.0 + STEP * 63, nsamps_out=3000)
    delay, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    a = gpu_dedisperse(p, x, 2, w.nsamps_out)
    dd.dedisp_set_kernel(p, dd.DEDISP_KERNEL_BITSLICE)
    b = gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_BITSLICE
    dd.dedisp_set_kernel(p, dd.DEDISP_KERNEL_PAIRS)
    c = gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert np.array_equal(a, b) and np.array_equal(a, c)
    assert np.array_equal(a[0], oracle.dedisperse(delay, x[0], 2, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_host_call_leaves_in_dm_group_ranges():
    w = HTRU.scaled(nchans=64, ndm=330, nsamps_out=3001, df=-6.0, dm_hi=15.0)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    out = torch.full((w.ndm, w.nsamps_out), -1, dtype=torch.int32).pin_memory()
    dd.dedisp_execute_host(p, 1, w.nsamps_out, torch.from_numpy(x).pin_memory(), 2, out, dd.DEDISP_OUT_U32)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    assert np.array_equal(out.numpy().view(np.uint32), oracle.dedisperse(delay, x, 2, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_plans_the_pair_rows_cannot_serve_are_refused_when_forced():
    # tiny config: one group of 32 trials spans > 100 delay differences of a pair; 1-bit samples
    w = W.CONFIGS["tiny"]
    delay, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    with pytest.raises(dd.DedispError) as e:
        gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    dd.dedisp_set_kernel(p, dd.DEDISP_KERNEL_AUTO)       # AUTO still serves the plan
    assert np.array_equal(gpu_dedisperse(p, x, 2, w.nsamps_out)[0], oracle.dedisperse(delay, x[0], 2, w.nsamps_out))
    dd.dedisp_destroy(p)
    w1 = HTRU.scaled(ndm=40, dm_hi=STEP * 39, nsamps_out=500, nbits=1, kind="uniform")
    _, md1, x1 = oracle_inputs(w1)
    p = make_plan(w1.nchans, w1.dt, w1.f_top, w1.df, w1.dms(), dd.DEDISP_KERNEL_PAIRS)
    with pytest.raises(dd.DedispError):      # pair rows exist for 2-, 4- and 8-bit samples
        gpu_dedisperse(p, x1, 1, w1.nsamps_out)
    dd.dedisp_destroy(p)


WIDE8 = W.CONFIGS["wide8"]
STEP8 = 2000.0 / 2047         # DM step of the wideband list


@pytest.mark.parametrize("nchans,dm_lo,ndm,nsamps,od", [
    (4096, 0.0, 40, 1500, "u32"), (4096, 1950.0, 50, 1409, "f32"), (1001, 900.0, 70, 3000, "u32"),
    (512, 1200.0, 33, 2817, "f32"), (2, 0.0, 3, 50, "u32"),
])
def test_eight_bit_pair_rows(nchans, dm_lo, ndm, nsamps, od):
    # 9-plane rows (Cfg9P): wideband channelisation, bottom and top of its DM range, odd channel count,
    # ragged tiles; bit-exact against the oracle
    w = WIDE8.scaled(nchans=nchans, ndm=ndm, dm_lo=dm_lo, dm_hi=dm_lo + STEP8 * (ndm - 1), nsamps_out=nsamps,
                     out_dtype=od)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x[None], 8, w.nsamps_out, od)[0]
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    want = oracle.dedisperse(delay, x, 8, w.nsamps_out)
    assert np.array_equal(got, want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


def test_eight_bit_delay_differences_beyond_one_word():
    # DM 4000 .. 4062 on the wideband channelisation: differences up to 39 samples, crossing the word boundary
    w = WIDE8.scaled(nchans=4096, ndm=64, dm_lo=4000.0, dm_hi=4000.0 + STEP8 * 63, nsamps_out=1500)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    delta = delay[1::2] - delay[0::2]
    assert np.any((delta.min(axis=1) < 32) & (delta.max(axis=1) >= 32))
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x[None], 8, w.nsamps_out)[0]
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    assert np.array_equal(got, oracle.dedisperse(delay, x, 8, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_eight_bit_extreme_values_and_beams():
    # all samples 255: every pair sum is 510 (all carries of the row adder), every output 255 * nchans
    w = WIDE8.scaled(nchans=4096, ndm=40, dm_hi=STEP8 * 39, nsamps_out=1000, nbeams=2)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = np.full((2, w.nchans, w.nsamps_out + md), 0xFF, dtype=np.uint8)
    x[1, ::3] = 0x80
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x, 8, w.nsamps_out)
    assert np.all(got[0] == 255 * w.nchans)
    assert np.array_equal(got[1], oracle.dedisperse(delay, x[1], 8, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_full_size_gulp_auto_takes_the_pair_rows_and_equals_the_plain_tiled_kernel():
    # BASELINE configs[1] at full size: AUTO = pair rows (checked against the oracle in test_gpu_fullsize.py);
    # here every output of the gulp against the plain tiled kernel on the same plan
    w = HTRU
    _, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    a = gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    dd.dedisp_set_kernel(p, dd.DEDISP_KERNEL_BITSLICE)
    b = gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_BITSLICE
    assert np.array_equal(a, b)
    dd.dedisp_destroy(p)


# ---------------------------------------------------------------- 4-bit samples (row f4): 5-plane rows (Cfg5P)
HTRU4 = W.CONFIGS["htru_gulp_4bit"]


@pytest.mark.parametrize("nchans,dm_lo,ndm,nsamps,od", [
    (1024, 0.0, 70, 3000, "u32"), (1024, 930.0, 84, 1409, "f32"), (1001, 480.0, 33, 2817, "u32"),
    (1024, 2050.0, 64, 1500, "u32"), (2, 0.0, 3, 50, "f32"),
])
def test_four_bit_pair_rows(nchans, dm_lo, ndm, nsamps, od):
    # 5-plane rows of two 4-bit channels: bottom, middle and top of the HTRU DM range, beyond it (delay
    # differences across a word boundary), odd channel count, ragged tiles; bit-exact against the oracle
    w = HTRU4.scaled(nchans=nchans, ndm=ndm, dm_lo=dm_lo, dm_hi=dm_lo + STEP * (ndm - 1), nsamps_out=nsamps,
                     out_dtype=od)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x[None], 4, w.nsamps_out, od)[0]
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    want = oracle.dedisperse(delay, x, 4, w.nsamps_out)
    assert np.array_equal(got, want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


def test_four_bit_extreme_values_and_beams():
    # all samples 15: every pair sum is 30 (all five planes of a row), every output 15 * nchans
    w = HTRU4.scaled(ndm=40, dm_hi=STEP * 39, nsamps_out=1000, nbeams=2)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = np.full((2, w.nchans, (w.nsamps_out + md + 1) // 2), 0xFF, dtype=np.uint8)
    x[1, ::3] = 0x8F
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    got = gpu_dedisperse(p, x, 4, w.nsamps_out)
    assert np.all(got[0] == 15 * w.nchans)
    assert np.array_equal(got[1], oracle.dedisperse(delay, x[1], 4, w.nsamps_out))
    dd.dedisp_destroy(p)


def test_four_bit_pairs_equal_the_plain_tiled_kernel_at_full_size():
    w = HTRU4
    _, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    a = gpu_dedisperse(p, x, 4, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    dd.dedisp_set_kernel(p, dd.DEDISP_KERNEL_BITSLICE)
    b = gpu_dedisperse(p, x, 4, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_BITSLICE
    assert np.array_equal(a, b)
    dd.dedisp_destroy(p)


def test_auto_falls_back_to_the_planes_when_the_row_scratch_cannot_be_allocated():
    # the gulp's rows need 373 MB of scratch; with less than that free AUTO must still serve the call (plain tiled
    # kernel), a forced PAIRS plan reports the failed allocation, and once memory is back AUTO takes the rows again
    w = HTRU
    _, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    q = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_PAIRS)
    ref = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), dd.DEDISP_KERNEL_BITSLICE)
    want = gpu_dedisperse(ref, x, 2, w.nsamps_out)
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    filler = torch.empty(free - (700 << 20), dtype=torch.uint8, device="cuda")   # in + out + planes fit, rows do not
    try:
        got = gpu_dedisperse(p, x, 2, w.nsamps_out)
        assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_BITSLICE
        assert np.array_equal(got, want)
        with pytest.raises(dd.DedispError) as e:
            gpu_dedisperse(q, x, 2, w.nsamps_out)
        assert e.value.status == dd.DEDISP_ERR_ALLOC
    finally:
        del filler
        torch.cuda.empty_cache()
    got = gpu_dedisperse(p, x, 2, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    assert np.array_equal(got, want)
    for h in (p, q, ref):
        dd.dedisp_destroy(h)
