"""-m gpu: dedisp_execute_static -- the dedispersion entry point that allocates nothing (bit planes in a fixed
32 MiB file-scope device array; include/dedisp.h) -- against the existing path (dedisp_execute) and the oracle.

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide other tests).  Tolerance 0, as
for every dedispersion test: out[d][t] = sum_c in[c][t + delay[c][d]] is an exact integer sum
(BASELINE.json:north_star).  Two calls in a row share the static array: a large call (the full HTRU gulp, 23.3 MB of
planes), then a smaller one with other data, sample width and shape -- stale contents of the first call must not
leak into the second."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402


def _both_paths(w, x, od):
    """(static result, existing-path result, device bytes the static call allocated, kernel the static call ran)."""
    f32 = od == "f32"
    code = dd.DEDISP_OUT_F32 if f32 else dd.DEDISP_OUT_U32
    ty = torch.float32 if f32 else torch.int32
    s = torch.cuda.current_stream().cuda_stream
    xin = torch.from_numpy(x).cuda()
    # existing path: plain tiled kernel, the plan's own cudaMalloc'ed scratch
    ref_plan = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    dd.dedisp_set_dm_list(ref_plan, list(w.dms()))
    dd.dedisp_set_kernel(ref_plan, dd.DEDISP_KERNEL_BITSLICE)
    ref = torch.full((w.ndm, w.nsamps_out), -7, dtype=ty, device="cuda")
    dd.dedisp_execute(ref_plan, w.nsamps_out, xin, w.nbits, ref, code, s)
    torch.cuda.synchronize()
    dd.dedisp_destroy(ref_plan)
    # new entry point: a fresh plan (its scratch pointer is NULL: nothing but the static array can serve the call)
    plan = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    dd.dedisp_set_dm_list(plan, list(w.dms()))
    out = torch.full((w.ndm, w.nsamps_out), -7, dtype=ty, device="cuda")
    dd.dedisp_execute_static(plan, w.nsamps_out, xin, w.nbits, out, code, s)
    torch.cuda.synchronize()
    first = out.cpu().numpy()
    # the same call again: by now the module that holds the array is loaded (CUDA loads modules lazily, so the very
    # first call on a device is when the driver reserves the 32 MiB), and the free device memory must not move
    out.fill_(-7)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    dd.dedisp_execute_static(plan, w.nsamps_out, xin, w.nbits, out, code, s)
    torch.cuda.synchronize()
    grown = free0 - torch.cuda.mem_get_info()[0]
    kern = dd.dedisp_get_last_kernel(plan)
    dd.dedisp_destroy(plan)
    assert np.array_equal(out.cpu().numpy(), first)
    return first, ref.cpu().numpy(), grown, kern


def test_static_scratch_two_calls_in_a_row_equal_the_existing_path():
    assert dd.dedisp_static_scratch_bytes() == 32 << 20
    # call 1: the full HTRU gulp (BASELINE configs[1]) -- 23.3 MB of the 32 MiB
    w1 = W.CONFIGS["htru_gulp"]
    delay1, md1 = oracle.delay_table(w1.nchans, w1.dt, w1.f_top, w1.df, w1.dms())
    x1 = W.generate(w1, md1)
    got1, ref1, grown1, kern1 = _both_paths(w1, x1, "u32")
    assert kern1 == dd.DEDISP_KERNEL_BITSLICE
    assert np.array_equal(got1, ref1)
    rows = [0, 1, 599, 1199]      # and sampled rows against the oracle itself
    sub = oracle.dedisperse(np.ascontiguousarray(delay1[:, rows]), x1, 2, w1.nsamps_out)
    assert np.array_equal(got1.view(np.uint32)[rows], sub)
    # call 2, straight after, on the same static array: 8-bit samples, fewer channels, float32 output, ragged tile
    w2 = W.CONFIGS["wide8"].scaled(nchans=200, ndm=70, dm_hi=2000.0 * 69 / 2047, nsamps_out=3001, out_dtype="f32",
                                   seed=77)
    delay2, md2 = oracle.delay_table(w2.nchans, w2.dt, w2.f_top, w2.df, w2.dms())
    x2 = W.generate(w2, md2)
    got2, ref2, grown2, kern2 = _both_paths(w2, x2, "f32")
    assert kern2 == dd.DEDISP_KERNEL_BITSLICE
    assert np.array_equal(got2, ref2)
    assert np.array_equal(got2, oracle.to_f32(oracle.dedisperse(delay2, x2, 8, w2.nsamps_out)))
    # no call allocated device memory
    assert grown1 <= 0 and grown2 <= 0, (grown1, grown2)


def test_static_scratch_limit_and_argument_errors():
    s = torch.cuda.current_stream().cuda_stream
    # the 8-bit wideband config needs 750 MB of bit planes: refused with its own status, nothing launched
    w = W.CONFIGS["wide8"]
    plan = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    dd.dedisp_set_dm_list(plan, list(w.dms()))
    dummy = torch.zeros(16, dtype=torch.int32, device="cuda")
    n0 = dd.dedisp_get_launch_count()
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_execute_static(plan, w.nsamps_out, dummy, 8, dummy, dd.DEDISP_OUT_U32, s)
    assert e.value.status == dd.DEDISP_ERR_SCRATCH_LIMIT and "static scratch" in str(e.value)
    assert dd.dedisp_get_launch_count() == n0
    for bad, status in (((0, dummy, 8, dummy, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_INVALID_ARG),
                        ((16, dummy, 3, dummy, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_UNSUPPORTED_NBITS),
                        ((16, dummy, 8, dummy, 5), dd.DEDISP_ERR_UNSUPPORTED_DTYPE),
                        ((16, 0, 8, dummy, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_INVALID_ARG)):
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_execute_static(plan, bad[0], bad[1], bad[2], bad[3], bad[4], s)
        assert e.value.status == status, bad
    dd.dedisp_destroy(plan)
    p2 = dd.dedisp_plan_create(8, 64e-6, 1500.0, -10.0)
    with pytest.raises(dd.DedispError) as e:      # no DM list yet
        dd.dedisp_execute_static(p2, 16, dummy, 2, dummy, dd.DEDISP_OUT_U32, s)
    assert e.value.status == dd.DEDISP_ERR_NO_DM_LIST
    dd.dedisp_destroy(p2)
