"""-m gpu tests of the plan's host-side contract (include/dedisp.h "Threading", "Streams and scratch"): two host
threads on two plans, two streams on one plan, CUDA-graph capture of the pair-row path, dedisp_reserve, launch limits.
Every result is compared with the oracle, tolerance 0 (BASELINE.json:north_star)."""
import threading

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import make_plan  # noqa: E402

HTRU = W.CONFIGS["htru_gulp"]
STEP = 1000.0 / 1199


def _pair_workload(seed=0, ndm=70, nsamps=4100, nchans=1024):
    w = HTRU.scaled(nchans=nchans, ndm=ndm, dm_lo=400.0, dm_hi=400.0 + STEP * (ndm - 1), nsamps_out=nsamps,
                    seed=HTRU.seed + seed)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    return w, delay, x


def test_two_host_threads_drive_two_plans():
    # the library's process-wide state (launch counter, per-kernel attribute flags) is atomic: two threads with a
    # plan and a stream each run the pair-row path and the plain tiled kernel at the same time
    cases = []
    for i, kern in enumerate((dd.DEDISP_KERNEL_PAIRS, dd.DEDISP_KERNEL_BITSLICE)):
        w, delay, x = _pair_workload(seed=i, ndm=64 + 6 * i, nsamps=3000 + 100 * i)
        cases.append((w, x, oracle.dedisperse(delay, x, 2, w.nsamps_out), kern))
    errors, n0 = [], dd.dedisp_get_launch_count()

    def worker(w, x, want, kern):
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), kern)
            xin = torch.from_numpy(x).cuda()
            for _ in range(6):
                out = torch.zeros((w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
                s.wait_stream(torch.cuda.current_stream())
                dd.dedisp_execute(p, w.nsamps_out, xin, 2, out, dd.DEDISP_OUT_U32, s.cuda_stream)
                s.synchronize()
                if not np.array_equal(out.cpu().numpy().view(np.uint32), want):
                    errors.append("mismatch")
            assert dd.dedisp_get_last_kernel(p) == kern
            dd.dedisp_destroy(p)
        except Exception as e:  # noqa: BLE001
            errors.append(repr(e))

    ts = [threading.Thread(target=worker, args=c) for c in cases]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    # every launch of both threads was counted (3 per pair-row execute, 2 per plain one, plus the table kernels)
    assert dd.dedisp_get_launch_count() - n0 >= 6 * 3 + 6 * 2


def test_two_streams_on_one_plan_are_ordered():
    # double-buffered caller: consecutive executes of ONE plan on alternating streams, no host synchronisation
    # in between; the plan's scratch (bit planes, pair rows) is re-used, so the second call must wait for the first
    w, delay, xa = _pair_workload(seed=1)
    _, _, xb = _pair_workload(seed=2)
    want = [oracle.dedisperse(delay, x, 2, w.nsamps_out) for x in (xa, xb)]
    for kern in (dd.DEDISP_KERNEL_PAIRS, dd.DEDISP_KERNEL_BITSLICE):
        p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), kern)
        xs = [torch.from_numpy(x).cuda() for x in (xa, xb)]
        outs = [torch.zeros((w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda") for _ in range(2)]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        torch.cuda.synchronize()
        for rep in range(4):
            for i in range(2):
                dd.dedisp_execute(p, w.nsamps_out, xs[i], 2, outs[i], dd.DEDISP_OUT_U32, streams[i].cuda_stream)
        torch.cuda.synchronize()
        for i in range(2):
            assert np.array_equal(outs[i].cpu().numpy().view(np.uint32), want[i]), (kern, i)
        dd.dedisp_destroy(p)


def test_cuda_graph_of_the_pair_row_path_after_reserve():
    # the path bench.py times (pre-passes + pair-row kernel) under stream capture: dedisp_reserve sizes the scratch
    # first; without it a capture that would have to allocate is refused, not corrupted
    w, delay, x = _pair_workload(seed=3)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    xin = torch.from_numpy(x).cuda()
    out = torch.zeros((w.ndm, w.nsamps_out), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    fresh = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    with torch.cuda.stream(side):
        g0 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g0, stream=side):
            with pytest.raises(dd.DedispError) as e:     # scratch would grow inside the capture
                dd.dedisp_execute(fresh, w.nsamps_out, xin, 2, out, dd.DEDISP_OUT_F32, side.cuda_stream)
            assert e.value.status == dd.DEDISP_ERR_CUDA and e.value.cuda_error == 900   # StreamCaptureUnsupported
    dd.dedisp_destroy(fresh)
    dd.dedisp_reserve(p, 1, w.nsamps_out, 2)
    with torch.cuda.stream(side):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            dd.dedisp_execute(p, w.nsamps_out, xin, 2, out, dd.DEDISP_OUT_F32, side.cuda_stream)
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_PAIRS
    want = oracle.to_f32(oracle.dedisperse(delay, x, 2, w.nsamps_out))
    for trial in range(2):
        if trial == 1:
            _, _, x2 = _pair_workload(seed=4)
            xin.copy_(torch.from_numpy(x2))
            want = oracle.to_f32(oracle.dedisperse(delay, x2, 2, w.nsamps_out))
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), want)
    # an ordinary execute on another stream after the capture still works (and is ordered by the plan)
    out2 = torch.zeros_like(out)
    dd.dedisp_execute(p, w.nsamps_out, xin, 2, out2, dd.DEDISP_OUT_F32, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(out2.cpu().numpy(), want)
    dd.dedisp_destroy(p)


def test_reserve_makes_execute_allocation_free_and_checks_arguments():
    w, delay, x = _pair_workload(seed=5, ndm=40, nsamps=2000, nchans=256)
    p = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_reserve(p, 1, w.nsamps_out, 2)
    assert e.value.status == dd.DEDISP_ERR_NO_DM_LIST
    dd.dedisp_set_dm_list(p, list(w.dms()))
    for bad in ((0, 100, 2), (1, 0, 2)):
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_reserve(p, *bad)
        assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_reserve(p, 1, 100, 3)
    assert e.value.status == dd.DEDISP_ERR_UNSUPPORTED_NBITS
    dd.dedisp_reserve(p, 2, w.nsamps_out, 2)
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    xin = torch.from_numpy(np.stack([x, x])).cuda()
    out = torch.zeros((2, w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
    mid = torch.cuda.mem_get_info()[0]
    dd.dedisp_execute_batch(p, 2, w.nsamps_out, xin, x.size, 2, out, w.ndm * w.nsamps_out * 4, dd.DEDISP_OUT_U32,
                            torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == mid <= before      # the execute itself allocated nothing
    want = oracle.dedisperse(delay, x, 2, w.nsamps_out)
    got = out.cpu().numpy().view(np.uint32)
    assert np.array_equal(got[0], want) and np.array_equal(got[1], want)
    dd.dedisp_destroy(p)


def test_more_beams_than_a_grid_dimension_fall_back_to_the_direct_kernel():
    # 65 536 beams of a 2-channel plan: beyond grid.z of the pre-pass; AUTO serves the call with the DIRECT kernel
    # (which loops over slabs of beams), a forced tiled kernel refuses it
    nb, ns = 65536, 8
    dms = [0.0, 1.0]
    delay, md = oracle.delay_table(2, 64e-6, 1500.0, -100.0, dms)
    stride = oracle.row_stride_bytes(ns + md, 2)
    rng = np.random.default_rng(9)
    x = rng.integers(0, 256, size=(nb, 2, stride), dtype=np.uint8)
    p = make_plan(2, 64e-6, 1500.0, -100.0, dms)
    xin = torch.from_numpy(x).cuda()
    out = torch.zeros((nb, 2, ns), dtype=torch.int32, device="cuda")
    dd.dedisp_execute_batch(p, nb, ns, xin, 2 * stride, 2, out, 2 * ns * 4, dd.DEDISP_OUT_U32,
                            torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert dd.dedisp_get_last_kernel(p) == dd.DEDISP_KERNEL_DIRECT
    got = out.cpu().numpy().view(np.uint32)
    for b in (0, 1, 40000, 65535):
        assert np.array_equal(got[b], oracle.dedisperse_literal(delay, x[b], 2, ns)), b
    dd.dedisp_set_kernel(p, dd.DEDISP_KERNEL_BITSLICE)
    with pytest.raises(dd.DedispError) as e:
        dd.dedisp_execute_batch(p, nb, ns, xin, 2 * stride, 2, out, 2 * ns * 4, dd.DEDISP_OUT_U32,
                                torch.cuda.current_stream().cuda_stream)
    assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    dd.dedisp_destroy(p)
