"""GPU parity for row f3 (13-beam coincidence RFI mask): the CUDA kernel through
the C ABI vs ``oracle.rfi_mask`` -- masks must be IDENTICAL (float32 comparisons and a count)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
from oracle import rfi_mask as RM  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import gpu_dedisperse, make_plan, oracle_inputs  # noqa: E402


def gpu_mask(x, mean, sigma, nsigma, k, u32=False, offset=0):
    """x: [nbeams, nseries, n] host.  offset: shift the device buffer by this many elements to
    exercise the unaligned (scalar) path."""
    nb, ns, n = x.shape
    flat = np.ascontiguousarray(x.astype(np.uint32).view(np.int32) if u32 else x.astype(np.float32))
    buf = torch.zeros(flat.size + offset, dtype=torch.int32 if u32 else torch.float32, device="cuda")
    buf[offset:] = torch.from_numpy(flat.reshape(-1)).cuda()
    xd = buf[offset:]
    md = torch.from_numpy(np.ascontiguousarray(mean, dtype=np.float32)).cuda()
    sd = torch.from_numpy(np.ascontiguousarray(sigma, dtype=np.float32)).cuda()
    m = torch.full((ns, n), 7, dtype=torch.uint8, device="cuda")
    dd.dedisp_rfi_mask(xd, dd.DEDISP_OUT_U32 if u32 else dd.DEDISP_OUT_F32, nb, ns, n, ns * n * 4, md, sd,
                       float(nsigma), int(k), m, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return m.cpu().numpy()


def test_hand_worked_example():
    x = np.array([[10.0, 17.0, 12.0, 20.0, 11.0, 16.5], [9.0, 18.0, 15.9, 21.0, 16.1, 10.0],
                  [12.0, 11.0, 10.0, 19.0, 16.0, 30.0], [8.0, 10.0, 16.5, 17.0, 12.0, 16.25]],
                 dtype=np.float32)[:, None, :]
    mean, sigma = np.full((4, 1), 10.0, np.float32), np.full((4, 1), 2.0, np.float32)
    assert gpu_mask(x, mean, sigma, 3.0, 2)[0].tolist() == [0, 1, 0, 1, 0, 1]


@pytest.mark.parametrize("n,offset", [(4096, 0), (4099, 0), (4096, 1), (5, 0), (1, 3)])
@pytest.mark.parametrize("k", [1, 4, 13])
def test_thirteen_beams_random(n, offset, k):
    rng = np.random.default_rng(100 + n + offset)
    x = rng.standard_normal((13, 3, n)).astype(np.float32)
    x[5, 1, 0] = np.nan
    mean = (0.2 * rng.standard_normal((13, 3))).astype(np.float32)
    sigma = (0.5 + rng.random((13, 3))).astype(np.float32)
    want = RM.coincidence_mask(x, mean, sigma, 1.0, k)
    assert np.array_equal(gpu_mask(x, mean, sigma, 1.0, k, offset=offset), want)
    assert 0 < want.mean() < 1 or k == 13 or n < 10


def test_uint32_input_and_limits():
    x = W.dedispersed_like(41, 13 * 2, 3000).reshape(13, 2, 3000)
    mean = np.full((13, 2), 1536.0, np.float32)
    sigma = np.full((13, 2), 30.1, np.float32)
    want = RM.coincidence_mask(x.astype(np.float32), mean, sigma, 1.0, 4)
    assert np.array_equal(gpu_mask(x, mean, sigma, 1.0, 4, u32=True), want)
    assert np.all(gpu_mask(x, mean, sigma, 1.0, 0, u32=True) == 1)
    assert np.all(gpu_mask(x, mean, sigma, 1.0, 14, u32=True) == 0)


def test_dm0_trial_of_a_batched_dedispersion():
    """The use the paper describes: the 13 beams' zero-DM time series, straight out of one
    batched dedisp_execute_batch output (nseries = 1, beam stride = ndm * nsamps * 4)."""
    w = W.CONFIGS["beams13"].scaled(ndm=3, dm_hi=1000.0 * 2 / 1199, nsamps_out=4096)
    delay, md, packed = oracle_inputs(w)
    plan = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    nb = packed.shape[0]
    xin = torch.from_numpy(packed).cuda()
    out = torch.empty((nb, w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    dd.dedisp_execute_batch(plan, nb, w.nsamps_out, xin, packed.shape[1] * packed.shape[2], w.nbits, out,
                            w.ndm * w.nsamps_out * 4, dd.DEDISP_OUT_U32, s)
    mean = torch.full((nb, 1), 1536.0, device="cuda")
    sigma = torch.full((nb, 1), 30.1, device="cuda")
    m = torch.zeros((1, w.nsamps_out), dtype=torch.uint8, device="cuda")
    dd.dedisp_rfi_mask(out, dd.DEDISP_OUT_U32, nb, 1, w.nsamps_out, w.ndm * w.nsamps_out * 4, mean, sigma,
                       1.0, 4, m, s)
    torch.cuda.synchronize()
    dd.dedisp_destroy(plan)
    x0 = np.stack([oracle.dedisperse(delay, packed[b], w.nbits, w.nsamps_out)[0] for b in range(nb)])
    want = RM.coincidence_mask(x0[:, None, :].astype(np.float32), mean.cpu().numpy(), sigma.cpu().numpy(), 1.0, 4)
    assert np.array_equal(m.cpu().numpy(), want) and 0 < want.mean() < 0.5


def test_full_size_13_beams():
    nb, n = 13, 1 << 22
    x = torch.randn((nb, 1, n), generator=torch.Generator().manual_seed(3)).numpy()
    mean, sigma = np.zeros((nb, 1), np.float32), np.ones((nb, 1), np.float32)
    want = RM.coincidence_mask(x, mean, sigma, 2.0, 2)
    assert np.array_equal(gpu_mask(x, mean, sigma, 2.0, 2), want) and want.sum() > 1000


def test_argument_errors():
    x = torch.zeros((2, 1, 64), device="cuda")
    ms = torch.zeros((2, 1), device="cuda")
    m = torch.zeros((1, 64), dtype=torch.uint8, device="cuda")
    def st(*a):
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_rfi_mask(*a)
        return e.value.status
    assert st(x, 1, 0, 1, 64, 256, ms, ms, 3.0, 1, m) == dd.DEDISP_ERR_INVALID_ARG
    assert st(x, 1, 2, 1, 64, 100, ms, ms, 3.0, 1, m) == dd.DEDISP_ERR_INVALID_ARG     # stride < beam
    assert st(x, 9, 2, 1, 64, 256, ms, ms, 3.0, 1, m) == dd.DEDISP_ERR_UNSUPPORTED_DTYPE
    assert st(0, 1, 2, 1, 64, 256, ms, ms, 3.0, 1, m) == dd.DEDISP_ERR_INVALID_ARG


def test_beam_counts_of_subsets_summed_equal_the_mask():
    # the multi-GPU form on one GPU: counts of two disjoint beam subsets, summed (what the all-reduce does), thresholded
    rng = np.random.default_rng(31)
    nb, ns, n = 13, 2, 5003                      # odd length: scalar tail
    x = rng.standard_normal((nb, ns, n)).astype(np.float32)
    x[:, 0, 100:110] += 6.0
    mean = rng.normal(0, 0.1, (nb, ns)).astype(np.float32)
    sigma = rng.uniform(0.8, 1.2, (nb, ns)).astype(np.float32)
    s = torch.cuda.current_stream().cuda_stream
    tot = torch.zeros((ns, n), dtype=torch.uint8, device="cuda")
    for a, b in ((0, 7), (7, 13)):
        xd = torch.from_numpy(np.ascontiguousarray(x[a:b])).cuda()
        c = torch.full((ns, n), 99, dtype=torch.uint8, device="cuda")
        dd.dedisp_rfi_beam_counts(xd, dd.DEDISP_OUT_F32, b - a, ns, n, ns * n * 4, torch.from_numpy(mean[a:b]).cuda(),
                                  torch.from_numpy(sigma[a:b]).cuda(), 2.0, c, s)
        torch.cuda.synchronize()
        assert np.array_equal(c.cpu().numpy(), RM.beam_count(x[a:b], mean[a:b], sigma[a:b], 2.0).astype(np.uint8))
        tot += c
    for k in (1, 4, 13, 14, 0):
        m = torch.full((ns, n), 7, dtype=torch.uint8, device="cuda")
        dd.dedisp_rfi_mask_from_counts(tot, ns, n, k, m, s)
        torch.cuda.synchronize()
        assert np.array_equal(m.cpu().numpy(), RM.coincidence_mask(x, mean, sigma, 2.0, k)), k
    with pytest.raises(dd.DedispError):
        dd.dedisp_rfi_beam_counts(tot, dd.DEDISP_OUT_F32, 256, ns, n, ns * n * 4, tot, tot, 2.0, tot, s)


def test_veto_events_marks_events_with_a_masked_peak():
    from oracle import peak_finding as PF
    z = W.filtered_like(9, 5, 6000, npulses=6).astype(np.float32)
    sigma = PF.series_rms(z).astype(np.float32)
    want = PF.find_events(z, sigma, 3.0)
    assert len(want) > 20
    rng = np.random.default_rng(2)
    mask = (rng.random(6000) < 0.3).astype(np.uint8)
    zd, sd = torch.from_numpy(z).cuda(), torch.from_numpy(sigma).cuda()
    wsb = dd.dedisp_find_events_workspace_bytes(5, 6000)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    cap = 1 << 16
    ev = torch.zeros((cap, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    kept = torch.full((1,), -5, dtype=torch.int64, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    dd.dedisp_find_events(zd, 5, 6000, sd, 3.0, ws, wsb, ev, cap, cnt, s)
    dd.dedisp_veto_events(ev, cnt, cap, torch.from_numpy(mask).cuda(), 6000, kept, s)
    torch.cuda.synchronize()
    exp, nkept = RM.veto_events(want, mask)
    got = ev[: int(cnt.item())].cpu().numpy()
    assert int(kept.item()) == nkept and 0 < nkept < len(want)
    assert np.array_equal(got[:, 0], exp["series"]) and np.array_equal(got[:, 3], exp["t_peak"])
    dd.dedisp_veto_events(ev, cnt, cap, torch.ones(6000, dtype=torch.uint8, device="cuda"), 6000, kept, s)   # again
    torch.cuda.synchronize()
    assert int(kept.item()) == 0 and (ev[: int(cnt.item()), 0] < 0).all()
