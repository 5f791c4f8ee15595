"""GPU parity for row f2 (sigma-cut + grouping into events): the CUDA kernels
through the C ABI vs ``oracle.peak_finding`` -- event lists must be IDENTICAL (comparisons
of float32 values and integer bookkeeping only); the RMS helper within 2^-22 relative
(float64 sums in a different order, one rounding to float32)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
from oracle import peak_finding as PF  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402


def gpu_events(z, sigma, nsigma, max_events=None):
    z = np.ascontiguousarray(z, dtype=np.float32)
    ns, n = z.shape
    zd = torch.from_numpy(z).cuda()
    sd = torch.from_numpy(np.asarray(sigma, dtype=np.float32)).cuda()
    wsb = dd.dedisp_find_events_workspace_bytes(ns, n)
    assert wsb > 0
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    cap = ns * n if max_events is None else max_events
    cap = min(cap, 4_000_000)
    ev = torch.zeros((max(cap, 1), 5), dtype=torch.int32, device="cuda")
    cnt = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    dd.dedisp_find_events(zd, ns, n, sd, float(nsigma), ws, wsb, ev if cap > 0 else None, cap, cnt,
                          torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    total = int(cnt.item())
    raw = ev[: min(total, cap)].cpu().numpy()
    out = np.empty(len(raw), dtype=PF.EVENT_DTYPE)
    for i, k in enumerate(("series", "t_start", "length", "t_peak")):
        out[k] = raw[:, i]
    out["peak"] = raw[:, 4].copy().view(np.float32)
    return total, out


def same(got, want):
    assert len(got) == len(want)
    for k in PF.EVENT_DTYPE.names:
        assert np.array_equal(got[k], want[k]), k


def test_hand_worked_example():
    z = np.array([[3.5, 4.0, 1.0, 3.0, 3.1, 0, 0, 5.0, 5.0, 4.0], [7.0, 0, 0, 0, 0, 0, 0, 0, 6.5, 7.5]],
                 dtype=np.float32)
    total, ev = gpu_events(z, [1.0, 2.0], 3.0)
    assert total == 5
    assert ev.tolist() == [(0, 0, 2, 1, 4.0), (0, 4, 1, 4, np.float32(3.1)), (0, 7, 3, 7, 5.0), (1, 0, 1, 0, 7.0),
                           (1, 8, 2, 9, 7.5)]


@pytest.mark.parametrize("nsigma", [0.0, 1.0, 3.0])
def test_dense_noise_every_event_identical(nsigma):
    z = W.filtered_like(31, 7, 5000, sigma=2.0)
    sigma = np.full(7, 2.0, dtype=np.float32)
    sigma[3] = 0.5
    total, ev = gpu_events(z, sigma, nsigma)
    want = PF.find_events(z, sigma, nsigma)
    assert total == len(want) > 100
    same(ev, want)


def test_long_runs_across_words_chunks_and_ends():
    n = 7000                                   # 6.8 chunks of 1024, ragged
    z = W.filtered_like(32, 6, n, sigma=1.0, npulses=6)
    z[0, :] = 50.0                             # the whole series is one run
    z[0, 4000] = 60.0
    z[1, :1500] = 40.0                         # run from the first sample across a chunk boundary
    z[2, 6000:] = 40.0                         # run to the last sample
    z[2, 6999] = 41.0
    z[3, 1023] = 99.0                          # single samples on either side of a chunk boundary
    z[3, 1024] = 98.0
    z[4, 31:33] = 77.0                         # across a word boundary
    z[5, 2048:3072] = 33.0                     # exactly one chunk
    total, ev = gpu_events(z, np.ones(6), 5.0)
    want = PF.find_events(z, np.ones(6), 5.0)
    assert total == len(want)
    same(ev, want)
    assert (0, 0, n, 4000, 60.0) == tuple(ev[0])


def test_capacity_truncates_but_counts_all():
    z = W.filtered_like(33, 4, 3000, sigma=1.0)
    want = PF.find_events(z, np.ones(4), 1.0)
    total, ev = gpu_events(z, np.ones(4), 1.0, max_events=37)
    assert total == len(want) > 37 and len(ev) == 37
    same(ev, want[:37])
    total, ev = gpu_events(z, np.ones(4), 1.0, max_events=0)
    assert total == len(want) and len(ev) == 0


def test_odd_sizes_nan_and_nothing_found():
    z = W.filtered_like(34, 3, 1, sigma=1.0, npulses=0)
    total, ev = gpu_events(z, np.ones(3), -10.0)
    same(ev, PF.find_events(z, np.ones(3), -10.0))
    assert total == 3
    z = W.filtered_like(35, 2, 33, sigma=1.0, npulses=1)
    z[0, 5] = np.nan
    z[1, 32] = 100.0
    total, ev = gpu_events(z, np.ones(2), 0.5)
    same(ev, PF.find_events(z, np.ones(2), 0.5))
    total, ev = gpu_events(np.zeros((5, 2049), np.float32), np.ones(5), 1.0)
    assert total == 0 and len(ev) == 0
    # a value equal to the float32 threshold product is not above it
    s, k = np.float32(0.1), np.float32(3.0)
    z = np.array([[s * k, np.nextafter(s * k, np.float32(1))]], dtype=np.float32)
    total, ev = gpu_events(z, [s], k)
    assert total == 1 and ev["t_start"][0] == 1


def test_series_rms():
    z = W.filtered_like(36, 9, 40001, sigma=30.1)
    zd = torch.from_numpy(z).cuda()
    r = torch.zeros(9, dtype=torch.float32, device="cuda")
    dd.dedisp_series_rms(zd, 9, 40001, r, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    np.testing.assert_allclose(r.cpu().numpy().astype(np.float64), PF.series_rms(z), rtol=2.0 ** -22, atol=0)
    zc = torch.full((2, 64), 3.0, device="cuda")
    dd.dedisp_series_rms(zc, 2, 64, r, 0)
    torch.cuda.synchronize()
    assert r[:2].tolist() == [3.0, 3.0]


def test_argument_errors():
    z = torch.zeros((2, 100), device="cuda")
    sg = torch.ones(2, device="cuda")
    wsb = dd.dedisp_find_events_workspace_bytes(2, 100)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    ev = torch.zeros((10, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    def st(*a):
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_find_events(*a)
        return e.value.status
    assert st(z, 2, 100, sg, 1.0, ws, wsb - 1, ev, 10, cnt) == dd.DEDISP_ERR_INVALID_ARG
    assert st(z, 0, 100, sg, 1.0, ws, wsb, ev, 10, cnt) == dd.DEDISP_ERR_INVALID_ARG
    assert st(z, 2, 100, sg, 1.0, ws, wsb, None, 10, cnt) == dd.DEDISP_ERR_INVALID_ARG
    assert st(z, 2, 100, sg, 1.0, ws, wsb, ev, -1, cnt) == dd.DEDISP_ERR_INVALID_ARG
    assert dd.dedisp_find_events_workspace_bytes(0, 5) == 0
    assert dd.dedisp_find_events_workspace_bytes(1, (1 << 30) + 1) == 0


def test_full_size_filtered_gulp():
    """7 widths x 1200 DM rows = 8400 series x 65536 samples, the bench's launch configuration:
    the total is checked against a vectorised rising-edge count over the whole array, the event
    records against the oracle on 40 sampled series."""
    ns, n = 8400, 65536
    g = torch.Generator().manual_seed(7)
    z = torch.randn((ns, n), generator=g, dtype=torch.float32).numpy() * np.float32(30.1)
    rows = sorted(set(np.linspace(0, ns - 1, 40).astype(int)))
    z[rows] = W.filtered_like(37, len(rows), n)
    sigma = np.full(ns, 30.1, dtype=np.float32)
    total, ev = gpu_events(z, sigma, 4.5)
    thr = np.float32(4.5) * np.float32(30.1)
    m = z > thr
    edges = int(m[:, 0].sum() + (m[:, 1:] & ~m[:, :-1]).sum())
    assert total == edges == len(ev)
    want = PF.find_events(z[rows], sigma[rows], 4.5)
    want["series"] = np.array(rows, dtype=np.int32)[want["series"]]
    same(ev[np.isin(ev["series"], rows)], want)
    key = ev["series"].astype(np.int64) * n + ev["t_start"]
    assert np.all(np.diff(key) > 0)


# ---- dedisp_find_events_hinted: block maxima let the sigma-cut skip chunks; the event list must not change ----
def ordered(x):
    """order-preserving int32 image of float32 values (include/dedisp.h, blockmax_dev)."""
    b = np.asarray(x, np.float32).view(np.int32)
    return np.where(b >= 0, b, b ^ 0x7FFFFFFF).astype(np.int32)


def gpu_events_hinted(z, sigma, nsigma, hint, hint_block, hint_offset):
    z = np.ascontiguousarray(z, dtype=np.float32)
    ns, n = z.shape
    zd = torch.from_numpy(z).cuda()
    sd = torch.from_numpy(np.asarray(sigma, dtype=np.float32)).cuda()
    hd = torch.from_numpy(np.ascontiguousarray(hint, dtype=np.int32)).cuda()
    wsb = dd.dedisp_find_events_workspace_bytes(ns, n)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    cap = min(ns * n, 4_000_000)
    ev = torch.zeros((cap, 5), dtype=torch.int32, device="cuda")
    cnt = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    dd.dedisp_find_events_hinted(zd, ns, n, sd, float(nsigma), hd, hint_block, hint_offset, ws, wsb, ev, cap, cnt,
                                 torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    total = int(cnt.item())
    raw = ev[: min(total, cap)].cpu().numpy()
    out = np.empty(len(raw), dtype=PF.EVENT_DTYPE)
    for i, k in enumerate(("series", "t_start", "length", "t_peak")):
        out[k] = raw[:, i]
    out["peak"] = raw[:, 4].copy().view(np.float32)
    return total, out


def exact_hint(z, block, offset):
    ns, n = z.shape
    nb = (n + offset + block - 1) // block
    h = np.full((ns, nb), np.iinfo(np.int32).min, np.int32)
    o = ordered(z)
    for b in range(nb):
        lo, hi = max(0, b * block - offset), min(n, (b + 1) * block - offset)
        if hi > lo:
            h[:, b] = o[:, lo:hi].max(axis=1)
    return h


@pytest.mark.parametrize("block,offset", [(2048, 64), (2048, 0), (100, 37), (5000, 4999), (1, 0)])
@pytest.mark.parametrize("nsigma", [2.0, 4.5, 50.0])
def test_hinted_events_equal_the_oracle(block, offset, nsigma):
    z = W.filtered_like(77, 6, 9001, npulses=5).astype(np.float32)
    z[2, 1020:1030] = 400.0            # runs across chunk (1024) and block boundaries
    z[4, 2040:2060] = 300.0
    z[5, -3:] = 500.0
    z[1, 0] = 600.0
    sigma = PF.series_rms(z).astype(np.float32)
    want = PF.find_events(z, sigma, nsigma)
    total, got = gpu_events_hinted(z, sigma, nsigma, exact_hint(z, block, offset), block, offset)
    assert total == len(want)
    same(got, want)
    # a looser (larger) hint is still valid
    total, got = gpu_events_hinted(z, sigma, nsigma, exact_hint(z, block, offset) + 12345, block, offset)
    assert total == len(want)
    same(got, want)


def test_matched_filter_hint_feeds_the_search():
    # the chain the bench times as --op search: matched_filter_rms (z, rms, block maxima) -> find_events_hinted
    from oracle import matched_filter as MF
    x = W.dedispersed_like(41, 6, 40001, npulses=6)
    widths = [1, 2, 4, 8, 16, 32, 64]
    nrows, n = x.shape
    nb, hb, ho = dd.dedisp_matched_filter_hint_blocks(n, widths)
    assert (hb, ho) == (2048, 64) and nb == (n + ho + hb - 1) // hb
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    z = torch.empty((len(widths), nrows, n), dtype=torch.float32, device="cuda")
    rms = torch.empty(len(widths) * nrows, dtype=torch.float32, device="cuda")
    hint = torch.zeros((len(widths) * nrows, nb), dtype=torch.int32, device="cuda")
    mwb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, len(widths))
    mws = torch.empty(mwb, dtype=torch.uint8, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, nrows, n, 700, widths, 3072, z, rms, mws, mwb, s, blockmax_ptr=hint)
    torch.cuda.synchronize()
    zh = z.cpu().numpy().reshape(-1, n)
    # the hint is exactly the block maxima of the z this call wrote
    assert np.array_equal(hint.cpu().numpy(), exact_hint(zh, hb, ho))
    sig = rms.cpu().numpy()
    for nsigma in (3.0, 6.0):
        want = PF.find_events(zh, sig, nsigma)
        total, got = gpu_events_hinted(zh, sig, nsigma, hint.cpu().numpy(), hb, ho)
        assert total == len(want) and (total > 0 or nsigma > 3.0)
        same(got, want)


def test_hinted_rejects_bad_arguments():
    z = torch.zeros((2, 64), dtype=torch.float32, device="cuda")
    sg = torch.ones(2, dtype=torch.float32, device="cuda")
    wsb = dd.dedisp_find_events_workspace_bytes(2, 64)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    h = torch.zeros((2, 1), dtype=torch.int32, device="cuda")
    for args in [(None, 64, 0), (h, 0, 0), (h, 64, -1)]:
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_find_events_hinted(z, 2, 64, sg, 5.0, args[0], args[1], args[2], ws, wsb, None, 0, cnt, 0)
        assert e.value.status == dd.DEDISP_ERR_INVALID_ARG


def test_matched_filter_hint_with_a_width_beyond_the_block():
    # widest boxcar 3000 > 2048-sample block: the first block of the hint covers no sample at all
    from oracle import matched_filter as MF
    x = W.dedispersed_like(43, 3, 20000, npulses=4)
    widths = [1, 3000]
    nrows, n = x.shape
    nb, hb, ho = dd.dedisp_matched_filter_hint_blocks(n, widths)
    assert (hb, ho) == (2048, 3000)
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    z = torch.empty((2, nrows, n), dtype=torch.float32, device="cuda")
    rms = torch.empty(2 * nrows, dtype=torch.float32, device="cuda")
    hint = torch.zeros((2 * nrows, nb), dtype=torch.int32, device="cuda")
    mwb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, 2)
    mws = torch.empty(mwb, dtype=torch.uint8, device="cuda")
    dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, nrows, n, 400, widths, 3072, z, rms, mws, mwb,
                                 torch.cuda.current_stream().cuda_stream, blockmax_ptr=hint)
    torch.cuda.synchronize()
    zh = z.cpu().numpy().reshape(-1, n)
    h = hint.cpu().numpy()
    assert (h[:, 1:] >= exact_hint(zh, hb, ho)[:, 1:]).all()
    for nsigma in (2.5, 5.0):
        want = PF.find_events(zh, rms.cpu().numpy(), nsigma)
        total, got = gpu_events_hinted(zh, rms.cpu().numpy(), nsigma, h, hb, ho)
        assert total == len(want)
        same(got, want)
