"""-m gpu: dedisp_search_events (rows f1 + f2 chained without materialising z; SURVEY.md Sec. 8(f) f1 "fusing the
S/N search would remove that write") against the two-call chain it replaces and against the oracle.

The event list must be IDENTICAL, field by field (peak values compared as float32 bit patterns), to
oracle.peak_finding.find_events applied to the z the DENSE pass writes, at the thresholds nsigma * rms the search itself
reports -- so every re-computed z value an event reads is bit-identical to what the dense pass writes (the dense z is
in turn checked against oracle.matched_filter within the f1 tolerance).  Low thresholds (1 sigma: a sixth of all
samples lie in events) make that a statement about a large share of z, not just about a few peaks.  The RMS of the
no-z pass (warp-autonomous kernel) and of the dense pass (CTA kernel) are both within 2^-20 of the definition; they sum
in a different order, so they are compared with that tolerance, not bit for bit."""
RMS_RTOL = 2.0 ** -19      # two values each within 2^-20 of the definition
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
from oracle import matched_filter as MF, peak_finding as PF  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402

WIDTHS = [1, 2, 4, 8, 16, 32, 64]


def _events(ev, cnt, cap):
    total = int(cnt[0].item())
    raw = ev[: min(total, cap)].cpu().numpy()
    out = np.empty(len(raw), dtype=PF.EVENT_DTYPE)
    for i, k in enumerate(("series", "t_start", "length", "t_peak")):
        out[k] = raw[:, i]
    out["peak"] = raw[:, 4].copy().view(np.float32)
    return total, out


def _same(got, want):
    assert len(got) == len(want)
    for k in ("series", "t_start", "length", "t_peak"):
        assert np.array_equal(got[k], want[k]), k
    assert np.array_equal(got["peak"].view(np.uint32), want["peak"].view(np.uint32)), "peak bits"


def _dense_chain(xd, x_dtype, nrows, n, radius, widths, x_max, nsigma, cap):
    s = torch.cuda.current_stream().cuda_stream
    ns = len(widths) * nrows
    nb, hb, ho = dd.dedisp_matched_filter_hint_blocks(n, widths)
    z = torch.empty((len(widths), nrows, n), dtype=torch.float32, device="cuda")
    rms = torch.empty(ns, dtype=torch.float32, device="cuda")
    hint = torch.empty((ns, nb), dtype=torch.int32, device="cuda")
    mwb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, len(widths))
    mws = torch.empty(mwb, dtype=torch.uint8, device="cuda")
    dd.dedisp_matched_filter_rms(xd, x_dtype, nrows, n, radius, widths, x_max, z, rms, mws, mwb, s, blockmax_ptr=hint)
    wsb = dd.dedisp_find_events_workspace_bytes(ns, n)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    ev = torch.zeros((cap, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    dd.dedisp_find_events_hinted(z, ns, n, rms, nsigma, hint, hb, ho, ws, wsb, ev, cap, cnt, s)
    torch.cuda.synchronize()
    return z, rms, hint, _events(ev, cnt, cap)


def _search(xd, x_dtype, nrows, n, radius, widths, x_max, nsigma, cap, max_blocks):
    s = torch.cuda.current_stream().cuda_stream
    ns = len(widths) * nrows
    wsb = dd.dedisp_search_events_workspace_bytes(nrows, n, widths, max_blocks)
    assert wsb > 0
    ws = torch.full((wsb,), 0xA5, dtype=torch.uint8, device="cuda")     # garbage: nothing may rely on zeroed scratch
    rms = torch.empty(ns, dtype=torch.float32, device="cuda")
    ev = torch.zeros((cap, 5), dtype=torch.int32, device="cuda")
    cnt = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    dd.dedisp_search_events(xd, x_dtype, nrows, n, radius, widths, x_max, nsigma, rms, max_blocks, ws, wsb, ev, cap, cnt, s)
    torch.cuda.synchronize()
    return rms, int(cnt[1].item()), _events(ev, cnt, cap)


@pytest.mark.parametrize("nsigma", [1.0, 3.0, 6.0])
@pytest.mark.parametrize("shape,radius,widths,x_max", [
    ((6, 40001), 700, WIDTHS, 3072),              # 32-bit sums, ragged last block, 3 segments
    ((3, 70000), 15625, WIDTHS, 3072),            # the bench's 2 s window: guarded 32-bit sums
    ((2, 30011), 4000, [1, 3, 100, 2500], 3072),  # a width beyond one 2048-sample step: history of two steps
    ((1, 700), 100, [1, 2, 4], 3072),             # one row shorter than a segment; prefix sums of 3 blocks
    ((2, 2049), 1000, [1, 5, 64], 3072),          # one sample beyond a 2048-block; odd length: scalar paths
    ((1, 257), 128, [1, 4], 3072),                # the window IS the series (N = n = 257)
    ((3, 12288), 6000, [4, 8, 16], 3072),         # only widths that are multiples of 4; whole segments
])
def test_search_events_equals_the_dense_chain_and_the_oracle(shape, radius, widths, x_max, nsigma):
    x = W.dedispersed_like(91, shape[0], shape[1], npulses=6)
    nrows, n = x.shape
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    cap = 1 << 20
    z, rms_d, hint, (tot_d, ev_d) = _dense_chain(xd, dd.DEDISP_OUT_U32, nrows, n, radius, widths, x_max, nsigma, cap)
    nb = hint.shape[1]
    rms_s, flagged, (tot_s, ev_s) = _search(xd, dd.DEDISP_OUT_U32, nrows, n, radius, widths, x_max, nsigma, cap,
                                            max_blocks=len(widths) * nrows * nb)
    assert np.allclose(rms_s.cpu().numpy(), rms_d.cpu().numpy(), rtol=RMS_RTOL, atol=0)
    assert tot_s <= cap and (tot_s > 0 or nsigma > 3.0 or n < 3000)
    zh = z.cpu().numpy().reshape(-1, n)
    assert np.allclose(rms_s.cpu().numpy(), PF.series_rms(zh), rtol=2.0 ** -20, atol=0)
    want = PF.find_events(zh, rms_s.cpu().numpy(), nsigma)
    assert tot_s == len(want)
    _same(ev_s, want)
    _same(ev_d, PF.find_events(zh, rms_d.cpu().numpy(), nsigma))      # the dense chain, at its own thresholds
    # and z itself is the oracle's within the f1 tolerance (the chain starts from the definition)
    zw = MF.matched_filter(x, radius, widths).reshape(-1, n)
    assert np.all(np.abs(zh - zw) <= 2.0 ** -22 * np.abs(zw))
    # blocks flagged = blocks whose maximum exceeds the float32 threshold
    thr = (np.float32(nsigma) * rms_s.cpu().numpy()).astype(np.float32)
    ordered = np.where(thr.view(np.int32) >= 0, thr.view(np.int32), thr.view(np.int32) ^ 0x7fffffff)
    assert flagged == int((hint.cpu().numpy() > ordered[:, None]).sum())


def test_float32_input_and_64bit_sums():
    # 8-bit wideband range with a long window: 64-bit prefix sums; x given as float32 (exact integers)
    x = W.dedispersed_like(17, 3, 30000, mean=524288.0, sigma=1024.0, x_max=1044480, wiggle=900.0, npulses=5)
    nrows, n = x.shape
    xd = torch.from_numpy(x.astype(np.float32)).cuda()
    widths = [1, 8, 64]
    z, rms_d, hint, (tot_d, ev_d) = _dense_chain(xd, dd.DEDISP_OUT_F32, nrows, n, 5000, widths, 1044480, 3.5, 1 << 18)
    rms_s, _, (tot_s, ev_s) = _search(xd, dd.DEDISP_OUT_F32, nrows, n, 5000, widths, 1044480, 3.5, 1 << 18,
                                      max_blocks=len(widths) * nrows * hint.shape[1])
    want = PF.find_events(z.cpu().numpy().reshape(-1, n), rms_s.cpu().numpy(), 3.5)
    assert tot_s == len(want) > 0
    _same(ev_s, want)
    assert np.allclose(rms_s.cpu().numpy(), rms_d.cpu().numpy(), rtol=RMS_RTOL, atol=0)


def test_capacity_of_the_compact_z_is_reported_and_event_capacity_truncates():
    x = W.dedispersed_like(5, 4, 20000, npulses=8)
    nrows, n = x.shape
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    z, _, hint, _ = _dense_chain(xd, dd.DEDISP_OUT_U32, nrows, n, 500, WIDTHS, 3072, 4.0, 1 << 16)
    # too few compact blocks: count[1] says how many are needed; a second call with that capacity is complete
    rms_s, flagged, (tot_few, _) = _search(xd, dd.DEDISP_OUT_U32, nrows, n, 500, WIDTHS, 3072, 4.0, 1 << 16, max_blocks=2)
    ev_d = PF.find_events(z.cpu().numpy().reshape(-1, n), rms_s.cpu().numpy(), 4.0)
    tot_d = len(ev_d)
    assert flagged > 2 and tot_few <= tot_d
    _, flagged2, (tot_s, ev_s) = _search(xd, dd.DEDISP_OUT_U32, nrows, n, 500, WIDTHS, 3072, 4.0, 1 << 16,
                                         max_blocks=flagged)
    assert flagged2 == flagged and tot_s == tot_d
    _same(ev_s, ev_d)
    # event capacity: the first `cap` events, the total still reported
    _, _, (tot_c, ev_c) = _search(xd, dd.DEDISP_OUT_U32, nrows, n, 500, WIDTHS, 3072, 4.0, 3, max_blocks=flagged)
    assert tot_c == tot_d and len(ev_c) == 3
    _same(ev_c, ev_d[:3])


def test_nothing_above_threshold_and_argument_errors():
    x = W.dedispersed_like(3, 2, 9000, npulses=0)
    nrows, n = x.shape
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    _, flagged, (tot, ev) = _search(xd, dd.DEDISP_OUT_U32, nrows, n, 300, [1, 4], 3072, 50.0, 16, max_blocks=4)
    assert flagged == 0 and tot == 0 and len(ev) == 0
    s = torch.cuda.current_stream().cuda_stream
    wsb = dd.dedisp_search_events_workspace_bytes(nrows, n, [1, 4], 4)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    rms = torch.empty(2 * nrows, dtype=torch.float32, device="cuda")
    evb = torch.zeros((16, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    assert dd.dedisp_search_events_workspace_bytes(nrows, n, [1, 4], 0) == 0
    assert dd.dedisp_search_events_workspace_bytes(nrows, n, [1, 0], 4) == 0
    for kw in (dict(wsb=wsb - 1), dict(max_blocks=5), dict(radius=n), dict(widths=[1, n + 1])):
        a = dict(radius=300, widths=[1, 4], max_blocks=4, wsb=wsb)
        a.update(kw)
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_search_events(xd, dd.DEDISP_OUT_U32, nrows, n, a["radius"], a["widths"], 3072, 5.0, rms,
                                    a["max_blocks"], ws, a["wsb"], evb, 16, cnt, s)
        assert e.value.status == dd.DEDISP_ERR_INVALID_ARG, kw
    # z_dev = NULL in dedisp_matched_filter_rms: RMS and block maxima without writing z
    nb, hb, ho = dd.dedisp_matched_filter_hint_blocks(n, [1, 4])
    hint = torch.empty((2 * nrows, nb), dtype=torch.int32, device="cuda")
    mwb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, 2)
    mws = torch.empty(mwb, dtype=torch.uint8, device="cuda")
    rms2 = torch.empty(2 * nrows, dtype=torch.float32, device="cuda")
    dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, nrows, n, 300, [1, 4], 3072, None, rms2, mws, mwb, s,
                                 blockmax_ptr=hint)
    z = torch.empty((2, nrows, n), dtype=torch.float32, device="cuda")
    rms3 = torch.empty_like(rms2)
    hint3 = torch.empty_like(hint)
    dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, nrows, n, 300, [1, 4], 3072, z, rms3, mws, mwb, s,
                                 blockmax_ptr=hint3)
    torch.cuda.synchronize()
    assert torch.allclose(rms2, rms3, rtol=RMS_RTOL, atol=0) and torch.equal(hint, hint3)   # maxima are exact
    with pytest.raises(dd.DedispError):      # the plain filter has nothing to return without z
        dd.dedisp_matched_filter(xd, dd.DEDISP_OUT_U32, nrows, n, 300, [1, 4], 3072, None, s)
