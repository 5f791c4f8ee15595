"""GPU parity for row f1 (baseline removal + boxcar matched filters):
the CUDA kernel through the C ABI vs ``oracle.matched_filter`` element by element.

Tolerance (R26): the kernel's integer numerators are exact; each
output is fl32(numerator) * fl32(1/(N sqrt(w))) = three float32 roundings, so
|got - want| <= ((1 + 2^-24)^3 - 1) |want| < 2^-22 |want|, and exact zeros stay zero."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
from oracle import matched_filter as MF  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import gpu_dedisperse, make_plan, oracle_inputs  # noqa: E402

RTOL = 2.0 ** -22


def gpu_mf(x, radius, widths, x_max, f32_in=False):
    x = np.ascontiguousarray(x)
    nrows, n = x.shape
    xd = torch.from_numpy(x.astype(np.float32) if f32_in else x.view(np.int32)).cuda()
    z = torch.full((len(widths), nrows, n), float("nan"), dtype=torch.float32, device="cuda")
    dd.dedisp_matched_filter(xd, dd.DEDISP_OUT_F32 if f32_in else dd.DEDISP_OUT_U32, nrows, n, radius,
                             widths, x_max, z, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return z.cpu().numpy()


def check(got, want):
    assert got.shape == want.shape and not np.isnan(got).any()
    err = np.abs(got.astype(np.float64) - want)
    bad = err > RTOL * np.abs(want)
    assert not bad.any(), f"{bad.sum()} of {bad.size} outside 2^-22 relative; worst {err.max()}"
    assert np.all(got[want == 0.0] == 0.0)


def test_hand_worked_example(golden_dir):
    x = np.array([[3, 1, 4, 1, 5, 9, 2, 6]], dtype=np.uint32)
    got = gpu_mf(x, 1, [1, 2, 4], 9)
    check(got, MF.matched_filter(x, 1, [1, 2, 4]))
    np.testing.assert_allclose(got[1, 0, :7], np.array([-4, 1, -1, -7, 11, 0, -10]) / (3 * np.sqrt(2)),
                               rtol=RTOL)


@pytest.mark.parametrize("f32_in", [False, True])
def test_random_rows_32bit_path(f32_in):
    x = W.dedispersed_like(21, 5, 5000)
    widths = [1, 2, 4, 8, 16, 32, 64]
    check(gpu_mf(x, 100, widths, 3072, f32_in), MF.matched_filter(x, 100, widths))


def test_several_segments_and_ragged_tail():
    x = W.dedispersed_like(22, 3, 40001)          # 3 segments of 16384, ragged, n % 4 != 0
    widths = [1, 3, 8, 50, 64]
    check(gpu_mf(x, 700, widths, 3072), MF.matched_filter(x, 700, widths))


def test_64bit_path_wideband_range():
    x = W.dedispersed_like(23, 2, 30000, mean=524288.0, sigma=1024.0, x_max=1044480, wiggle=3000.0)
    widths = [1, 2, 64, 512]
    check(gpu_mf(x, 2000, widths, 1044480), MF.matched_filter(x, 2000, widths))
    # same data with the default bound (x_max = 0 -> 2^24 - 1)
    check(gpu_mf(x, 2000, widths, 0), MF.matched_filter(x, 2000, widths))


def test_two_second_window_htru():
    """N = 31251 samples = 2 s at 64 us: the window is half the gulp; 64-bit numerators."""
    x = W.dedispersed_like(24, 2, 65536)
    widths = [1, 2, 4, 8, 16, 32, 64]
    check(gpu_mf(x, 15625, widths, 3072), MF.matched_filter(x, 15625, widths))


def test_guarded_32bit_path_spikes_force_exact_fallback():
    """N*x_max < 2^31 <= wmax*N*x_max: the guarded 32-bit kernel.  Rows 0-1 are noise (fast
    path); rows 2-3 carry runs of x_max over a zero floor whose boxcar numerators exceed 2^31,
    so the flagged steps must take the exact sample-by-sample fallback."""
    n, R = 40000, 15625
    x = W.dedispersed_like(28, 4, n)
    x[2:] = 0
    x[2, 20000:20064] = 3072                    # 64 * 31251 * 3072 = 6.1e9 > 2^31
    x[2, 36860:36870] = 3072                    # run straddling a step boundary region
    x[3, ::4096] = 3072
    x[3, 2040:2120] = 3072                      # across the first step boundary (E = 2048)
    widths = [1, 2, 4, 8, 16, 32, 64]
    want = MF.matched_filter(x, R, widths)
    assert np.abs(want[-1, 2] * (2 * R + 1) * 8).max() > 2 ** 31      # the bound really is crossed
    check(gpu_mf(x, R, widths, 3072), want)
    check(gpu_mf(x, R, widths, 3072, f32_in=True), want)


def test_edges_and_degenerate_cases():
    x = W.dedispersed_like(25, 2, 301, npulses=1)
    check(gpu_mf(x, 150, [1, 301], 3072), MF.matched_filter(x, 150, [1, 301]))   # N == n, w == n
    check(gpu_mf(x, 0, [1, 2], 3072), MF.matched_filter(x, 0, [1, 2]))           # R = 0: y == 0
    assert np.all(gpu_mf(x, 0, [1, 2], 3072) == 0)
    one = np.array([[7]], dtype=np.uint32)
    check(gpu_mf(one, 0, [1], 7), MF.matched_filter(one, 0, [1]))
    big = W.dedispersed_like(26, 1, 20000)
    check(gpu_mf(big, 10, [8192], 3072), MF.matched_filter(big, 10, [8192]))     # widest boxcar
    const = np.full((2, 5000), 1536, dtype=np.uint32)
    assert np.all(gpu_mf(const, 77, [1, 4, 64], 3072) == 0)


def test_argument_errors():
    x = torch.zeros((1, 100), dtype=torch.int32, device="cuda")
    z = torch.zeros((1, 1, 100), dtype=torch.float32, device="cuda")
    def st(*a):
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_matched_filter(*a)
        return e.value.status
    assert st(x, 0, 1, 100, 50, [1], 0, z) == dd.DEDISP_ERR_INVALID_ARG        # N > n
    assert st(x, 0, 1, 100, 1, [101], 0, z) == dd.DEDISP_ERR_INVALID_ARG       # w > n
    assert st(x, 0, 1, 100, 1, [0], 0, z) == dd.DEDISP_ERR_INVALID_ARG
    assert st(x, 0, 1, 100, 1, list(range(1, 18)), 0, z) == dd.DEDISP_ERR_INVALID_ARG
    assert st(x, 5, 1, 100, 1, [1], 0, z) == dd.DEDISP_ERR_UNSUPPORTED_DTYPE
    assert st(x, 0, 1, 100, 1, [1], 1 << 24, z) == dd.DEDISP_ERR_OVERFLOW
    assert st(0, 0, 1, 100, 1, [1], 0, z) == dd.DEDISP_ERR_INVALID_ARG


def test_chain_dedisperse_then_matched_filter():
    """The real chain: dedispersed output (device, u32 and f32) -> matched filter."""
    w = W.CONFIGS["htru_gulp"].scaled(ndm=40, dm_hi=1000.0 * 39 / 1199, nsamps_out=9000)
    delay, md, packed = oracle_inputs(w)
    want_x = oracle.dedisperse(delay, packed[0], w.nbits, w.nsamps_out)
    widths = [1, 2, 4, 8, 16, 32, 64]
    want = MF.matched_filter(want_x, 1000, widths)
    plan = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    for od in ("u32", "f32"):
        x = gpu_dedisperse(plan, packed, w.nbits, w.nsamps_out, od)[0]
        assert np.array_equal(x.astype(np.uint32), want_x)
        check(gpu_mf(x.astype(np.uint32), 1000, widths, 3 * w.nchans, f32_in=(od == "f32")), want)
    dd.dedisp_destroy(plan)


def test_full_size_htru_gulp_sampled_rows():
    """1200 rows x 65536 samples x 7 widths in the bench's launch configuration; the
    oracle checks 24 sampled rows (rows are independent)."""
    nrows, n, R = 1200, 65536, 15625
    widths = [1, 2, 4, 8, 16, 32, 64]
    rows = sorted(set(np.linspace(0, nrows - 1, 24).astype(int)))
    x = torch.randint(1400, 1700, (nrows, n), dtype=torch.int32,
                      generator=torch.Generator().manual_seed(5)).numpy().view(np.uint32).copy()
    x[rows] = W.dedispersed_like(27, len(rows), n)
    got = gpu_mf(x, R, widths, 3072)
    check(got[:, rows, :], MF.matched_filter(x[rows], R, widths))
    assert not np.isnan(got).any()


# ---- dedisp_matched_filter_rms: the same z plus the RMS of every filtered series in one pass ----
def gpu_mf_rms(x, radius, widths, x_max):
    x = np.ascontiguousarray(x)
    nrows, n = x.shape
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    z = torch.full((len(widths), nrows, n), float("nan"), dtype=torch.float32, device="cuda")
    rms = torch.full((len(widths) * nrows,), float("nan"), dtype=torch.float32, device="cuda")
    nb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, len(widths))
    assert nb > 0
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, nrows, n, radius, widths, x_max, z, rms, ws, nb,
                                 torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return z.cpu().numpy(), rms.cpu().numpy().reshape(len(widths), nrows), z


@pytest.mark.parametrize("shape,radius,widths,kw", [
    ((5, 5000), 100, [1, 2, 4, 8, 16, 32, 64], {}),                       # one segment, 32-bit words
    ((3, 40001), 700, [1, 3, 8, 50, 64], {}),                             # 3 segments, ragged tail
    ((2, 65536), 15625, [1, 2, 4, 8, 16, 32, 64], {}),                    # 2 s window: guarded 32-bit words
    ((2, 30000), 2000, [1, 2, 64, 512], dict(mean=524288.0, sigma=1024.0, x_max=1044480, wiggle=3000.0)),  # 64-bit
])
def test_fused_rms_equals_the_definition(shape, radius, widths, kw):
    from oracle import peak_finding as PF
    x = W.dedispersed_like(31, shape[0], shape[1], **kw)
    x_max = kw.get("x_max", 3072)
    want_z = MF.matched_filter(x, radius, widths)
    z, rms, zd = gpu_mf_rms(x, radius, widths, x_max)
    check(z, want_z)                                           # z is what dedisp_matched_filter writes
    assert np.array_equal(z, gpu_mf(x, radius, widths, x_max))
    # tolerance (include/dedisp.h): z within 2^-22 => z^2 within 2^-21; float32 partial sums of <= 64 squares
    # and float64 above => sum within ~2^-19.4, its square root within 2^-20
    want = PF.series_rms(want_z.reshape(-1, shape[1])).reshape(len(widths), shape[0])
    np.testing.assert_allclose(rms.astype(np.float64), want, rtol=2.0 ** -20, atol=0)
    # and against the stand-alone kernel on the z this call wrote
    r2 = torch.empty(len(widths) * shape[0], dtype=torch.float32, device="cuda")
    dd.dedisp_series_rms(zd, len(widths) * shape[0], shape[1], r2, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    np.testing.assert_allclose(rms.reshape(-1), r2.cpu().numpy(), rtol=2.0 ** -20, atol=0)


def test_fused_rms_is_deterministic_and_checks_its_arguments():
    x = W.dedispersed_like(32, 4, 33000)
    _, a, _ = gpu_mf_rms(x, 300, [1, 4, 16], 3072)
    _, b, _ = gpu_mf_rms(x, 300, [1, 4, 16], 3072)
    assert np.array_equal(a, b)
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    z = torch.empty((3, 4, 33000), dtype=torch.float32, device="cuda")
    rms = torch.empty(12, dtype=torch.float32, device="cuda")
    nb = dd.dedisp_matched_filter_rms_workspace_bytes(4, 33000, 3)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    for args in [(z, None, ws, nb), (z, rms, None, nb), (z, rms, ws, 8)]:
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, 4, 33000, 300, [1, 4, 16], 3072, *args, 0)
        assert e.value.status == dd.DEDISP_ERR_INVALID_ARG
    assert dd.dedisp_matched_filter_rms_workspace_bytes(0, 10, 1) == 0
