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
