"""GPU parity for dedispersion at reduced time resolution (row f4, reading R38): dedisp_execute_tscrunch
through the C ABI vs oracle/tscrunch.py, element by element, tolerance 0."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
from oracle import tscrunch as TS  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import make_plan  # noqa: E402

FAST = [(1, 2), (1, 4), (1, 8), (1, 16), (2, 2), (2, 4), (2, 8), (2, 16), (4, 2), (4, 4), (4, 8)]


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (no CPU fallback exists)"


def run_gpu(plan, k, packed, nbits, nout, f32=False, offset=0):
    """packed: uint8 [nbeams, nchans, stride] host.  offset: misalign the device input by this many bytes."""
    nbeams, nchans, stride = packed.shape
    ndm = dd.dedisp_get_ndm(plan)
    assert stride == dd.dedisp_get_in_row_stride_bytes_tscrunch(plan, k, nout, nbits)
    buf = torch.zeros(packed.size + 16, dtype=torch.uint8, device="cuda")
    x = buf[offset:offset + packed.size]
    x.copy_(torch.from_numpy(packed.reshape(-1)))
    out = torch.full((nbeams, ndm, nout), -7, dtype=torch.float32 if f32 else torch.int32, device="cuda")
    s = torch.cuda.current_stream()
    dd.dedisp_execute_tscrunch(plan, k, nbeams, nout, x, nchans * stride, nbits, out, ndm * nout * 4,
                               dd.DEDISP_OUT_F32 if f32 else dd.DEDISP_OUT_U32, s.cuda_stream)
    s.synchronize()
    res = out.cpu().numpy()
    return res if f32 else res.view(np.uint32)


def case(nchans, ndm, dm_hi, nout, nbits, k, seed, nbeams=1, dt=64e-6, f_top=1581.8, bw=400.0):
    """Cut-down HTRU-like shape on the coarse grid dt' = k*dt; returns (plan args, delay', packed)."""
    df = -bw / nchans
    dms = np.linspace(0.0, dm_hi, ndm)
    delay, md = oracle.delay_table(nchans, k * dt, f_top, df, dms)
    n_fine = k * (nout + md)
    packed = np.stack([W.random_small(seed + 17 * b, nchans, n_fine, nbits) for b in range(nbeams)])
    return (nchans, k * dt, f_top, df, dms), delay, packed


@pytest.mark.parametrize("nbits,k", FAST)
def test_bit_sliced_factors_equal_oracle(nbits, k):
    args, delay, packed = case(96, 70, 300.0, 4001, nbits, k, 100 * nbits + k)
    plan = make_plan(*args)
    got = run_gpu(plan, k, packed, nbits, 4001)
    assert dd.dedisp_get_last_kernel(plan) == dd.DEDISP_KERNEL_BITSLICE
    want = TS.dedisperse_tscrunch_bytes(delay, packed[0], nbits, k, 4001)
    assert np.array_equal(got[0], want)
    dd.dedisp_destroy(plan)


@pytest.mark.parametrize("offset", [1, 2, 3])
@pytest.mark.parametrize("nbits,k", [(2, 2), (2, 16), (1, 4), (4, 2)])
def test_unaligned_input_and_ragged_rows(nbits, k, offset):
    # odd row strides (tight rows) and a misaligned base pointer; several beams
    args, delay, packed = case(40, 33, 150.0, 1237, nbits, k, 7 + offset, nbeams=3)
    plan = make_plan(*args)
    got = run_gpu(plan, k, packed, nbits, 1237, offset=offset)
    for b in range(3):
        assert np.array_equal(got[b], TS.dedisperse_tscrunch_bytes(delay, packed[b], nbits, k, 1237))
    dd.dedisp_destroy(plan)


@pytest.mark.parametrize("nbits,k", [(2, 3), (2, 5), (1, 7), (4, 17), (8, 1), (2, 32), (1, 255)])
def test_other_factors_run_the_direct_kernel(nbits, k):
    args, delay, packed = case(24, 9, 80.0, 300, nbits, k, 50 + k)
    plan = make_plan(*args)
    got = run_gpu(plan, k, packed, nbits, 300)
    if k > 1:
        assert dd.dedisp_get_last_kernel(plan) == dd.DEDISP_KERNEL_DIRECT
    want = TS.dedisperse_tscrunch(delay, packed[0], nbits, k, 300)
    assert np.array_equal(got[0], want)
    dd.dedisp_destroy(plan)


def test_forced_direct_kernel_and_float_output():
    args, delay, packed = case(64, 20, 200.0, 999, 2, 4, 5)
    want = TS.dedisperse_tscrunch_bytes(delay, packed[0], 2, 4, 999)
    for kernel in (dd.DEDISP_KERNEL_DIRECT, dd.DEDISP_KERNEL_BITSLICE):
        plan = make_plan(*args, kernel=kernel)
        got = run_gpu(plan, 4, packed, 2, 999, f32=True)
        assert dd.dedisp_get_last_kernel(plan) == kernel
        assert got.dtype == np.float32 and np.array_equal(got[0], want.astype(np.float32))
        dd.dedisp_destroy(plan)


def test_many_channels_run_in_channel_blocks():
    # 2-bit x 16: block sums up to 48, 1500 channels => 72 000 >= 2^16 counter range: two channel blocks
    args, delay, packed = case(1500, 24, 60.0, 700, 2, 16, 9)
    plan = make_plan(*args)
    for f32 in (False, True):
        got = run_gpu(plan, 16, packed, 2, 700, f32=f32)
        assert dd.dedisp_get_last_kernel(plan) == dd.DEDISP_KERNEL_BITSLICE
        want = TS.dedisperse_tscrunch_bytes(delay, packed[0], 2, 16, 700)
        assert np.array_equal(got[0], want.astype(np.float32) if f32 else want)
    dd.dedisp_destroy(plan)


def test_hand_worked_example():
    # tests/test_tscrunch_pins.py::test_hand_worked_example, through the C ABI
    rows = ["00123112210323301010313010001232", "03223323011210301101113222230111",
            "30021003222332100112130230003221", "00120122033202211333122202230022"]
    packed = np.stack([W.pack_bits(np.array([int(ch) for ch in r], np.uint8), 2) for r in rows])[None]
    for kernel in (dd.DEDISP_KERNEL_AUTO, dd.DEDISP_KERNEL_DIRECT):
        plan = make_plan(4, 2e-3, 1500.0, -100.0, [0.0, 10.0, 25.0], kernel=kernel)
        assert dd.dedisp_get_max_delay(plan) == 13
        got = run_gpu(plan, 2, packed, 2, 3)
        assert got[0].tolist() == [[6, 12, 12], [12, 15, 17], [11, 7, 15]]
        dd.dedisp_destroy(plan)


def test_factor_one_is_dedisp_execute():
    args, delay, packed = case(48, 25, 120.0, 2000, 2, 1, 3)
    plan = make_plan(*args)
    got = run_gpu(plan, 1, packed, 2, 2000)
    assert np.array_equal(got[0], oracle.dedisperse(delay, packed[0], 2, 2000))
    assert dd.dedisp_get_in_row_stride_bytes_tscrunch(plan, 1, 2000, 2) == dd.dedisp_get_in_row_stride_bytes(plan, 2000, 2)
    dd.dedisp_destroy(plan)


def test_rejected_arguments():
    plan = make_plan(16, 128e-6, 1500.0, -10.0, [0.0, 10.0])
    x = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    out = torch.zeros((2, 64), dtype=torch.int32, device="cuda")
    for k, nbits, status in [(0, 2, dd.DEDISP_ERR_INVALID_ARG), (-2, 2, dd.DEDISP_ERR_INVALID_ARG),
                             (86, 2, dd.DEDISP_ERR_INVALID_ARG), (2, 8, dd.DEDISP_ERR_INVALID_ARG),
                             (18, 4, dd.DEDISP_ERR_INVALID_ARG), (2, 3, dd.DEDISP_ERR_UNSUPPORTED_NBITS)]:
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_execute_tscrunch(plan, k, 1, 64, x, 0, nbits, out, 0, dd.DEDISP_OUT_U32, 0)
        assert e.value.status == status, (k, nbits)
    assert dd.dedisp_get_in_row_stride_bytes_tscrunch(plan, 0, 64, 2) == 0
    dd.dedisp_destroy(plan)


@pytest.mark.parametrize("k", [2, 4])
def test_full_size_gulp_sampled_trials(k):
    # the HTRU gulp at its full size, in the launch configuration bench.py --tscrunch times:
    # 65 536 * k fine samples summed to 65 536 coarse output samples, 1200 trials; the oracle
    # computes sampled trials one by one
    w = W.CONFIGS["htru_gulp"]
    delay, md = oracle.delay_table(w.nchans, k * w.dt, w.f_top, w.df, w.dms())
    packed = W.generate(w, k * (w.nsamps_out + md) - w.nsamps_out)[None]
    plan = make_plan(w.nchans, k * w.dt, w.f_top, w.df, w.dms())
    got = run_gpu(plan, k, packed, 2, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(plan) == dd.DEDISP_KERNEL_BITSLICE
    want = np.zeros((w.ndm, w.nsamps_out), np.uint32)
    for d in (0, 1, 31, 32, 600, 777, 1198, 1199):
        TS.dedisperse_tscrunch_bytes(delay, packed[0], 2, k, w.nsamps_out, d_begin=d, d_end=d + 1, out=want)
        assert np.array_equal(got[0, d], want[d]), d
    # conservation over all trials: every output row sums the same samples as the prefix sums say
    s = TS.scrunch_rows(packed[0], 2, k, w.nsamps_out + md).astype(np.int64)
    pre = np.concatenate([np.zeros((w.nchans, 1), np.int64), np.cumsum(s, axis=1)], axis=1)
    rows = np.arange(w.nchans)[:, None]
    tot = (pre[rows, delay + w.nsamps_out] - pre[rows, delay]).sum(axis=0)
    assert np.array_equal(got[0].sum(axis=1, dtype=np.int64), tot)
    dd.dedisp_destroy(plan)
