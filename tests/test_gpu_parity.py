"""GPU parity: the CUDA path (through the C ABI) vs the CPU oracle, element by
element, tolerance 0 (integer sums; BASELINE.json:north_star "GPU output must be
bit-exact against the oracle")."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import gpu_dedisperse, make_plan, oracle_inputs  # noqa: E402

KERNELS = [dd.DEDISP_KERNEL_AUTO, dd.DEDISP_KERNEL_DIRECT]
TILED = (dd.DEDISP_KERNEL_BITSLICE, dd.DEDISP_KERNEL_PAIRS, dd.DEDISP_KERNEL_QUADS)   # the tiled kernel: planes, pair or quad rows


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device (no CPU fallback exists)"


# ------------------------------------------------------------ delay table (a1)
@pytest.mark.parametrize("name", ["tiny", "htru_gulp", "wide8"])
def test_device_delay_table_equals_oracle(name):
    w = W.CONFIGS[name]
    want, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    got = dd.dedisp_get_delay_table(p)
    assert dd.dedisp_get_max_delay(p) == md
    assert np.array_equal(got, want)
    assert dd.dedisp_get_in_row_stride_bytes(p, w.nsamps_out, w.nbits) == \
        oracle.row_stride_bytes(w.nsamps_out + md, w.nbits)
    dd.dedisp_destroy(p)


def test_delay_table_unsorted_duplicate_dms_and_reset():
    dms = [300.0, 0.0, 12.5, 300.0, 77.7, 1.0]
    want, md = oracle.delay_table(96, 64e-6, 1400.0, -3.0, dms)
    p = make_plan(96, 64e-6, 1400.0, -3.0, dms)
    assert np.array_equal(dd.dedisp_get_delay_table(p), want) and dd.dedisp_get_max_delay(p) == md
    dd.dedisp_set_dm_list(p, [5.0])      # replace the list
    want2, md2 = oracle.delay_table(96, 64e-6, 1400.0, -3.0, [5.0])
    assert np.array_equal(dd.dedisp_get_delay_table(p), want2) and dd.dedisp_get_max_delay(p) == md2
    dd.dedisp_destroy(p)


def test_delay_rounding_ties_away_on_device():
    K = 4148.808
    dms = [0.5, 1.5, 2.5, 3.5, 4.5]
    want, _ = oracle.delay_table(2, K * 0.75, 2.0, -1.0, dms)
    p = make_plan(2, K * 0.75, 2.0, -1.0, dms)
    got = dd.dedisp_get_delay_table(p)
    assert np.array_equal(got, want) and got[1, 0] == 1 and got[1, 2] == 3
    dd.dedisp_destroy(p)


# ------------------------------------------------------------ small cases
@pytest.mark.parametrize("kernel", KERNELS)
def test_hand_worked_example(kernel, golden_dir):
    from test_oracle_pins import _read_hand
    h = _read_hand(golden_dir)
    dms = [float(v) for v in h["dms"]]
    packed = np.array([[int(b, 16) for b in r] for r in h["packed"]], dtype=np.uint8)[None]
    want = np.array([[int(v) for v in r] for r in h["out"]], dtype=np.uint32)
    p = make_plan(4, 1e-3, 1500.0, -100.0, dms, kernel)
    assert np.array_equal(gpu_dedisperse(p, packed, 2, 6)[0], want)
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("out_dtype", ["u32", "f32"])
def test_tiny_config(kernel, out_dtype):
    w = W.CONFIGS["tiny"]
    delay, md, x = oracle_inputs(w)
    want = oracle.dedisperse(delay, x[0], 2, w.nsamps_out)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), kernel)
    got = gpu_dedisperse(p, x, 2, w.nsamps_out, out_dtype)[0]
    if out_dtype == "f32":
        assert got.dtype == np.float32 and np.array_equal(got, oracle.to_f32(want))
    else:
        assert np.array_equal(got, want)
    dd.dedisp_destroy(p)


SHAPES = [  # nchans, ndm, nsamps_out, nbits, dm_hi, df
    (1, 1, 1, 2, 0.0, -1.0), (3, 1, 5, 2, 50.0, -20.0), (37, 5, 333, 2, 120.0, -7.0),
    (64, 33, 4097, 2, 90.0, -4.0), (130, 70, 2049, 2, 300.0, -2.5), (100, 31, 1000, 8, 150.0, -3.0),
    (257, 3, 77, 8, 40.0, -1.0), (1024, 40, 3000, 2, 1000.0, -0.390625), (5, 64, 8192, 8, 10.0, -50.0),
    # row f4: 1- and 4-bit samples
    (1, 1, 1, 1, 0.0, -1.0), (37, 5, 333, 1, 120.0, -7.0), (64, 33, 4097, 1, 90.0, -4.0),
    (1024, 70, 5000, 1, 1000.0, -0.390625), (4096, 40, 2100, 1, 400.0, -0.09765625),
    (3, 1, 5, 4, 50.0, -20.0), (130, 70, 2049, 4, 300.0, -2.5), (1024, 40, 3000, 4, 1000.0, -0.390625),
    (4096, 33, 1300, 4, 400.0, -0.09765625),
]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape", SHAPES)
def test_random_shapes(kernel, shape):
    nchans, ndm, nso, nbits, dm_hi, df = shape
    dms = np.linspace(0.0, dm_hi, ndm)
    delay, md = oracle.delay_table(nchans, 64e-6, 1500.0, df, dms)
    x = W.random_small(nchans * 1000 + ndm, nchans, nso + md, nbits)
    want = oracle.dedisperse(delay, x, nbits, nso)
    p = make_plan(nchans, 64e-6, 1500.0, df, dms, kernel)
    for od in ("u32", "f32"):
        got = gpu_dedisperse(p, x[None], nbits, nso, od)[0]
        assert np.array_equal(got, want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("kernel", KERNELS)
def test_unsorted_dm_list_and_big_steps(kernel):
    dms = [250.0, 0.0, 999.0, 3.0, 3.0, 500.0, 42.0]
    delay, md = oracle.delay_table(200, 64e-6, 1500.0, -1.5, dms)
    x = W.random_small(99, 200, 1500 + md, 2)
    want = oracle.dedisperse(delay, x, 2, 1500)
    p = make_plan(200, 64e-6, 1500.0, -1.5, dms, kernel)
    assert np.array_equal(gpu_dedisperse(p, x[None], 2, 1500)[0], want)
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("kernel", KERNELS)
def test_extreme_values_and_impulse(kernel):
    w = W.CONFIGS["tiny"]
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    nin = w.nsamps_out + md
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), kernel)
    ones = np.full((1, w.nchans, W.row_stride_bytes(nin, 2)), 0xFF, np.uint8)
    assert (gpu_dedisperse(p, ones, 2, w.nsamps_out) == 3 * w.nchans).all()
    full8 = np.full((1, w.nchans, nin), 255, np.uint8)
    assert (gpu_dedisperse(p, full8, 8, w.nsamps_out) == 255 * w.nchans).all()
    u8 = np.zeros((w.nchans, nin), np.uint8)
    for c in range(w.nchans):
        u8[c, 1000 + delay[c, 16]] = 3
    got = gpu_dedisperse(p, np.stack([W.pack2(r) for r in u8])[None], 2, w.nsamps_out)[0]
    assert got[16, 1000] == 3 * w.nchans and (got == 3 * w.nchans).sum() == 1
    dd.dedisp_destroy(p)


def test_max_channels_8bit_no_overflow():
    # 4096 channels of 255: the largest sum the ABI admits (1 044 480 < 2^24), f32 exact
    dms = [0.0, 30.0]
    delay, md = oracle.delay_table(4096, 64e-6, 1500.0, -0.09765625, dms)
    x = np.full((1, 4096, 300 + md), 255, np.uint8)
    p = make_plan(4096, 64e-6, 1500.0, -0.09765625, dms)
    got = gpu_dedisperse(p, x, 8, 300, "f32")
    assert (got == np.float32(4096 * 255)).all()
    dd.dedisp_destroy(p)


# ------------------------------------------------------------ batch / strides / streams / host
@pytest.mark.parametrize("kernel", KERNELS)
def test_batch_with_padded_beam_strides_and_side_stream(kernel):
    w = W.CONFIGS["beams13"].scaled(nchans=48, ndm=40, nsamps_out=3000, df=-8.0, dm_hi=300.0)
    delay, md, x = oracle_inputs(w)
    nb, nch, stride = x.shape
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms(), kernel)
    in_bs, out_bs = nch * stride + 13, (w.ndm * w.nsamps_out + 5) * 4
    xin = torch.zeros(nb * in_bs, dtype=torch.uint8, device="cuda")
    for b in range(nb):
        xin[b * in_bs: b * in_bs + nch * stride] = torch.from_numpy(x[b].ravel()).cuda()
    out = torch.zeros(nb * out_bs // 4, dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        dd.dedisp_execute_batch(p, nb, w.nsamps_out, xin, in_bs, 2, out, out_bs, dd.DEDISP_OUT_U32,
                                s.cuda_stream)
    s.synchronize()
    got = out.cpu().numpy().view(np.uint32)
    for b in range(nb):
        want = oracle.dedisperse(delay, x[b], 2, w.nsamps_out)
        o = got[b * out_bs // 4: b * out_bs // 4 + w.ndm * w.nsamps_out].reshape(w.ndm, -1)
        assert np.array_equal(o, want), b
        assert not got[b * out_bs // 4 + w.ndm * w.nsamps_out: (b + 1) * out_bs // 4].any()
    dd.dedisp_destroy(p)


def test_unaligned_input_pointer():
    w = W.CONFIGS["tiny"]
    delay, md, x = oracle_inputs(w)
    want = oracle.dedisperse(delay, x[0], 2, w.nsamps_out)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    buf = torch.zeros(x.size + 16, dtype=torch.uint8, device="cuda")
    for off in (1, 3, 8):
        buf[off: off + x.size] = torch.from_numpy(x.ravel()).cuda()
        out = torch.zeros((w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
        dd.dedisp_execute(p, w.nsamps_out, buf.data_ptr() + off, 2, out, dd.DEDISP_OUT_U32,
                          torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), want), off
    dd.dedisp_destroy(p)


def test_execute_host_end_to_end():
    w = W.CONFIGS["beams13"].scaled(nchans=64, ndm=48, nsamps_out=5000, df=-6.0, dm_hi=200.0, nbeams=3)
    delay, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    xin = torch.from_numpy(x).pin_memory()
    for od, code in (("u32", dd.DEDISP_OUT_U32), ("f32", dd.DEDISP_OUT_F32)):
        out = torch.empty((3, w.ndm, w.nsamps_out),
                          dtype=torch.int32 if od == "u32" else torch.float32).pin_memory()
        dd.dedisp_execute_host(p, 3, w.nsamps_out, xin, 2, out, code)
        for b in range(3):
            want = oracle.dedisperse(delay, x[b], 2, w.nsamps_out)
            got = out[b].numpy()
            assert np.array_equal(got.view(np.uint32) if od == "u32" else got,
                                  want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("order", ["ascending", "shuffled", "direct"])
@pytest.mark.parametrize("ndm", [1, 33, 330, 1000])
def test_execute_host_single_beam_pieces(order, ndm):
    # one beam: ascending DM lists leave in up to 8 ranges of DM groups (copy overlapped with the kernel);
    # any other list, or the DIRECT kernel, takes the one-piece path.  All must equal the oracle.
    w = W.CONFIGS["htru_gulp"].scaled(nchans=64, ndm=ndm, nsamps_out=3001, df=-6.0, dm_hi=250.0)
    dms = w.dms()
    if order == "shuffled":
        dms = np.random.default_rng(ndm).permutation(dms)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, dms)
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, dms,
                  kernel=dd.DEDISP_KERNEL_DIRECT if order == "direct" else dd.DEDISP_KERNEL_AUTO)
    out = torch.full((ndm, w.nsamps_out), -1, dtype=torch.int32).pin_memory()
    for _ in range(2):      # the second call re-uses the staging buffers, streams and events
        out.fill_(-1)
        dd.dedisp_execute_host(p, 1, w.nsamps_out, torch.from_numpy(x).pin_memory(), 2, out, dd.DEDISP_OUT_U32)
        assert np.array_equal(out.numpy().view(np.uint32), oracle.dedisperse(delay, x, 2, w.nsamps_out))
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("nbits,nchans,od", [(2, 2048, "u32"), (2, 4100, "f32"), (1, 9000, "u32"), (4, 4400, "f32"),
                                             (8, 4200, "u32"), (8, 9000, "f32")])
def test_many_channels_run_in_channel_blocks(nbits, nchans, od):
    # sums beyond the counter planes of the bit-sliced kernel (e.g. 2-bit: 3 * nchans >= 4096): the channels
    # are summed in blocks and later blocks add to the partial sums in out -- still the bit-sliced kernel
    w = W.CONFIGS["htru_gulp"].scaled(nchans=nchans, nbits=nbits, ndm=40, nsamps_out=1500, df=-400.0 / nchans,
                                      dm_hi=60.0, kind="uniform", out_dtype=od)
    delay, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    got = gpu_dedisperse(p, x, nbits, w.nsamps_out, od)
    assert dd.dedisp_get_last_kernel(p) in TILED
    want = oracle.dedisperse(delay, x[0], nbits, w.nsamps_out)
    assert np.array_equal(got[0], want if od == "u32" else oracle.to_f32(want))
    dd.dedisp_destroy(p)


@pytest.mark.parametrize("nbits", [1, 2, 4, 8])
@pytest.mark.parametrize("ndm", [3, 20, 150, 400])
def test_coarse_dm_steps_stay_on_the_bit_sliced_kernel(nbits, ndm):
    # DM steps so coarse that the delays of 32 neighbouring trials do not fit a tile window: the groups
    # then hold 16, 8, ... 1 trials (idle lanes) instead of handing the plan to the DIRECT kernel
    w = W.CONFIGS["htru_gulp"].scaled(nchans=256, nbits=nbits, ndm=ndm, nsamps_out=2500, df=-400.0 / 256,
                                      kind="uniform")
    dms = np.random.default_rng(ndm).permutation(w.dms())          # and in any order
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, dms)
    x = W.generate(w, md)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, dms)
    got = gpu_dedisperse(p, x[None], nbits, w.nsamps_out)
    assert dd.dedisp_get_last_kernel(p) in TILED
    assert np.array_equal(got[0], oracle.dedisperse(delay, x, nbits, w.nsamps_out))
    out = torch.empty((ndm, w.nsamps_out), dtype=torch.int32).pin_memory()
    dd.dedisp_execute_host(p, 1, w.nsamps_out, torch.from_numpy(x).pin_memory(), nbits, out, dd.DEDISP_OUT_U32)
    assert np.array_equal(out.numpy().view(np.uint32), got[0])
    dd.dedisp_destroy(p)


def test_execute_host_many_beams():
    # more beams than the plan holds events for (16): one piece per beam
    w = W.CONFIGS["beams13"].scaled(nchans=32, ndm=40, nsamps_out=700, df=-12.0, dm_hi=100.0, nbeams=19)
    delay, md, x = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    out = torch.empty((19, w.ndm, w.nsamps_out), dtype=torch.float32).pin_memory()
    dd.dedisp_execute_host(p, 19, w.nsamps_out, torch.from_numpy(x).pin_memory(), 2, out, dd.DEDISP_OUT_F32)
    for b in range(19):
        assert np.array_equal(out[b].numpy(), oracle.to_f32(oracle.dedisperse(delay, x[b], 2, w.nsamps_out)))
    dd.dedisp_destroy(p)


def test_execute_errors():
    p = make_plan(8, 64e-6, 1500.0, -10.0, [0.0, 10.0])
    x = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    o = torch.zeros(1 << 16, dtype=torch.int32, device="cuda")
    cases = [((p, 100, x, 3, o, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_UNSUPPORTED_NBITS),
             ((p, 100, x, 2, o, 5), dd.DEDISP_ERR_UNSUPPORTED_DTYPE),
             ((p, 0, x, 2, o, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_INVALID_ARG),
             ((p, 100, 0, 2, o, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_INVALID_ARG),
             ((p, 100, x, 2, o.data_ptr() + 2, dd.DEDISP_OUT_U32), dd.DEDISP_ERR_INVALID_ARG)]
    for args, code in cases:
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_execute(*args)
        assert e.value.status == code
    dd.dedisp_destroy(p)
    big = make_plan(70000, 64e-6, 1500.0, -0.01, [0.0])
    with pytest.raises(dd.DedispError) as e:   # 70000*255 >= 2^24
        dd.dedisp_execute(big, 10, x, 8, o, dd.DEDISP_OUT_U32)
    assert e.value.status == dd.DEDISP_ERR_OVERFLOW
    dd.dedisp_destroy(big)


def test_launch_counter_and_probe():
    n0 = dd.dedisp_get_launch_count()
    p = make_plan(8, 64e-6, 1500.0, -10.0, [0.0, 10.0])
    assert dd.dedisp_get_launch_count() > n0
    dd.dedisp_destroy(p)
    import bench_probe
    bench_probe.build()
    r = bench_probe.probe_alu_rate(0)
    assert 1e12 < r < 1e15


@pytest.mark.parametrize("nbits", [1, 4])
def test_sub_byte_variants_use_the_tiled_kernel_and_extreme_values(nbits):
    """Row f4: HTRU channelisation with 1- and 4-bit samples runs on the bit-sliced kernel (not the
    DIRECT fallback); all-ones input gives nchans * (2^nbits - 1) everywhere."""
    w = W.CONFIGS["htru_gulp"].scaled(ndm=96, dm_hi=1000.0 * 95 / 1199, nsamps_out=6000)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.random_small(77 + nbits, w.nchans, w.nsamps_out + md, nbits)
    want = oracle.dedisperse(delay, x, nbits, w.nsamps_out)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    assert np.array_equal(gpu_dedisperse(p, x[None], nbits, w.nsamps_out)[0], want)
    assert dd.dedisp_get_last_kernel(p) in TILED
    assert np.array_equal(gpu_dedisperse(p, x[None], nbits, w.nsamps_out, "f32")[0], oracle.to_f32(want))
    ones = np.full_like(x, 0xFF)
    got = gpu_dedisperse(p, ones[None], nbits, w.nsamps_out)[0]
    assert np.all(got == w.nchans * ((1 << nbits) - 1))
    # two beams in one batched call, beam 1 = all ones
    both = np.stack([x, ones])
    got2 = gpu_dedisperse(p, both, nbits, w.nsamps_out)
    assert np.array_equal(got2[0], want) and np.all(got2[1] == w.nchans * ((1 << nbits) - 1))
    dd.dedisp_destroy(p)
    with pytest.raises(dd.DedispError) as e:
        p = make_plan(8, 64e-6, 1500.0, -1.0, [0.0])
        dd.dedisp_execute(p, 8, torch.zeros(64, dtype=torch.uint8, device="cuda"), 3,
                          torch.zeros(8, dtype=torch.int32, device="cuda"), dd.DEDISP_OUT_U32, 0)
    assert e.value.status == dd.DEDISP_ERR_UNSUPPORTED_NBITS


def test_cuda_graph_capture_and_replay():
    """execute only enqueues kernels (no allocation, no sync in the steady state), so a whole
    dedispersion step can be captured in a CUDA graph and replayed on new input."""
    w = W.CONFIGS["tiny"]
    delay, md, packed = oracle_inputs(w)
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = torch.from_numpy(packed[0]).cuda()
    out = torch.zeros((w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        dd.dedisp_execute(p, w.nsamps_out, x, w.nbits, out, dd.DEDISP_OUT_U32, side.cuda_stream)   # warm-up
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            dd.dedisp_execute(p, w.nsamps_out, x, w.nbits, out, dd.DEDISP_OUT_U32,
                              torch.cuda.current_stream().cuda_stream)
    want = oracle.dedisperse(delay, packed[0], w.nbits, w.nsamps_out)
    for trial in range(2):
        if trial == 1:      # new data in the same buffers
            packed2 = W.generate(w.scaled(seed=w.seed + 5), md)
            x.copy_(torch.from_numpy(packed2))
            want = oracle.dedisperse(delay, packed2, w.nbits, w.nsamps_out)
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), want)
    print("tiny kernel:", dd.dedisp_get_last_kernel(p))
    dd.dedisp_destroy(p)
