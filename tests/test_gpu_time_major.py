"""GPU parity for row f4b: telescope-order stream -> channel-major rows, byte-exact vs the
oracle, and the chain stream -> transpose -> dedisperse vs the oracle chain."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
from oracle import time_major as TM  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
from gpu_helpers import gpu_dedisperse, make_plan  # noqa: E402


def gpu_tm(stream, nchans, nsamps, nbits):
    sd = torch.from_numpy(stream).cuda()
    stride = (nsamps * nbits + 7) // 8
    out = torch.full((nchans, stride), 0xAB, dtype=torch.uint8, device="cuda")
    dd.dedisp_transpose_time_major(sd, nchans, nsamps, nbits, out, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("nbits,nchans,nsamps", [
    (2, 1024, 3000), (2, 1024, 257), (2, 16, 1), (1, 32, 5), (1, 1024, 1001), (1, 96, 300), (4, 8, 7),
    (4, 1024, 777), (8, 4, 3), (8, 4096, 513), (2, 48, 1023), (1, 4096, 130),
    # rows of a multiple of 4 bytes (word-aligned store path), small and large grids, and a large ragged one
    (8, 4096, 516), (2, 1024, 4112), (1, 64, 96), (4, 40, 2056), (8, 100, 4100), (8, 1024, 40000), (8, 1024, 40001)])
def test_transpose_matches_oracle(nbits, nchans, nsamps):
    rng = np.random.default_rng(nbits * 7 + nchans + nsamps)
    stream = rng.integers(0, 256, nsamps * nchans * nbits // 8, dtype=np.uint8)
    assert np.array_equal(gpu_tm(stream, nchans, nsamps, nbits), TM.to_channel_major(stream, nchans, nsamps, nbits))


def test_stream_to_dedispersed_output():
    nchans, nbits, nso = 1024, 2, 5000
    dms = np.linspace(0, 60, 40)
    delay, md = oracle.delay_table(nchans, 64e-6, 1581.8, -0.390625, dms)
    n = nso + md
    stream = np.random.default_rng(3).integers(0, 256, n * nchans * nbits // 8, dtype=np.uint8)
    cm = TM.to_channel_major(stream, nchans, n, nbits)
    want = oracle.dedisperse(delay, cm, nbits, nso)
    p = make_plan(nchans, 64e-6, 1581.8, -0.390625, dms)
    got_cm = gpu_tm(stream, nchans, n, nbits)
    assert np.array_equal(gpu_dedisperse(p, got_cm[None], nbits, nso)[0], want)
    dd.dedisp_destroy(p)


def test_argument_errors():
    x = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    def st(*a):
        with pytest.raises(dd.DedispError) as e:
            dd.dedisp_transpose_time_major(*a)
        return e.value.status
    assert st(x, 12, 10, 2, x) == dd.DEDISP_ERR_INVALID_ARG          # 24 bits per time sample
    assert st(x, 16, 10, 3, x) == dd.DEDISP_ERR_UNSUPPORTED_NBITS
    assert st(x, 16, 0, 2, x) == dd.DEDISP_ERR_INVALID_ARG
    assert st(x.data_ptr() + 1, 16, 10, 2, x) == dd.DEDISP_ERR_INVALID_ARG
