"""Full-size parity on the five BASELINE.json configs, in the launch configuration
bench.py times (default kernel selection, one execute / execute_batch call).

Checks per config: (1) sha256 + sum + spot values of the whole GPU output against
tests/golden/full_size.json (written from the oracle by make_golden.py);
(2) a sample of whole DM rows against the oracle run right here; (3) the
prefix-sum conservation identity on every row (holds at any size)."""
import hashlib
import json

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import oracle  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import gpu_dedisperse, make_plan, oracle_inputs  # noqa: E402


def _conservation(delay, packed, nbits, nso, got_row_sums):
    nchans, ndm = delay.shape
    nin = nso + int(delay.max())
    want = np.zeros(ndm, dtype=np.int64)
    for c in range(nchans):
        u8 = packed[c, :nin] if nbits == 8 else W.unpack2(packed[c], nin)
        S = np.concatenate([[0], np.cumsum(u8, dtype=np.int64)])
        want += S[nso + delay[c]] - S[delay[c]]
    assert np.array_equal(want, got_row_sums)


@pytest.mark.parametrize("name", W.CONFIG_ORDER)
def test_full_size_config(name, golden_dir):
    assert torch.cuda.is_available()
    gold = json.loads((golden_dir / "full_size.json").read_text())[name]
    w = W.CONFIGS[name]
    delay, md, x = oracle_inputs(w)
    assert md == gold["max_delay"] and W.sha256(x) == gold["in_sha256"]
    p = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    assert np.array_equal(dd.dedisp_get_delay_table(p), delay)
    got = gpu_dedisperse(p, x, w.nbits, w.nsamps_out, w.out_dtype)
    used = dd.dedisp_get_last_kernel(p)
    dd.dedisp_destroy(p)
    assert used in (dd.DEDISP_KERNEL_DIRECT, dd.DEDISP_KERNEL_BITSLICE, dd.DEDISP_KERNEL_PAIRS,
                    dd.DEDISP_KERNEL_QUADS)
    if name == "wide8":
        assert used == dd.DEDISP_KERNEL_QUADS      # 8-bit samples, 64 DM groups: the quad rows pay
    elif name != "tiny":
        assert used == dd.DEDISP_KERNEL_PAIRS      # the HTRU and wideband DM lists pay for the pair rows
    # (2) sampled whole rows, element by element against the oracle
    rows = sorted({0, 1, w.ndm // 3, w.ndm // 2, w.ndm - 2, w.ndm - 1} & set(range(w.ndm)))
    for b in sorted({0, w.nbeams - 1}):
        for d in rows:
            want = oracle.dedisperse(delay, x[b], w.nbits, w.nsamps_out, d_begin=d, d_end=d + 1)[d]
            wv = oracle.to_f32(want) if w.out_dtype == "f32" else want
            assert np.array_equal(got[b, d], wv), (b, d)
    # (3) conservation on every row of beam 0
    _conservation(delay, x[0], w.nbits, w.nsamps_out,
                  got[0].astype(np.int64).sum(axis=1) if w.out_dtype == "u32"
                  else got[0].astype(np.float64).sum(axis=1).astype(np.int64))
    # (1) whole-output golden
    for key, val in gold["spots"].items():
        b, d, t = (int(v) for v in key.split(","))
        assert int(got[b, d, t]) == val
    total = int(got.sum(dtype=np.uint64)) if w.out_dtype == "u32" else int(got.sum(dtype=np.float64))
    assert total == gold["out_sum"]
    assert int(got.min()) == gold["out_min"] and int(got.max()) == gold["out_max"]
    h = hashlib.sha256()
    for b in range(w.nbeams):
        h.update(np.ascontiguousarray(got[b]).tobytes())
    assert h.hexdigest() == gold["out_sha256"]
