"""Small invocations of every hazard-prone kernel path (SURVEY.md Sec. 4 tier T3, Sec. 5 "race detection":
"compute-sanitizer racecheck on the smem pipeline (mbarrier phases are the risk)").

    python tests/hazard_cases.py [case ...]                       # parity + guard zones + scratch poisoning
    DEDISP_B200_LIB=paper_1112_0065_b200/libdedisp_b200_checks.so python tests/hazard_cases.py   # + in-kernel checks
    compute-sanitizer --tool memcheck|racecheck|initcheck|synccheck python tests/hazard_cases.py  # where the tool exists

compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md), so the hazards it would look for are
checked by the library's own instrumentation instead.  Each case runs the CUDA path through the C ABI on a shape
chosen to reach one hazard and compares the result with the oracle, and in every case
  * the input sits at a byte offset inside a buffer of random bytes (a read outside the caller's rows changes sums),
  * the output sits between two canary zones that must come back untouched (out-of-bounds writes),
  * the plan's scratch is pre-filled with 0x00, 0xFF and 0xA5 in turn (dedisp_debug_set_poison): a kernel that
    consumes scratch words no pre-pass wrote (initcheck's job) cannot give the oracle's result for all three,
  * with the -DDEDISP_CHECKS build the in-kernel counters must stay zero: shared-memory read ranges, the
    (work item, chunk) tag of a ring stage before and after it is consumed (producer/consumer phase errors,
    racecheck's job), TMA source ranges, output row ranges.
tests/test_gpu_selfcheck.py runs both builds over all cases.  Cases:
  tiny_auto / tiny_direct   BASELINE configs[0] through the tiled kernel (plain planes, 1-D TMA) / the DIRECT kernel
  pairs3     cut-down HTRU shape at the top of the DM range: pair rows, 3 variants per slot, negative-x TMA boxes
  pairs8     8-bit wideband channelisation on 9-plane pair rows (Cfg9P)
  quads8     ... on 10-plane quad rows (Cfg10Q): per-variant box starts, boxes that begin before / end after a row
  blocks     4100 channels of 2-bit samples: channel blocks, the epilogue reads `out` back (accumulate)
  unaligned  input base pointer at odd byte offsets: the guarded 128-bit straddling loads of the unpack pre-pass
  multi      several persistent work items per CTA (the ring wraps many times) and a ragged last tile
  search     dedisp_matched_filter_rms + dedisp_find_events_hinted (rows f1 + f2)
  fault_injection   a deliberately wrong ring-stage tag must be counted by the checks build (the checks can fail)
"""
import sys
from pathlib import Path

import numpy as np
import torch

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
import oracle  # noqa: E402
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402

HTRU = W.CONFIGS["htru_gulp"]
STEP = 1000.0 / 1199
STEP8 = 2000.0 / 2047


POISONS = (0x00, 0xFF, 0xA5)
GUARD = 4096          # canary words on either side of the output
CANARY = -1234567


def _run(w, kernel, nbits, od="u32", offset=0, expect=None):
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    want = oracle.dedisperse(delay, x, nbits, w.nsamps_out)
    f32 = od == "f32"
    want = oracle.to_f32(want) if f32 else want
    p = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    dd.dedisp_set_dm_list(p, list(w.dms()))
    dd.dedisp_set_kernel(p, kernel)
    # input: at `offset` inside random bytes
    g = torch.Generator(device="cuda").manual_seed(7 + offset)
    buf = torch.randint(0, 256, (x.size + 64,), dtype=torch.uint8, device="cuda", generator=g)
    buf[offset: offset + x.size] = torch.from_numpy(x.ravel()).cuda()
    n = w.ndm * w.nsamps_out
    for poison in POISONS:
        dd.dedisp_debug_set_poison(p, poison)
        whole = torch.full((n + 2 * GUARD,), CANARY, dtype=torch.int32, device="cuda")
        out = whole[GUARD: GUARD + n]
        dd.dedisp_execute(p, w.nsamps_out, buf.data_ptr() + offset, nbits, out.data_ptr(),
                          dd.DEDISP_OUT_F32 if f32 else dd.DEDISP_OUT_U32, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        h = whole.cpu().numpy()
        assert (h[:GUARD] == CANARY).all() and (h[GUARD + n:] == CANARY).all(), "write outside out"
        got = h[GUARD: GUARD + n].reshape(w.ndm, w.nsamps_out)
        assert np.array_equal(got.view(np.float32) if f32 else got.view(np.uint32), want), f"poison {poison:#x}"
    if expect is not None:
        assert dd.dedisp_get_last_kernel(p) == expect, dd.dedisp_get_last_kernel(p)
    errs = dd.dedisp_debug_check_errors(p)
    assert errs[0] == 0, f"in-kernel checks failed: {errs}"
    dd.dedisp_destroy(p)


def tiny_auto():
    _run(W.CONFIGS["tiny"], dd.DEDISP_KERNEL_AUTO, 2, expect=dd.DEDISP_KERNEL_BITSLICE)


def tiny_direct():
    _run(W.CONFIGS["tiny"].scaled(nsamps_out=1000), dd.DEDISP_KERNEL_DIRECT, 2, expect=dd.DEDISP_KERNEL_DIRECT)


def pairs3():
    w = HTRU.scaled(ndm=84, dm_lo=930.0, dm_hi=930.0 + STEP * 83, nsamps_out=4100)
    _run(w, dd.DEDISP_KERNEL_PAIRS, 2, expect=dd.DEDISP_KERNEL_PAIRS)


def pairs8():
    w = W.CONFIGS["wide8"].scaled(nchans=1001, ndm=70, dm_lo=900.0, dm_hi=900.0 + STEP8 * 69, nsamps_out=3000)
    _run(w, dd.DEDISP_KERNEL_PAIRS, 8, expect=dd.DEDISP_KERNEL_PAIRS)


def quads8():
    w = W.CONFIGS["wide8"].scaled(nchans=1001, ndm=262, dm_lo=1744.0, dm_hi=1744.0 + STEP8 * 261, nsamps_out=3000)
    _run(w, dd.DEDISP_KERNEL_QUADS, 8, expect=dd.DEDISP_KERNEL_QUADS)
    w = W.CONFIGS["wide8"].scaled(nchans=64, ndm=256, dm_hi=STEP8 * 255, nsamps_out=1409)
    _run(w, dd.DEDISP_KERNEL_QUADS, 8, od="f32", expect=dd.DEDISP_KERNEL_QUADS)


def blocks():
    w = HTRU.scaled(nchans=4100, df=-400.0 / 4100, ndm=40, dm_hi=30.0, nsamps_out=1500, kind="uniform2")
    _run(w, dd.DEDISP_KERNEL_BITSLICE, 2, od="f32", expect=dd.DEDISP_KERNEL_BITSLICE)
    _run(w, dd.DEDISP_KERNEL_PAIRS, 2, od="f32", expect=dd.DEDISP_KERNEL_PAIRS)


def unaligned():
    for off in (1, 3, 8, 15):
        _run(W.CONFIGS["tiny"].scaled(nsamps_out=2001), dd.DEDISP_KERNEL_AUTO, 2, offset=off)
    w8 = W.CONFIGS["wide8"].scaled(nchans=40, ndm=33, dm_hi=STEP8 * 32, nsamps_out=1501)
    _run(w8, dd.DEDISP_KERNEL_BITSLICE, 8, offset=5)


def multi():
    # 10 DM groups x 5 tiles = 50 items on a 16-channel plan: with few CTAs' worth of work per item the
    # persistent CTAs wrap the ring many times (producer/consumer phase parity across work items)
    w = HTRU.scaled(nchans=96, df=-4.0, ndm=300, dm_hi=60.0, nsamps_out=1920 * 4 + 77, kind="uniform2")
    _run(w, dd.DEDISP_KERNEL_BITSLICE, 2, od="f32")
    w = HTRU.scaled(nchans=96, df=-0.4, ndm=300, dm_hi=STEP * 299, nsamps_out=1920 * 4 + 77)
    _run(w, dd.DEDISP_KERNEL_PAIRS, 2, od="u32", expect=dd.DEDISP_KERNEL_PAIRS)


def search():
    from oracle import matched_filter as MF, peak_finding as PF
    x = W.dedispersed_like(41, 5, 20001, npulses=4)
    widths = [1, 2, 4, 8, 16, 32, 64]
    nrows, n = x.shape
    ns = len(widths) * nrows
    s = torch.cuda.current_stream().cuda_stream
    nb, hb, ho = dd.dedisp_matched_filter_hint_blocks(n, widths)
    xd = torch.from_numpy(x.view(np.int32)).cuda()
    z = torch.zeros((len(widths), nrows, n), dtype=torch.float32, device="cuda")
    rms = torch.zeros(ns, dtype=torch.float32, device="cuda")
    hint = torch.zeros((ns, nb), dtype=torch.int32, device="cuda")
    mwb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, len(widths))
    mws = torch.zeros(mwb, dtype=torch.uint8, device="cuda")
    dd.dedisp_matched_filter_rms(xd, dd.DEDISP_OUT_U32, nrows, n, 700, widths, 3072, z, rms, mws, mwb, s,
                                 blockmax_ptr=hint)
    wsb = dd.dedisp_find_events_workspace_bytes(ns, n)
    ws = torch.zeros(wsb, dtype=torch.uint8, device="cuda")
    ev = torch.zeros((1 << 14, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    dd.dedisp_find_events_hinted(z, ns, n, rms, 4.0, hint, hb, ho, ws, wsb, ev, 1 << 14, cnt, s)
    torch.cuda.synchronize()
    zw = MF.matched_filter(x, 700, widths)
    zh = z.cpu().numpy()
    assert np.all(np.abs(zh - zw) <= 2.0 ** -22 * np.abs(zw))
    want = PF.find_events(zh.reshape(ns, n), rms.cpu().numpy(), 4.0)
    got = ev[: int(cnt.item())].cpu().numpy()
    assert len(got) == len(want) and len(want) > 0
    assert np.array_equal(got[:, 1], want["t_start"]) and np.array_equal(got[:, 3], want["t_peak"])


def fault_injection():
    """The checks can fail: with a wrong tag stamped on one ring stage per CTA (dedisp_debug_inject_fault) the
    -DDEDISP_CHECKS build counts stage-tag failures -- and nothing else, the data being right the result still
    equals the oracle.  A product build has no checks compiled in and counts nothing."""
    w = HTRU.scaled(ndm=84, dm_lo=930.0, dm_hi=930.0 + STEP * 83, nsamps_out=4100)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    want = oracle.dedisperse(delay, x, 2, w.nsamps_out)
    counted = []
    for kernel in (dd.DEDISP_KERNEL_PAIRS, dd.DEDISP_KERNEL_BITSLICE):
        p = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
        dd.dedisp_set_dm_list(p, list(w.dms()))
        dd.dedisp_set_kernel(p, kernel)
        dd.dedisp_debug_inject_fault(p, 1)
        out = torch.zeros((w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
        dd.dedisp_execute(p, w.nsamps_out, torch.from_numpy(x).cuda(), 2, out, dd.DEDISP_OUT_U32,
                          torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), want)
        errs = dd.dedisp_debug_check_errors(p)
        if dd.dedisp_debug_checks_compiled():
            assert errs[2] > 0 and errs[0] == errs[2], errs        # CHK_STAGE_TAG only
        else:
            assert errs[0] == 0, errs
        counted.append(errs[2])
        dd.dedisp_destroy(p)
    return f"bit-exact vs oracle; injected wrong stage tags counted by the checks: {counted} (pair rows, planes)"


CASES = {f.__name__: f for f in (tiny_auto, tiny_direct, pairs3, pairs8, quads8, blocks, unaligned, multi, search, fault_injection)}


def main(argv):
    assert torch.cuda.is_available(), "needs a CUDA device (there is no CPU fallback)"
    names = argv or list(CASES)
    for n in names:
        note = CASES[n]()
        print(f"case {n}: ok ({note or 'bit-exact vs oracle, guards intact, 3 scratch poisons, 0 check failures'})",
              flush=True)
    print(f"hazard_cases: {len(names)} cases ok; in-kernel checks compiled: {dd.dedisp_debug_checks_compiled()}; "
          f"launches={dd.dedisp_get_launch_count()}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
