"""Helpers for the -m gpu parity tests: run a workload through the C ABI with torch
owning device memory, and produce the oracle-side inputs."""
import numpy as np
import torch

import oracle
import paper_1112_0065_b200 as dd
import workloads as W


def oracle_inputs(w):
    """(delay, max_delay, packed[nbeams, nchans, stride]) from the ORACLE's delay table."""
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    kw = {}
    if w.kind == "gauss2_pulses":
        p = W.pulse_params(w)
        sweep, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, p.dm)
        kw = dict(pulse_sweep=sweep, pulses=p)
    return delay, md, W.generate_all_beams(w, md, **kw)


def make_plan(nchans, dt, f_top, df, dms, kernel=dd.DEDISP_KERNEL_AUTO):
    p = dd.dedisp_plan_create(nchans, dt, f_top, df)
    dd.dedisp_set_dm_list(p, list(dms))
    dd.dedisp_set_kernel(p, kernel)
    return p


def gpu_dedisperse(plan, packed, nbits, nsamps_out, out_dtype="u32", stream=None):
    """packed: uint8 [nbeams, nchans, stride] (host).  Returns host array [nbeams, ndm, nsamps_out]."""
    nbeams, nchans, stride = packed.shape
    ndm = dd.dedisp_get_ndm(plan)
    assert stride == dd.dedisp_get_in_row_stride_bytes(plan, nsamps_out, nbits)
    x = torch.from_numpy(packed).cuda()
    f32 = out_dtype == "f32"
    out = torch.full((nbeams, ndm, nsamps_out), -7, dtype=torch.float32 if f32 else torch.int32,
                     device="cuda")
    s = stream if stream is not None else torch.cuda.current_stream()
    code = dd.DEDISP_OUT_F32 if f32 else dd.DEDISP_OUT_U32
    if nbeams == 1:
        dd.dedisp_execute(plan, nsamps_out, x, nbits, out, code, s.cuda_stream)
    else:
        dd.dedisp_execute_batch(plan, nbeams, nsamps_out, x, nchans * stride, nbits, out,
                                ndm * nsamps_out * 4, code, s.cuda_stream)
    s.synchronize()
    res = out.cpu().numpy()
    return res if f32 else res.view(np.uint32)
