"""The whole detection chain on the GPU (RFI mitigation, incoherent dedispersion,
baseline removal, matched filtering, peak finding) on a cut-down injected-pulse gulp: a sanity
property of the definitions (SURVEY.md Sec. 8(c) "Injected pulses"), not an oracle parity test --
every stage has its own parity test; here the stages are chained on the device and must find the
pulses that the seeded generator injected along their exact dispersion sweeps."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1112_0065_b200 as dd  # noqa: E402
import workloads as W  # noqa: E402
from gpu_helpers import make_plan, oracle_inputs  # noqa: E402


def test_injected_pulses_are_found_at_their_dm_time_and_width():
    w = W.CONFIGS["htru_long_pulses"].scaled(ndm=300, nsamps_out=65536, npulses=6)
    delay, md, packed = oracle_inputs(w)             # seeded input with 6 dispersed pulses
    pulses = W.pulse_params(w)
    s = torch.cuda.current_stream().cuda_stream
    plan = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = torch.empty((w.ndm, w.nsamps_out), dtype=torch.int32, device="cuda")
    dd.dedisp_execute(plan, w.nsamps_out, torch.from_numpy(packed[0]).cuda(), w.nbits, x, dd.DEDISP_OUT_U32, s)
    dd.dedisp_destroy(plan)
    widths = [1, 2, 4, 8, 16, 32, 64]
    z = torch.empty((len(widths), w.ndm, w.nsamps_out), dtype=torch.float32, device="cuda")
    dd.dedisp_matched_filter(x, dd.DEDISP_OUT_U32, w.ndm, w.nsamps_out, 4000, widths, 3 * w.nchans, z, s)
    ns = len(widths) * w.ndm
    rms = torch.empty(ns, dtype=torch.float32, device="cuda")
    dd.dedisp_series_rms(z, ns, w.nsamps_out, rms, s)
    wsb = dd.dedisp_find_events_workspace_bytes(ns, w.nsamps_out)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    ev = torch.zeros((1 << 20, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    dd.dedisp_find_events(z, ns, w.nsamps_out, rms, 8.0, ws, wsb, ev, 1 << 20, cnt, s)
    torch.cuda.synchronize()
    n = int(cnt.item())
    assert 0 < n < (1 << 20)
    e = ev[:n].cpu().numpy()
    series, t_peak = e[:, 0], e[:, 3]
    snr = e[:, 4].copy().view(np.float32) / rms.cpu().numpy()[series]
    wi, dmi = series // w.ndm, series % w.ndm
    dms = w.dms()
    found = 0
    for p in range(w.npulses):
        d_near = int(np.argmin(np.abs(dms - pulses.dm[p])))
        near = (np.abs(dmi - d_near) <= 2) & (np.abs(t_peak - pulses.t0[p]) <= 2 * int(pulses.width[p]) + 8)
        assert near.any(), f"pulse {p} (DM {pulses.dm[p]:.1f}, t0 {pulses.t0[p]}, width {pulses.width[p]}) not found"
        best = np.argmax(np.where(near, snr, -1))
        # the best-matching boxcar is within a factor 2 of the injected width (or the widest filter)
        wb = widths[wi[best]]
        assert wb >= min(pulses.width[p], 64) / 2 and wb <= 2 * pulses.width[p] + 1, (wb, pulses.width[p])
        found += 1
    # and the strongest event of all belongs to an injected pulse
    top = int(np.argmax(snr))
    assert any(abs(t_peak[top] - pulses.t0[p]) <= 200 for p in range(w.npulses))
    assert found == w.npulses
