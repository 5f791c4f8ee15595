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


def test_all_beam_burst_is_masked_and_vetoed_while_the_dispersed_pulse_survives():
    """RFI mitigation -> dedispersion -> filter + search -> veto, chained on the device:
    four beams see the same undispersed burst (terrestrial interference: every channel at the same time, every
    beam), beam 0 also holds a dispersed pulse.  The coincidence mask of the beams' DM-0 series flags the burst;
    events of beam 0 whose peak sample is flagged are vetoed, the pulse's events are not."""
    import oracle
    nb, t_rfi, t_pulse, dm_pulse = 4, 20000, 40000, 300.0
    w = W.CONFIGS["htru_long_pulses"].scaled(ndm=128, dm_hi=400.0, nsamps_out=65536, nbeams=nb)
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    sweep, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, [0.0, dm_pulse])
    beams = []
    for b in range(nb):
        npl = 2 if b == 0 else 1
        p = W.Pulses(dm=np.array([0.0, dm_pulse][:npl]), width=np.array([4, 8][:npl]), t0=np.array([t_rfi, t_pulse][:npl]))
        beams.append(W.generate(w.scaled(npulses=npl), md, beam=b, pulse_sweep=sweep[:, :npl], pulses=p))
    packed = np.stack(beams)
    s = torch.cuda.current_stream().cuda_stream
    plan = make_plan(w.nchans, w.dt, w.f_top, w.df, w.dms())
    n, ndm = w.nsamps_out, w.ndm
    out = torch.empty((nb, ndm, n), dtype=torch.int32, device="cuda")
    dd.dedisp_execute_batch(plan, nb, n, torch.from_numpy(packed).cuda(), packed[0].size, w.nbits, out, ndm * n * 4,
                            dd.DEDISP_OUT_U32, s)
    dd.dedisp_destroy(plan)
    # stage 1: the DM-0 series of every beam against 3 sigma in >= 4 beams
    dm0 = out[:, 0, :].float()
    mean, sigma = dm0.mean(dim=1, keepdim=True).contiguous(), dm0.std(dim=1, keepdim=True).contiguous()
    mask = torch.zeros((1, n), dtype=torch.uint8, device="cuda")
    dd.dedisp_rfi_mask(out, dd.DEDISP_OUT_U32, nb, 1, n, ndm * n * 4, mean, sigma, 3.0, 4, mask, s)
    # stages 3-5 on beam 0: filter + sigma-cut + grouping without materialising z
    widths, nsigma, cap, max_blocks = [1, 2, 4, 8, 16], 8.0, 1 << 18, 1 << 12
    wsb = dd.dedisp_search_events_workspace_bytes(ndm, n, widths, max_blocks)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    rms = torch.empty(len(widths) * ndm, dtype=torch.float32, device="cuda")
    ev = torch.zeros((cap, 5), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    kept = torch.zeros(1, dtype=torch.int64, device="cuda")
    dd.dedisp_search_events(out[0], dd.DEDISP_OUT_U32, ndm, n, 4000, widths, 3 * w.nchans, nsigma, rms, max_blocks, ws,
                            wsb, ev, cap, cnt, s)
    dd.dedisp_veto_events(ev, cnt, cap, mask, n, kept, s)
    torch.cuda.synchronize()
    m = mask.cpu().numpy()[0]
    assert m[t_rfi:t_rfi + 4].all() and m.sum() < 64 and not m[t_pulse - 200:t_pulse + 200].any()
    total, blocks = int(cnt[0].item()), int(cnt[1].item())
    assert 0 < total < cap and blocks <= max_blocks
    e = ev[:total].cpu().numpy()
    vetoed = e[:, 0] < 0
    series = np.where(vetoed, -1 - e[:, 0], e[:, 0])
    dmi, t_peak = series % ndm, e[:, 3]
    assert int(kept.item()) == int((~vetoed).sum()) and vetoed.any() and (~vetoed).any()
    # every event of the DM-0 trial that peaks inside the burst is vetoed ...
    in_burst = (dmi == 0) & (t_peak >= t_rfi) & (t_peak < t_rfi + 4)
    assert in_burst.any() and vetoed[in_burst].all()
    # ... and the dispersed pulse is still there, at its DM and time
    d_near = int(np.argmin(np.abs(w.dms() - dm_pulse)))
    pulse = (np.abs(dmi - d_near) <= 2) & (np.abs(t_peak - t_pulse) <= 24)
    assert pulse.any() and not vetoed[pulse].any()
