#!/usr/bin/env python
"""bench.py -- DM-trial-samples/s of direct incoherent dedispersion on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config htru_gulp] [--impl ours|reference]

One "step" = one pass of the whole hot path (delay table already built in
set_dm_list; unpack/bit-plane pre-pass + gather-sum + output write) over one
synthetic HTRU-shaped gulp already resident in HBM.  Prints ONE JSON line.
N > 1 (torchrun): every rank dedisperses its own independently seeded beam
(replicas, no data-path collective) -- "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))
from paper_1112_0065_b200 import replicas  # noqa: E402
import workloads as W  # noqa: E402

SM_COUNT_NOMINAL = 148
ADDS_PER_CLK_PER_SM = 128          # FP32/INT32 lane-adds per clock per SM
PAPER_CONTEXT = [
    "paper context (PAPER.md:22): whole CPU pipeline > 30 min per 10-min observation (unnamed CPU cluster)",
    "paper context (PAPER.md:48): dedispersion ~20 min (unnamed CPU) -> 2.5 min (unnamed 2011 CUDA GPU) "
    "per 10-min observation = 7.5e7 DM-trial-samples/s, RTF 4.0",
]


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    return json.loads(p.read_text()) if p.exists() else {}


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [s.strip() for s in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # samples under load = upper half (idle samples before/after the kernels drag the median)
        hi = sorted(sm)[len(sm) // 2:]
        return {"sm_mhz": statistics.median(hi), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def dist_setup(ngpus: int):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        torch.cuda.set_device(0)
    return rank, world, local


def cpu_model() -> str:
    try:
        for line in Path("/proc/cpuinfo").read_text().splitlines():
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(w: W.Workload, tscrunch: int = 1) -> dict:
    """The oracle as it stands, on this box's host cores, on a bounded sample of the workload: all cores and one
    thread, best of 3 each (SURVEY.md Sec. 8(d) "CPU baseline timed beside it")."""
    import oracle
    delay, md = oracle.delay_table(w.nchans, tscrunch * w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w.scaled(nbeams=1), tscrunch * (w.nsamps_out + md) - w.nsamps_out)
    stride = max(1, (w.ndm * w.nsamps_out) // (1200 * 65536))   # ~ one HTRU gulp of work for all cores

    def run(sub, nthreads):
        best, used = None, 0
        for _ in range(3):
            t0 = time.perf_counter()
            if tscrunch > 1:
                from oracle import tscrunch as TS
                _, used = TS.dedisperse_tscrunch_bytes(sub, x, w.nbits, tscrunch, w.nsamps_out, return_threads=True)
            else:
                _, used = oracle.dedisperse(sub, x, w.nbits, w.nsamps_out, nthreads=nthreads, return_threads=True)
            dt = time.perf_counter() - t0
            best = dt if best is None or dt < best else best
        return best, used

    sub = np.ascontiguousarray(delay[:, ::stride])
    dt_all, used = run(sub, os.cpu_count() or 1)
    units = sub.shape[1] * w.nsamps_out
    res = {"value": units / dt_all, "unit": "DM-trial-samples/s", "cores": used, "kind": "oracle",
           "cpu_model": cpu_model(), "nproc": os.cpu_count(), "best_of": 3, "seconds": dt_all,
           "sample": f"{sub.shape[1]} of {w.ndm} DM trials (every {stride}th) x {w.nsamps_out} samples "
                     f"x {w.nchans} channels of {w.name}, best of 3 passes, {dt_all:.2f} s",
           "rtf": (w.nsamps_out * w.dt) / (dt_all * w.ndm / sub.shape[1])}
    if tscrunch == 1:
        sub1 = np.ascontiguousarray(delay[:, ::stride * 8])      # one thread: an eighth of that
        dt_1, used1 = run(sub1, 1)
        res["one_thread"] = {"value": sub1.shape[1] * w.nsamps_out / dt_1, "unit": "DM-trial-samples/s", "cores": used1,
                             "seconds": dt_1, "sample": f"{sub1.shape[1]} of {w.ndm} DM trials (every {stride * 8}th), "
                                                        f"best of 3 passes, {dt_1:.2f} s"}
    return res


def ncu_traffic(config: str, kernel: str | None = None):
    """(DRAM bytes per launch of the dominant kernel, source file, commit of the capture) from the committed ncu
    captures (profiles/traffic.csv: config,bytes_per_launch,source,commit[,kernel]), or (None, None, None).  A row that
    names a kernel only serves a run of that kernel (--kernel can force another one than the capture saw)."""
    p = ROOT / "profiles" / "traffic.csv"
    if not p.exists():
        return None, None, None
    for line in p.read_text().splitlines():
        f = [v.strip() for v in line.split(",")]
        if len(f) >= 2 and f[0] == config:
            if kernel is not None and len(f) > 4 and f[4] and f[4] != kernel:
                continue
            try:
                return float(f[1]), (f[2] if len(f) > 2 else None), (f[3] if len(f) > 3 else None)
            except ValueError:
                return None, None, None
    return None, None, None


def ncu_traffic_bytes(config: str):
    return ncu_traffic(config)[0]


KERNEL_NAMES = {1: "direct_kernel", 2: "bitslice_dedisperse", 3: "bitslice_dedisperse on pair rows",
                4: "bitslice_dedisperse on quad rows"}
# ALU-pipe (LOP3 / SHF / LEA: 64 lanes per clock and SM) instructions per addition of the dominant kernel's hot loop,
# counted on the SASS / the ncu source page: (kernel, nbits) -> (lane-instructions per add, where it was counted)
ALU_PIPE_INSTR_PER_ADD = {
    (3, 2): (626.0 / 4096.0, "profiles/r2_sass_cfg3p.txt: 626 ALU-pipe of 918 instructions per 4096 adds"),
    (3, 8): (0.455, "profiles/r2_wide8.md: ncu source page, LOP3 + SHF share of 23.97 G instructions"),
    (4, 8): (531.0 / 2048.0, "profiles/r2_sass_cfg10q.txt: 531 ALU-pipe of 774 instructions per 2048 adds"),
}
ALU_PIPE_LANES_PER_CLK_PER_SM = 64


def measure_dedisperse(torch, dd, w, k, kernel, steps, warmup, rank, world, dev, stream, flush, e2e_steps):
    """W warm-ups + K timed steps of the hot path on workload w (inputs resident in HBM), CUDA events on the launching
    stream, L2 flushed between iterations; optionally the end-to-end leg through dedisp_execute_host.  Returns the raw
    measurements; nothing here is specific to the headline config."""
    plan = dd.dedisp_plan_create(w.nchans, k * w.dt, w.f_top, w.df)
    t0 = time.perf_counter()
    dd.dedisp_set_dm_list(plan, list(w.dms()))
    set_dm_ms = (time.perf_counter() - t0) * 1e3
    dd.dedisp_set_kernel(plan, {"auto": dd.DEDISP_KERNEL_AUTO, "bitslice": dd.DEDISP_KERNEL_BITSLICE,
                                "pairs": dd.DEDISP_KERNEL_PAIRS, "quads": dd.DEDISP_KERNEL_QUADS}[kernel])
    md = dd.dedisp_get_max_delay(plan)
    kw = {}
    if w.kind == "gauss2_pulses":   # pulse sweeps from the product's own delay builder
        pp = W.pulse_params(w)
        p2 = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
        dd.dedisp_set_dm_list(p2, list(pp.dm))
        kw = dict(pulse_sweep=dd.dedisp_get_delay_table(p2), pulses=pp)
        dd.dedisp_destroy(p2)
    # each rank gets its own seeded beam(s): beam index offset by rank
    beams = [W.generate(w, k * (w.nsamps_out + md) - w.nsamps_out, beam=b, **kw)
             for b in replicas.beam_indices(rank, w.nbeams)]
    host_in = torch.from_numpy(np.stack(beams)).pin_memory()
    nb, nch, stride = host_in.shape
    assert stride == dd.dedisp_get_in_row_stride_bytes_tscrunch(plan, k, w.nsamps_out, w.nbits)
    x = host_in.to(dev)
    f32 = w.out_dtype == "f32"
    code = dd.DEDISP_OUT_F32 if f32 else dd.DEDISP_OUT_U32
    out = torch.empty((nb, w.ndm, w.nsamps_out), dtype=torch.float32 if f32 else torch.int32, device=dev)
    in_bs, out_bs = nch * stride, w.ndm * w.nsamps_out * 4
    if k == 1:
        dd.dedisp_reserve(plan, nb, w.nsamps_out, w.nbits)     # the timed steps never allocate

    def step():
        dd.dedisp_execute_tscrunch(plan, k, nb, w.nsamps_out, x, in_bs, w.nbits, out, out_bs, code,
                                   stream.cuda_stream)

    dd.dedisp_set_timing(plan, True)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    time.sleep(0.15)
    launches0 = dd.dedisp_get_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    main_ms, pre_ms = [], []
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()                 # L2 flush between timed iterations (outside the events)
        a.record(stream)
        step()
        b.record(stream)
        pm, mm = dd.dedisp_get_last_kernel_ms(plan)   # waits for this step's kernels
        pre_ms.append(pm)
        main_ms.append(mm)
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    launches = dd.dedisp_get_launch_count() - launches0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    if world > 1:
        dist.barrier()
    m = {"plan_md": md, "set_dm_ms": set_dm_ms, "step_ms": step_ms, "main_ms": main_ms, "pre_ms": pre_ms,
         "launches": launches, "clocks": clocks, "wall": wall, "nb": nb, "in_bytes": nb * in_bs, "out_bytes": nb * out_bs,
         "kernel_used": dd.dedisp_get_last_kernel(plan), "e2e_s": None, "same": None, "e2e_steps": e2e_steps}
    if e2e_steps > 0:
        # ---- end to end through the public host-buffer call (H2D + kernels + D2H inside the timing)
        host_out = torch.empty((nb, w.ndm, w.nsamps_out), dtype=out.dtype).pin_memory()
        dd.dedisp_set_timing(plan, False)

        def host_step():
            if k == 1:
                return dd.dedisp_execute_host(plan, nb, w.nsamps_out, host_in, w.nbits, host_out, code)
            x.copy_(host_in, non_blocking=True)
            step()
            host_out.copy_(out, non_blocking=True)
            stream.synchronize()

        host_step()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            host_step()
        m["e2e_s"] = (time.perf_counter() - t0) / e2e_steps
        m["same"] = bool(torch.equal(host_out.to(dev), out))
        m["kernel_used"] = dd.dedisp_get_last_kernel(plan)
        del host_out
    dd.dedisp_destroy(plan)
    del x, out, host_in
    torch.cuda.empty_cache()
    return m


def instr_bound(w, m, achieved_adds_per_s, props, sm_max_mhz):
    """Fraction of the 64-lane ALU pipe the dominant kernel's hot loop keeps busy, from its counted ALU-pipe
    instructions per addition (None where no count is committed)."""
    ent = ALU_PIPE_INSTR_PER_ADD.get((m["kernel_used"], w.nbits))
    if ent is None:
        return None
    per_add, src = ent
    pipe_peak = props.multi_processor_count * ALU_PIPE_LANES_PER_CLK_PER_SM * sm_max_mhz * 1e6
    return {"bound": "alu_pipe", "alu_pipe_instr_per_add": per_add, "achieved": per_add * achieved_adds_per_s / 1e12,
            "peak": pipe_peak / 1e12, "unit": "T lane-instr/s", "frac": per_add * achieved_adds_per_s / pipe_peak,
            "source": src}


def roofline_of(w, k, m, ms_per_step, props, peaks, config_name):
    """north_star's roofline: the slower of nchans*ndm*nsamps adds at the ALU peak and the compulsory bytes at the HBM
    bandwidth; `achieved` = adds / the dominant kernel's mean launch time (CUDA events inside the library, live)."""
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak = props.multi_processor_count * ADDS_PER_CLK_PER_SM * sm_max_mhz * 1e6   # adds/s
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0)) * 1e9
    adds = w.adds() * k          # every fine sample is added once
    t_alu, t_hbm = adds / alu_peak, (m["in_bytes"] + m["out_bytes"]) / hbm_peak
    mm = statistics.mean(m["main_ms"]) * 1e-3
    achieved = adds / mm
    traffic, tsrc, tcommit = ncu_traffic(config_name, KERNEL_NAMES.get(m["kernel_used"], "direct_kernel"))
    return {"bound": "alu", "achieved": achieved / 1e12, "peak": alu_peak / 1e12, "unit": "Tadd/s",
            "frac": achieved / alu_peak, "traffic": traffic, "traffic_source": tsrc, "traffic_capture_commit": tcommit,
            "kernel": KERNEL_NAMES.get(m["kernel_used"], "direct_kernel"),
            "kernel_ms": mm * 1e3, "prepass_ms": statistics.mean(m["pre_ms"]),
            "kernel_share_of_step": mm * 1e3 / ms_per_step,
            "peak_source": f"{props.multi_processor_count} SMs x {ADDS_PER_CLK_PER_SM} adds/clk x "
                           f"{sm_max_mhz:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz); see DESIGN.md",
            "algorithmic_bytes": m["in_bytes"] + m["out_bytes"],
            "hbm_frac": ((m["in_bytes"] + m["out_bytes"]) / mm) / hbm_peak,
            "step_roofline_frac": max(t_alu, t_hbm) / (ms_per_step * 1e-3),
            "frac_note": "north_star's fraction counts one add per lane-op; a bit-sliced LOP3 pair adds 32 samples and "
                         "pair rows share two-channel sums, so it can exceed 1 -- instr_bound is the physical limiter",
            "instr_bound": instr_bound(w, m, achieved, props, sm_max_mhz) if k == 1 else None}


def run_ours(args) -> None:
    import torch
    import paper_1112_0065_b200 as dd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    rank, world, local = dist_setup(args.gpus)
    w = W.CONFIGS[args.config]
    dev = torch.device("cuda", torch.cuda.current_device())
    props = torch.cuda.get_device_properties(dev)
    stream = torch.cuda.current_stream()
    peaks = measured_peaks()

    k = args.tscrunch   # row f4: blocks of k samples summed, trials dedispersed on the grid k*dt (reading R38)
    if k > 1 and w.kind == "gauss2_pulses":
        raise SystemExit("bench.py: --tscrunch is benched on the noise-only configs")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    m = measure_dedisperse(torch, dd, w, k, args.kernel, args.steps, args.warmup, rank, world, dev, stream, flush,
                           e2e_steps=max(2, min(args.steps, 5)))
    total_ms = replicas.max_over_ranks(sum(m["step_ms"]), dev)
    ms_per_step = total_ms / args.steps
    value = replicas.job_throughput(w.dm_trial_samples(), world, ms_per_step * 1e-3)
    e2e_s = replicas.max_over_ranks(m["e2e_s"], dev)
    e2e_value = replicas.job_throughput(w.dm_trial_samples(), world, e2e_s)

    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()
        return
    roofline = roofline_of(w, k, m, ms_per_step, props, peaks, args.config)
    try:
        import bench_probe
        bench_probe.build()
        probe = {n: bench_probe.probe_alu_rate(i) / 1e12 for i, n in enumerate(bench_probe.NAMES)}
    except Exception as e:  # noqa: BLE001
        probe = {"error": str(e)}

    # ---- the other BASELINE.json configs, timed the same way in the same run (N = 1, default config only)
    per_config = None
    if world == 1 and args.per_config and k == 1 and args.kernel == "auto" and args.config == "htru_gulp":
        per_config = {}
        for name in W.CONFIG_ORDER:
            wc = W.CONFIGS[name]
            if name == args.config:
                mc, ms_c, rc, nsteps = m, ms_per_step, roofline, args.steps
            else:
                nsteps = max(5, min(args.steps, 10))
                log(f"per_config: {name} ...")
                mc = measure_dedisperse(torch, dd, wc, 1, "auto", nsteps, max(3, args.warmup), 0, 1, dev, stream, flush,
                                        e2e_steps=0)
                ms_c = statistics.mean(mc["step_ms"])
                rc = roofline_of(wc, 1, mc, ms_c, props, peaks, name)
            per_config[name] = {
                "ms_per_step": ms_c, "kernel_ms": rc["kernel_ms"], "prepass_ms": rc["prepass_ms"],
                "value": wc.dm_trial_samples() / (ms_c * 1e-3), "unit": "DM-trial-samples/s",
                "real_time_factor": wc.obs_seconds() / (ms_c * 1e-3), "kernel": rc["kernel"],
                "roofline": {"bound": "alu", "frac": rc["frac"], "achieved": rc["achieved"], "peak": rc["peak"],
                             "unit": "Tadd/s", "traffic": rc["traffic"], "traffic_source": rc["traffic_source"]},
                "step_roofline_frac": rc["step_roofline_frac"], "steps": nsteps, "warmup": max(3, args.warmup),
                "dtype": wc.out_dtype, "gpu_launches": mc["launches"], "clocks": mc["clocks"],
                "step_ms_min_med_max": [min(mc["step_ms"]), statistics.median(mc["step_ms"]), max(mc["step_ms"])],
                "config": {"workload": name, "nchans": wc.nchans, "ndm": wc.ndm, "nsamps_out": wc.nsamps_out,
                           "nbits": wc.nbits, "nbeams": wc.nbeams, "out_dtype": wc.out_dtype, "max_delay": mc["plan_md"]},
                "note": "3 work items: launch-latency sized, roofline fraction meaningless" if name == "tiny" else None}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(w, tscrunch=k)
    for line in PAPER_CONTEXT:
        log(line)
    res = {
        "metric": "DM-trial samples/sec", "value": value, "unit": "DM-trial-samples/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": w.out_dtype,
        "data": "synthetic",
        "config": {"workload": w.name, "nchans": w.nchans, "ndm": w.ndm, "nsamps_out": w.nsamps_out,
                   "nbits": w.nbits, "tscrunch": k, "nbeams_per_gpu": w.nbeams, "out_dtype": w.out_dtype,
                   "max_delay": m["plan_md"], "l2": "256 MiB flush buffer zeroed between timed iterations",
                   "parallelism": f"replicas x{world} (one seeded beam set per GPU, no collective)"},
        "real_time_factor": k * w.obs_seconds() / (ms_per_step * 1e-3),
        "roofline": roofline, "cpu_baseline": cpu,
        "e2e": {"value": e2e_value, "unit": "DM-trial-samples/s", "h2d_bytes_per_step": m["in_bytes"],
                "d2h_bytes_per_step": m["out_bytes"], "steps": m["e2e_steps"], "matches_device_run": m["same"]},
        "gpu_launches": m["launches"], "clocks": m["clocks"], "alu_probe_Tlaneops": probe,
        "set_dm_list_ms": m["set_dm_ms"], "wall_s_timed_region": m["wall"],
        "step_ms_min_med_max": [min(m["step_ms"]), statistics.median(m["step_ms"]), max(m["step_ms"])],
        "per_config": per_config,
        "paper_context": {"gpu_2011_dm_trial_samples_per_s": 7.5e7, "cpu_dm_trial_samples_per_s": 9.4e6,
                          "source": "PAPER.md:48, unnamed hardware; context, not target"},
    }
    print(json.dumps(res), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def run_matched_filter(args) -> None:
    """--op matched_filter: row f1 on the dedispersed output of --config,
    one GPU.  A step = one dedisp_matched_filter call over all DM trials (x resident in HBM);
    HBM-bound: algorithmic bytes = x read once + nwidths float32 series written."""
    import torch
    import paper_1112_0065_b200 as dd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(0)
    w = W.CONFIGS[args.config].scaled(nbeams=1)
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream()
    plan = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    dd.dedisp_set_dm_list(plan, list(w.dms()))
    md = dd.dedisp_get_max_delay(plan)
    host_in = torch.from_numpy(W.generate(w, md)).pin_memory()
    x = torch.empty((w.ndm, w.nsamps_out), dtype=torch.int32, device=dev)
    dd.dedisp_execute(plan, w.nsamps_out, host_in.to(dev), w.nbits, x, dd.DEDISP_OUT_U32, stream.cuda_stream)
    dd.dedisp_destroy(plan)
    widths = [1, 2, 4, 8, 16, 32, 64]
    radius = min(int(round(1.0 / w.dt)), (w.nsamps_out - 1) // 2)   # 2 s window (R21)
    x_max = w.nchans * ((1 << w.nbits) - 1)
    z = None if (args.op == "search" and args.search_mode == "fused") else \
        torch.empty((len(widths), w.ndm, w.nsamps_out), dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        dd.dedisp_matched_filter(x, dd.DEDISP_OUT_U32, w.ndm, w.nsamps_out, radius, widths, x_max, z,
                                 stream.cuda_stream)

    if args.op == "find_events":
        return _bench_find_events(args, dd, torch, w, widths, z, step, flush, stream)
    if args.op == "search":
        return _bench_search(args, dd, torch, w, widths, radius, x_max, x, z, flush, stream)
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.15)
    launches0 = dd.dedisp_get_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    launches = dd.dedisp_get_launch_count() - launches0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    ms = statistics.mean(step_ms)
    units = w.ndm * w.nsamps_out * len(widths)
    # end to end: host x -> device, filter, z -> host
    hx = x.cpu().pin_memory()
    hz = torch.empty(z.shape, dtype=torch.float32).pin_memory()
    e2e_steps = 2
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        x.copy_(hx, non_blocking=True)
        step()
        hz.copy_(z, non_blocking=True)
        torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    alg_bytes = x.numel() * 4 + z.numel() * 4
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import matched_filter as MF
        rows = x[:: max(1, w.ndm // 48)].cpu().numpy().view(np.uint32)
        t0 = time.perf_counter()
        MF.matched_filter(rows, radius, widths)
        dt = time.perf_counter() - t0
        cpu = {"value": rows.size * len(widths) / dt, "unit": "filtered samples/s", "cores": 1, "kind": "oracle",
               "sample": f"{rows.shape[0]} of {w.ndm} rows x {w.nsamps_out} samples x {len(widths)} widths, {dt:.2f} s"}
    res = {"metric": "matched-filter output samples/sec", "value": units / (ms * 1e-3), "unit": "filtered samples/s",
           "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32/int64 -> f32",
           "data": "synthetic",
           "config": {"workload": f"matched_filter on dedispersed {w.name}", "nrows": w.ndm,
                      "nsamps": w.nsamps_out, "radius": radius, "widths": widths, "x_max": x_max,
                      "l2": "256 MiB flush buffer zeroed between timed iterations"},
           "roofline": {"bound": "hbm", "achieved": alg_bytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": alg_bytes / (ms * 1e-3) / 1e9 / hbm_peak,
                        "traffic": ncu_traffic_bytes("matched_filter_" + w.name),
                        "kernel": "matched_filter_kernel", "kernel_ms": ms,
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s"},
           "cpu_baseline": cpu,
           "e2e": {"value": units / e2e_s, "unit": "filtered samples/s", "h2d_bytes_per_step": x.numel() * 4,
                   "d2h_bytes_per_step": z.numel() * 4, "steps": e2e_steps},
           "gpu_launches": launches, "clocks": clocks,
           "step_ms_min_med_max": [min(step_ms), statistics.median(step_ms), max(step_ms)]}
    print(json.dumps(res), flush=True)


def _bench_find_events(args, dd, torch, w, widths, z, make_z, flush, stream) -> None:
    """--op find_events: row f2 on the matched-filter output of --config.  A step =
    dedisp_series_rms (the sigma estimate) + dedisp_find_events at 6 sigma over all
    nwidths*ndm filtered series; HBM-bound: z is read twice (once per call), the bit mask
    (1/32 of z) is written and read once."""
    make_z()
    dev = z.device
    ns, n = z.shape[0] * z.shape[1], z.shape[2]
    nsigma, cap = 6.0, 1 << 20
    wsb = dd.dedisp_find_events_workspace_bytes(ns, n)
    ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
    rms = torch.empty(ns, dtype=torch.float32, device=dev)
    ev = torch.empty((cap, 5), dtype=torch.int32, device=dev)
    cnt = torch.zeros(1, dtype=torch.int64, device=dev)

    def step():
        dd.dedisp_series_rms(z, ns, n, rms, stream.cuda_stream)
        dd.dedisp_find_events(z, ns, n, rms, nsigma, ws, wsb, ev, cap, cnt, stream.cuda_stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.15)
    launches0 = dd.dedisp_get_launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(args.steps)]
    for a, b in evs:
        flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    launches = dd.dedisp_get_launch_count() - launches0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    ms = statistics.mean(step_ms)
    found = int(cnt.item())
    # end to end: z from pinned host memory, events + count back to the host
    hz = z.cpu().pin_memory()
    hev = torch.empty((cap, 5), dtype=torch.int32).pin_memory()
    t0 = time.perf_counter()
    z.copy_(hz, non_blocking=True)
    step()
    k = min(int(cnt.item()), cap)
    hev[:k].copy_(ev[:k], non_blocking=True)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    alg_bytes = 2 * z.numel() * 4 + 2 * (z.numel() // 8)
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import peak_finding as PF
        rows = z.reshape(ns, n)[:: max(1, ns // 48)].cpu().numpy()
        t0 = time.perf_counter()
        PF.find_events(rows, PF.series_rms(rows).astype(np.float32), nsigma)
        dt = time.perf_counter() - t0
        cpu = {"value": rows.size / dt, "unit": "searched samples/s", "cores": 1, "kind": "oracle",
               "sample": f"{rows.shape[0]} of {ns} series x {n} samples (rms + find_events), {dt:.2f} s"}
    res = {"metric": "peak-finding input samples/sec", "value": ns * n / (ms * 1e-3), "unit": "searched samples/s",
           "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32 compare / f64 sum",
           "data": "synthetic",
           "config": {"workload": f"series_rms + find_events on matched-filtered {w.name}", "nseries": ns,
                      "nsamps": n, "nsigma": nsigma, "events_found": found, "widths": widths,
                      "l2": "256 MiB flush buffer zeroed between timed iterations"},
           "roofline": {"bound": "hbm", "achieved": alg_bytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": alg_bytes / (ms * 1e-3) / 1e9 / hbm_peak,
                        "traffic": ncu_traffic_bytes("find_events_" + w.name),
                        "kernel": "series_rms_kernel + sigma_cut_kernel (+ 3 small kernels)", "kernel_ms": ms,
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s"},
           "cpu_baseline": cpu,
           "e2e": {"value": ns * n / e2e_s, "unit": "searched samples/s", "h2d_bytes_per_step": z.numel() * 4,
                   "d2h_bytes_per_step": k * 20 + 8, "steps": 1},
           "gpu_launches": launches, "clocks": clocks,
           "step_ms_min_med_max": [min(step_ms), statistics.median(step_ms), max(step_ms)]}
    print(json.dumps(res), flush=True)


def _bench_search(args, dd, torch, w, widths, radius, x_max, x, z, flush, stream) -> None:
    """--op search: rows f1 + f2 chained on the dedispersed output of --config, one call:
    dedisp_search_events (RMS + block maxima of z in one pass over x without writing z, the blocks above the threshold
    re-computed into a compact z, sigma-cut + grouping on that) at 6 sigma.  Algorithmic bytes: x read once.
    --search-mode dense times the round-1 chain instead (dedisp_matched_filter_rms writing all of z +
    dedisp_find_events_hinted).  The end-to-end leg starts from the PACKED filterbank in pinned host memory:
    H2D (22 MB) -> dedisp_execute -> dedisp_search_events -> event list D2H."""
    dev = x.device
    nw, nrows, n = len(widths), x.shape[0], x.shape[1]
    ns = nw * nrows
    nsigma, cap = 6.0, 1 << 20
    dense = args.search_mode == "dense"
    rms = torch.empty(ns, dtype=torch.float32, device=dev)
    ev = torch.empty((cap, 5), dtype=torch.int32, device=dev)
    cnt = torch.zeros(2, dtype=torch.int64, device=dev)
    if dense:
        wsb = dd.dedisp_find_events_workspace_bytes(ns, n)
        ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        mwb = dd.dedisp_matched_filter_rms_workspace_bytes(nrows, n, nw)
        mws = torch.empty(mwb, dtype=torch.uint8, device=dev)
        nblk, hblock, hoff = dd.dedisp_matched_filter_hint_blocks(n, widths)
        hint = torch.empty((ns, nblk), dtype=torch.int32, device=dev)

        def step():
            dd.dedisp_matched_filter_rms(x, dd.DEDISP_OUT_U32, nrows, n, radius, widths, x_max, z, rms, mws, mwb,
                                         stream.cuda_stream, blockmax_ptr=hint)
            dd.dedisp_find_events_hinted(z, ns, n, rms, nsigma, hint, hblock, hoff, ws, wsb, ev, cap, cnt,
                                         stream.cuda_stream)
        alg_bytes = x.numel() * 4 + z.numel() * 4 + 2 * (z.numel() // 8)
        what, kern = "matched_filter_rms + find_events_hinted (dense z)", "matched_filter_kernel + sigma_cut_kernel (+ 4 small kernels)"
    else:
        max_blocks = 1 << 14      # 128 MiB of compact z: 6 sigma on noise flags a few dozen blocks
        wsb = dd.dedisp_search_events_workspace_bytes(nrows, n, widths, max_blocks)
        ws = torch.empty(wsb, dtype=torch.uint8, device=dev)

        def step():
            dd.dedisp_search_events(x, dd.DEDISP_OUT_U32, nrows, n, radius, widths, x_max, nsigma, rms, max_blocks,
                                    ws, wsb, ev, cap, cnt, stream.cuda_stream)
        alg_bytes = x.numel() * 4
        what, kern = "search_events (no z written)", "matched_filter_kernel<RMS, no z> (+ sparse re-computation, 6 small kernels)"

    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.15)
    launches0 = dd.dedisp_get_launch_count()
    step_ms = _time_steps(torch, step, flush, stream, args.warmup, args.steps)
    launches = (dd.dedisp_get_launch_count() - launches0) * args.steps // (args.steps + args.warmup)
    clocks = sampler.stop()
    ms = statistics.mean(step_ms)
    found, flagged = int(cnt[0].item()), int(cnt[1].item())
    # end to end from the packed filterbank in pinned host memory to the event list in host memory
    plan = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
    dd.dedisp_set_dm_list(plan, list(w.dms()))
    md = dd.dedisp_get_max_delay(plan)
    host_in = torch.from_numpy(W.generate(w, md)).pin_memory()
    xin = torch.empty_like(host_in, device=dev)
    hev = torch.empty((cap, 5), dtype=torch.int32).pin_memory()
    hcnt = torch.zeros(2, dtype=torch.int64).pin_memory()
    dd.dedisp_reserve(plan, 1, n, w.nbits)

    def e2e():
        xin.copy_(host_in, non_blocking=True)
        dd.dedisp_execute(plan, n, xin, w.nbits, x, dd.DEDISP_OUT_U32, stream.cuda_stream)
        step()
        hcnt.copy_(cnt, non_blocking=True)
        stream.synchronize()
        k = min(int(hcnt[0].item()), cap)
        hev[:k].copy_(ev[:k], non_blocking=True)
        stream.synchronize()
        return k

    e2e()
    e2e_steps = 3
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        k = e2e()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    dd.dedisp_destroy(plan)
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import matched_filter as MF, peak_finding as PF
        rows = x[:: max(1, nrows // 24)].cpu().numpy().view(np.uint32)
        t0 = time.perf_counter()
        zz = MF.matched_filter(rows, radius, widths).astype(np.float32).reshape(-1, n)
        PF.find_events(zz, PF.series_rms(zz).astype(np.float32), nsigma)
        dt = time.perf_counter() - t0
        cpu = {"value": zz.size / dt, "unit": "searched samples/s", "cores": 1, "kind": "oracle",
               "sample": f"{rows.shape[0]} of {nrows} rows x {n} samples x {nw} widths "
                         f"(matched filter + rms + find_events), {dt:.2f} s"}
    traffic, tsrc, tcommit = ncu_traffic(("search_dense_" if dense else "search_") + w.name)
    res = {"metric": "filtered and searched samples/sec", "value": ns * n / (ms * 1e-3), "unit": "searched samples/s",
           "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "exact int -> f32",
           "data": "synthetic",
           "config": {"workload": f"{what} on dedispersed {w.name}", "nrows": nrows,
                      "nsamps": n, "widths": widths, "radius": radius, "nsigma": nsigma, "events_found": found,
                      "blocks_recomputed": flagged, "l2": "256 MiB flush buffer zeroed between timed iterations"},
           "roofline": {"bound": "hbm", "achieved": alg_bytes / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": alg_bytes / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": traffic, "traffic_source": tsrc,
                        "traffic_capture_commit": tcommit, "algorithmic_bytes": alg_bytes,
                        "kernel": kern, "kernel_ms": ms,
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s"},
           "cpu_baseline": cpu,
           "e2e": {"value": ns * n / e2e_s, "unit": "searched samples/s", "h2d_bytes_per_step": host_in.numel(),
                   "d2h_bytes_per_step": k * 20 + 16, "steps": e2e_steps, "ms_per_step": e2e_s * 1e3,
                   "path": "packed host input -> H2D -> dedisp_execute -> search -> event list D2H"},
           "gpu_launches": launches, "clocks": clocks,
           "step_ms_min_med_max": [min(step_ms), statistics.median(step_ms), max(step_ms)]}
    print(json.dumps(res), flush=True)


def _time_steps(torch, step, flush, stream, warmup, steps):
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in ev]


def run_small_op(args) -> None:
    """--op rfi_mask: row f3 on 13 beams x 2^24 float32 samples (the multibeam
    zero-DM series of ~18 min at 64 us), 3 sigma in >= 4 beams.
    --op transpose: row f4 (telescope-order stream -> channel-major rows) on the packed input of
    --config.  Both HBM-bound single kernels; a step = one call, inputs resident in HBM."""
    import torch
    import paper_1112_0065_b200 as dd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    cpu = None
    if args.op == "rfi_mask":
        nb, n = 13, 1 << 24
        hx = torch.randn((nb, 1, n), generator=torch.Generator().manual_seed(1301)).pin_memory()
        x = hx.to(dev)
        mean, sigma = torch.zeros((nb, 1), device=dev), torch.ones((nb, 1), device=dev)
        m = torch.empty((1, n), dtype=torch.uint8, device=dev)
        hm = torch.empty((1, n), dtype=torch.uint8).pin_memory()

        def step():
            dd.dedisp_rfi_mask(x, dd.DEDISP_OUT_F32, nb, 1, n, n * 4, mean, sigma, 3.0, 4, m, stream.cuda_stream)

        def e2e():
            x.copy_(hx, non_blocking=True)
            step()
            hm.copy_(m, non_blocking=True)
            torch.cuda.synchronize()
        units, unit, alg = n, "masked samples/s", nb * n * 4 + n
        h2d, d2h = nb * n * 4, n
        cfg = {"workload": "rfi_mask, seeded unit Gaussian series", "nbeams": nb, "nseries": 1, "nsamps": n,
               "nsigma": 3.0, "min_beams": 4}
        kern, metric, dtype = "rfi_mask_kernel", "RFI-mask samples/sec", "f32 compare"
        if not args.no_cpu_baseline:
            from oracle import rfi_mask as RM
            sub = hx[:, :, : 1 << 21].numpy()
            t0 = time.perf_counter()
            RM.coincidence_mask(sub, np.zeros((nb, 1)), np.ones((nb, 1)), 3.0, 4)
            dt = time.perf_counter() - t0
            cpu = {"value": sub.shape[2] / dt, "unit": unit, "cores": 1, "kind": "oracle",
                   "sample": f"first {sub.shape[2]} of {n} samples x {nb} beams, {dt:.2f} s"}
    else:
        w = W.CONFIGS[args.config].scaled(nbeams=1)
        plan = dd.dedisp_plan_create(w.nchans, w.dt, w.f_top, w.df)
        dd.dedisp_set_dm_list(plan, list(w.dms()))
        nin = w.nsamps_out + dd.dedisp_get_max_delay(plan)
        dd.dedisp_destroy(plan)
        nbytes = nin * w.nchans * w.nbits // 8
        hs = torch.from_numpy(np.random.default_rng(w.seed).integers(0, 256, nbytes, dtype=np.uint8)).pin_memory()
        sd = hs.to(dev)
        stride = (nin * w.nbits + 7) // 8
        out = torch.empty((w.nchans, stride), dtype=torch.uint8, device=dev)
        ho = torch.empty((w.nchans, stride), dtype=torch.uint8).pin_memory()

        def step():
            dd.dedisp_transpose_time_major(sd, w.nchans, nin, w.nbits, out, stream.cuda_stream)

        def e2e():
            sd.copy_(hs, non_blocking=True)
            step()
            ho.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        units, unit, alg = nin * w.nchans, "transposed samples/s", nbytes + w.nchans * stride
        h2d, d2h = nbytes, w.nchans * stride
        cfg = {"workload": f"time-major stream of {w.name} -> channel-major rows", "nchans": w.nchans,
               "nsamps_in": nin, "nbits": w.nbits}
        kern, metric, dtype = "time_major_kernel", "transposed samples/sec", "u8 bit re-layout"
        if not args.no_cpu_baseline:
            from oracle import time_major as TM
            k = min(nin, 1 << 16)
            t0 = time.perf_counter()
            TM.to_channel_major(hs.numpy(), w.nchans, k, w.nbits)
            dt = time.perf_counter() - t0
            cpu = {"value": k * w.nchans / dt, "unit": unit, "cores": 1, "kind": "oracle",
                   "sample": f"first {k} of {nin} time samples x {w.nchans} channels, {dt:.2f} s"}
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.15)
    launches0 = dd.dedisp_get_launch_count()
    step_ms = _time_steps(torch, step, flush, stream, args.warmup, args.steps)
    launches = dd.dedisp_get_launch_count() - launches0 - args.warmup
    clocks = sampler.stop()
    ms = statistics.mean(step_ms)
    e2e()
    t0 = time.perf_counter()
    e2e()
    e2e_s = time.perf_counter() - t0
    res = {"metric": metric, "value": units / (ms * 1e-3), "unit": unit, "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": dtype, "data": "synthetic",
           "config": dict(cfg, l2="256 MiB flush buffer zeroed between timed iterations"),
           "roofline": {"bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                        "frac": alg / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": ncu_traffic_bytes(args.op),
                        "kernel": kern, "kernel_ms": ms,
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s"},
           "cpu_baseline": cpu,
           "e2e": {"value": units / e2e_s, "unit": unit, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "steps": 1},
           "gpu_launches": launches, "clocks": clocks,
           "step_ms_min_med_max": [min(step_ms), statistics.median(step_ms), max(step_ms)]}
    print(json.dumps(res), flush=True)


def run_reference(args) -> None:
    """The oracle, as it stands, on the host cores: the base contract's reference arm."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w = W.CONFIGS[args.config]
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w.scaled(nbeams=1), md)
    stride = max(1, w.ndm // 120)
    sub = np.ascontiguousarray(delay[:, ::stride])
    units = sub.shape[1] * w.nsamps_out
    used = 0
    for _ in range(args.warmup):
        oracle.dedisperse(sub, x, w.nbits, w.nsamps_out)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, used = oracle.dedisperse(sub, x, w.nbits, w.nsamps_out, return_threads=True)
    dt = (time.perf_counter() - t0) / args.steps
    value = units / dt
    sample = (f"{sub.shape[1]} of {w.ndm} DM trials (every {stride}th) x {w.nsamps_out} samples x "
              f"{w.nchans} channels of {w.name} per step")
    res = {"impl": "reference", "metric": "DM-trial samples/sec", "value": value,
           "unit": "DM-trial-samples/s", "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32",
           "data": "synthetic",
           # the same config block as the CUDA arm prints (the bounded sample is described under cpu_baseline)
           "config": {"workload": w.name, "nchans": w.nchans, "ndm": w.ndm, "nsamps_out": w.nsamps_out,
                      "nbits": w.nbits, "tscrunch": 1, "nbeams_per_gpu": w.nbeams, "out_dtype": w.out_dtype,
                      "max_delay": md, "l2": "256 MiB flush buffer zeroed between timed iterations",
                      "parallelism": f"replicas x{int(os.environ.get('WORLD_SIZE', '1'))} (one seeded beam set per GPU, "
                                     "no collective)"},
           "sample": sample,
           "cpu_baseline": {"value": value, "unit": "DM-trial-samples/s", "cores": used,
                            "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": "DM-trial-samples/s", "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(res), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="htru_gulp", choices=W.CONFIG_ORDER + W.EXTRA_CONFIGS)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false",
                    help="skip the per_config block (the other four BASELINE configs, timed in the default run)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "bitslice", "pairs", "quads"],
                    help="A/B: force the plain tiled kernel or its pair-row variant (dedisp_set_kernel)")
    ap.add_argument("--search-mode", default="fused", choices=["fused", "dense"],
                    help="--op search: dedisp_search_events (no z written; default) or the dense two-call chain")
    ap.add_argument("--tscrunch", type=int, default=1,
                    help="--op dedisperse only: sum blocks of K input samples and dedisperse on the grid K*dt "
                         "(row f4; the input then holds K x as many samples per output sample)")
    ap.add_argument("--op", default="dedisperse", choices=["dedisperse", "matched_filter", "find_events", "search", "rfi_mask", "transpose"],
                    help="dedisperse = the hot path (default, the metric BASELINE.json names); "
                         "matched_filter = row f1 downstream of it; find_events = row f2 downstream of f1; search = f1 + f2 chained (matched_filter_rms + find_events); rfi_mask = row f3; transpose = row f4")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.op in ("matched_filter", "find_events", "search"):
        run_matched_filter(args)
    elif args.op in ("rfi_mask", "transpose"):
        run_small_op(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
