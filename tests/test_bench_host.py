"""-m "not gpu": the host-side bookkeeping of bench.py -- the roofline arithmetic, the table of committed ncu
captures (profiles/traffic.csv), the instruction-level bound and the reference arm's JSON line.  No kernel runs here;
the numbers checked are definitions (BASELINE.json:north_star: adds = nchans * ndm * nsamps_out against
SMs x 128 adds/clk x clock), not measurements."""
import json
import subprocess
import sys
from pathlib import Path
from types import SimpleNamespace

import pytest

import bench
import workloads as W

ROOT = Path(__file__).resolve().parent.parent


def test_traffic_table_rows_are_kernel_aware():
    quads, pairs = bench.KERNEL_NAMES[4], bench.KERNEL_NAMES[3]
    tq = bench.ncu_traffic("wide8", quads)
    tp = bench.ncu_traffic("wide8", pairs)
    assert tq[0] and tp[0] and tq[0] != tp[0]          # one row per kernel the config was captured with
    assert tq[1] == tp[1] == "profiles/r2_wide8.md" and (ROOT / tq[1]).exists()
    assert bench.ncu_traffic("wide8", bench.KERNEL_NAMES[2]) == (None, None, None)    # no capture of that kernel
    assert bench.ncu_traffic("htru_gulp", pairs)[0] == bench.ncu_traffic_bytes("htru_gulp")
    assert bench.ncu_traffic("no_such_config") == (None, None, None)
    # rows without a kernel column serve any caller; every source file named in the table is committed
    assert bench.ncu_traffic("rfi_mask", "anything")[0] == bench.ncu_traffic_bytes("rfi_mask")
    for line in (ROOT / "profiles" / "traffic.csv").read_text().splitlines():
        f = line.split(",")
        if line.startswith("#") or f[0] == "config":
            continue
        assert float(f[1]) > 0 and (ROOT / f[2]).exists(), line
        if len(f) > 4 and f[4]:
            assert f[4] in bench.KERNEL_NAMES.values(), line


def test_instruction_bound_table_names_known_kernels_and_widths():
    for (kernel, nbits), (per_add, src) in bench.ALU_PIPE_INSTR_PER_ADD.items():
        assert kernel in bench.KERNEL_NAMES and nbits in (1, 2, 4, 8)
        assert 0.05 < per_add < 1.0           # bit-sliced: far fewer than one instruction per addition
        assert src.split(":")[0].startswith(("profiles/", "DESIGN.md"))
        if src.startswith("profiles/"):
            assert (ROOT / src.split(":")[0]).exists()


def test_roofline_arithmetic_of_the_headline_config():
    w = W.CONFIGS["htru_gulp"]
    props = SimpleNamespace(multi_processor_count=148)
    peaks = {"sm_max_mhz": 1965.0, "hbm_gbs": 6650.0}
    kernel_ms, pre_ms, step_ms = 0.931, 0.094, 1.034
    m = {"main_ms": [kernel_ms] * 3, "pre_ms": [pre_ms] * 3, "kernel_used": 3,
         "in_bytes": 22_000_000, "out_bytes": 314_572_800}
    r = bench.roofline_of(w, 1, m, step_ms, props, peaks, "htru_gulp")
    adds = 1024 * 1200 * 65536
    assert w.adds() == adds
    peak = 148 * bench.ADDS_PER_CLK_PER_SM * 1965.0e6
    assert r["bound"] == "alu" and r["unit"] == "Tadd/s"
    assert r["peak"] == pytest.approx(peak / 1e12) and r["achieved"] == pytest.approx(adds / (kernel_ms * 1e-3) / 1e12)
    assert r["frac"] == pytest.approx(r["achieved"] / r["peak"])
    assert r["kernel"] == "bitslice_dedisperse on pair rows" and r["traffic"] == bench.ncu_traffic_bytes("htru_gulp")
    assert r["kernel_share_of_step"] == pytest.approx(kernel_ms / step_ms)
    assert r["algorithmic_bytes"] == m["in_bytes"] + m["out_bytes"]
    # the step's fraction: the same adds over the whole step (pre-passes inside)
    assert r["step_roofline_frac"] == pytest.approx(adds / (step_ms * 1e-3) / peak)
    # the instruction-level bound of this kernel: counted ALU-pipe instructions per add against the 64-lane pipe
    ib = r["instr_bound"]
    per_add = bench.ALU_PIPE_INSTR_PER_ADD[(3, 2)][0]
    assert ib["frac"] == pytest.approx(per_add * adds / (kernel_ms * 1e-3) / (148 * 64 * 1965.0e6))
    assert 0.5 < ib["frac"] < 1.0
    # time-scrunched runs carry no instruction count
    assert bench.roofline_of(w, 4, m, step_ms, props, peaks, "htru_gulp")["instr_bound"] is None


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["metric"] == "DM-trial samples/sec" and j["higher_is_better"] is True
    assert j["n_gpus"] == 1 and j["steps"] == 1 and j["warmup"] == 0 and j["vs_baseline"] is None
    assert j["config"]["workload"] == "htru_gulp" and j["config"]["nchans"] == 1024 and j["config"]["ndm"] == 1200
    assert j["e2e"] == {"value": j["value"], "unit": j["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    cb = j["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == j["value"] and cb["sample"]
    assert j["value"] > 0 and j["ms_per_step"] > 0
