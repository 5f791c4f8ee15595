"""Builds libdedisp_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch).

    python -m paper_1112_0065_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libdedisp_b200.so"
SOURCES = ["dedisp_api.cu", "delay_table.cu", "direct_kernel.cu", "bitslice_prepare.cu", "bitslice_kernel.cu",
           "pair_rows.cu", "probe.cu", "matched_filter.cu", "peak_finding.cu", "rfi_mask.cu", "time_major.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=false", "-Xptxas", "-v"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    raise RuntimeError("nvcc not found")


def stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = [CSRC / s for s in SOURCES] + list(CSRC.glob("*.h")) + list(CSRC.glob("*.cuh")) \
        + [INCLUDE / "dedisp.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False, defs: list[str] | None = None,
          out: Path | None = None) -> Path:
    """defs/out: tuning variants for A/B runs (e.g. defs=["BS_NW=20"], out=Path("x.so"))."""
    target = Path(out) if out else LIB
    if not force and not defs and not out and not stale():
        return LIB
    tmp = target.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [_nvcc(), *NVCC_FLAGS, *[f"-D{d}" for d in (defs or [])], f"-I{INCLUDE}", f"-I{CSRC}",
           "-o", str(tmp)] + [str(CSRC / s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libdedisp_b200.so")
    (target.parent / (target.stem + "_ptxas.log")).write_text(r.stdout + r.stderr)
    os.replace(tmp, target)
    return target


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
