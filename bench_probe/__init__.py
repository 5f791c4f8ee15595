"""Bench-side instruction-rate probe (not part of the product library).

``probe_alu_rate(which)`` runs the register-only micro-benchmark of ``probe.cu`` on the current CUDA
device and returns lane-operations per second; ``bench.py`` prints it beside the ALU roofline
denominator ("run a register-only FADD / IADD3 microbenchmark and print the
measured peak").  Built in-tree by ``build()`` into ``bench_probe/libdedisp_probe.so``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

_DIR = Path(__file__).resolve().parent
LIB = _DIR / "libdedisp_probe.so"
NAMES = ["iadd3", "lop3", "shf", "fadd", "imad", "lop3+imad", "lds32", "lds128", "prmt", "dp4a"]
_lib = None


def build(force: bool = False) -> Path:
    src = _DIR / "probe.cu"
    if not force and LIB.exists() and LIB.stat().st_mtime >= src.stat().st_mtime:
        return LIB
    nvcc = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
           "-shared", "-o", str(tmp), str(src)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libdedisp_probe.so\n" + r.stdout + r.stderr)
    os.replace(tmp, LIB)
    return LIB


def probe_alu_rate(which: int) -> float:
    global _lib
    if _lib is None:
        if not LIB.exists():
            raise RuntimeError(f"{LIB} is not built: run bench_probe.build()")
        _lib = ctypes.CDLL(str(LIB))
        _lib.probe_alu_rate.restype = ctypes.c_int
        _lib.probe_alu_rate.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    v = ctypes.c_double()
    st = _lib.probe_alu_rate(which, ctypes.byref(v))
    if st != 0:
        raise RuntimeError(f"probe_alu_rate({which}) failed with status {st}")
    return v.value
