"""CPU oracle for direct incoherent dedispersion -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_1112_0065_b200``) never does, and this package never imports the product.

The arithmetic lives in ``dedisp_oracle.c`` (plain C, gcc, fp64 delays with C99
``round()``, exact integer sums); this file only builds it and marshals NumPy
arrays through ctypes.  Definition and citations: see the C file's header
(BASELINE.json:north_star; Sec. 2.2).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "dedisp_oracle.c"
_LIB = _HERE / "libdedisp_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O3, OpenMP, no FMA contraction, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-std=c99", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        i32p = ctypes.POINTER(ctypes.c_int32)
        u8p = ctypes.POINTER(ctypes.c_uint8)
        u32p = ctypes.POINTER(ctypes.c_uint32)
        f64p = ctypes.POINTER(ctypes.c_double)
        lib.oracle_delay_table.restype = ctypes.c_int64
        lib.oracle_delay_table.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                           ctypes.c_double, f64p, ctypes.c_int, i32p]
        lib.oracle_row_stride_bytes.restype = ctypes.c_int64
        lib.oracle_row_stride_bytes.argtypes = [ctypes.c_int64, ctypes.c_int]
        lib.oracle_dedisperse_literal.restype = ctypes.c_int
        lib.oracle_dedisperse_literal.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int64, i32p,
                                                  u8p, ctypes.c_int64, ctypes.c_int, u32p]
        lib.oracle_dedisperse.restype = ctypes.c_int
        lib.oracle_dedisperse.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int64, i32p,
                                          ctypes.c_int64, u8p, ctypes.c_int64, ctypes.c_int, u32p,
                                          ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.oracle_u32_to_f32.restype = None
        lib.oracle_u32_to_f32.argtypes = [u32p, ctypes.POINTER(ctypes.c_float), ctypes.c_int64]
        _lib = lib
    return _lib


def _ptr(a: np.ndarray, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def delay_table(nchans: int, dt: float, f_top: float, df: float, dms) -> tuple[np.ndarray, int]:
    """``delay[c][d]`` (int32, shape [nchans, ndm]) and ``max_delay``."""
    dms = np.ascontiguousarray(dms, dtype=np.float64)
    ndm = dms.shape[0]
    out = np.empty((nchans, ndm), dtype=np.int32)
    md = _load().oracle_delay_table(nchans, dt, f_top, df, _ptr(dms, ctypes.c_double), ndm,
                                    _ptr(out, ctypes.c_int32))
    if md < 0:
        raise ValueError("oracle_delay_table: bad argument")
    return out, int(md)


def row_stride_bytes(nsamps: int, nbits: int) -> int:
    return int(_load().oracle_row_stride_bytes(nsamps, nbits))


def _check_in(packed: np.ndarray, nchans: int):
    if packed.dtype != np.uint8 or packed.ndim != 2 or packed.shape[0] != nchans \
            or not packed.flags.c_contiguous:
        raise ValueError("packed input must be a C-contiguous uint8 array [nchans, row_stride]")


def dedisperse_literal(delay: np.ndarray, packed: np.ndarray, nbits: int,
                       nsamps_out: int) -> np.ndarray:
    """O1: literal triple loop on the packed bytes -> uint32 [ndm, nsamps_out]."""
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nchans, ndm = delay.shape
    _check_in(packed, nchans)
    need = row_stride_bytes(nsamps_out + int(delay.max()), nbits)
    if packed.shape[1] < need:
        raise ValueError("packed rows too short for nsamps_out + max_delay")
    out = np.empty((ndm, nsamps_out), dtype=np.uint32)
    rc = _load().oracle_dedisperse_literal(nchans, ndm, nsamps_out, _ptr(delay, ctypes.c_int32),
                                           _ptr(packed, ctypes.c_uint8), packed.shape[1], nbits,
                                           _ptr(out, ctypes.c_uint32))
    if rc != 0:
        raise ValueError("oracle_dedisperse_literal: bad argument")
    return out


def dedisperse(delay: np.ndarray, packed: np.ndarray, nbits: int, nsamps_out: int,
               d_begin: int = 0, d_end: int | None = None, nthreads: int = 0,
               out: np.ndarray | None = None, return_threads: bool = False):
    """O2: unpack rows once, then ``for d: for c: for t`` (OpenMP over d).

    Only trials ``d_begin <= d < d_end`` are computed (rows outside are left as
    allocated: zero for a fresh array).
    """
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nchans, ndm = delay.shape
    _check_in(packed, nchans)
    if d_end is None:
        d_end = ndm
    max_delay = int(delay.max())
    need = row_stride_bytes(nsamps_out + max_delay, nbits)
    if packed.shape[1] < need:
        raise ValueError("packed rows too short for nsamps_out + max_delay")
    if out is None:
        out = np.zeros((ndm, nsamps_out), dtype=np.uint32)
    used = _load().oracle_dedisperse(nchans, ndm, nsamps_out, _ptr(delay, ctypes.c_int32), max_delay,
                                     _ptr(packed, ctypes.c_uint8), packed.shape[1], nbits,
                                     _ptr(out, ctypes.c_uint32), d_begin, d_end, nthreads)
    if used < 0:
        raise ValueError("oracle_dedisperse: bad argument")
    return (out, used) if return_threads else out


def to_f32(out_u32: np.ndarray) -> np.ndarray:
    """Exact float32 conversion of the integer result (all sums < 2**24)."""
    src = np.ascontiguousarray(out_u32, dtype=np.uint32)
    dst = np.empty(src.shape, dtype=np.float32)
    _load().oracle_u32_to_f32(_ptr(src, ctypes.c_uint32), _ptr(dst, ctypes.c_float), src.size)
    return dst
