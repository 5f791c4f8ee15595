"""Seeded synthetic filterbank workloads (the five BASELINE.json configs).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, so
it holds none of the method's arithmetic: no delay formula, no dedispersion
sum.  Anything that depends on the delay table (``max_delay`` for the row
length, the sweep of an injected pulse) is passed in by the caller, who gets it
from whichever implementation it is exercising.

The inputs stand in for HTRU survey recordings (Sec. 1: 1024
channels over 400 MHz centred at 1381.8 MHz, 64 us, 2 bits per sample), which
are not available here.  Recipes follow SURVEY.md Sec. 8(d); DESIGN.md restates
them.  NumPy only (no torch, no CUDA).
"""
from __future__ import annotations

import hashlib
import math
from dataclasses import dataclass, replace
from typing import Callable

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    nchans: int
    f_top: float          # MHz, frequency of channel 0
    df: float             # MHz, channel spacing (negative)
    dt: float             # s
    nbits: int            # 1, 2, 4 or 8
    ndm: int
    dm_lo: float
    dm_hi: float
    nsamps_out: int
    out_dtype: str        # "u32" | "f32"
    nbeams: int
    seed: int
    kind: str             # "uniform2" | "gauss2" | "gauss2_pulses" | "gauss8" | "uniform"
    npulses: int = 0

    def dms(self) -> np.ndarray:
        """Trial DM list: inclusive linear spacing (numpy.linspace), float64."""
        return np.linspace(self.dm_lo, self.dm_hi, self.ndm, dtype=np.float64)

    def obs_seconds(self) -> float:
        return self.nsamps_out * self.dt

    def dm_trial_samples(self) -> int:
        return self.nbeams * self.ndm * self.nsamps_out

    def adds(self) -> int:
        return self.dm_trial_samples() * self.nchans

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


CONFIGS: dict[str, Workload] = {
    "tiny": Workload("tiny", 64, 1581.8, -6.25, 64e-6, 2, 32, 0.0, 200.0, 4096, "u32", 1, 1001,
                     "uniform2"),
    "htru_gulp": Workload("htru_gulp", 1024, 1581.8, -0.390625, 64e-6, 2, 1200, 0.0, 1000.0, 65536,
                          "u32", 1, 1002, "gauss2"),
    "htru_long_pulses": Workload("htru_long_pulses", 1024, 1581.8, -0.390625, 64e-6, 2, 1200, 0.0,
                                 1000.0, 524288, "f32", 1, 1003, "gauss2_pulses", npulses=16),
    "wide8": Workload("wide8", 4096, 1500.0, -0.09765625, 64e-6, 8, 2048, 0.0, 2000.0, 131072,
                      "u32", 1, 1004, "gauss8"),
    "beams13": Workload("beams13", 1024, 1581.8, -0.390625, 64e-6, 2, 1200, 0.0, 1000.0, 65536,
                        "u32", 13, 1100, "gauss2"),
}
CONFIG_ORDER = ["tiny", "htru_gulp", "htru_long_pulses", "wide8", "beams13"]   # BASELINE.json configs
# input-format variants: the HTRU gulp shape with 1- and 4-bit samples,
# levels uniform on [0, 2^nbits) -- not BASELINE configs, bench/profile lines only
CONFIGS["htru_gulp_1bit"] = replace(CONFIGS["htru_gulp"], name="htru_gulp_1bit", nbits=1, seed=1201,
                                    kind="uniform")
CONFIGS["htru_gulp_4bit"] = replace(CONFIGS["htru_gulp"], name="htru_gulp_4bit", nbits=4, seed=1204,
                                    kind="uniform")
EXTRA_CONFIGS = ["htru_gulp_1bit", "htru_gulp_4bit"]


def _phi(x: float) -> float:
    """Standard normal CDF."""
    return 0.5 * (1.0 + math.erf(x / math.sqrt(2.0)))


# Quantiser thresholds at -1, 0, +1 sigma expressed on the uniform variate.
_THR = np.array([_phi(-1.0), 0.5, _phi(1.0)], dtype=np.float64)


def row_stride_bytes(nsamps_in: int, nbits: int) -> int:
    """Tight packed row length in bytes."""
    return (nsamps_in * nbits + 7) // 8


def pack2(levels: np.ndarray) -> np.ndarray:
    """Pack 2-bit levels (values 0..3, 1-D) LSB-first, 4 per byte, zero padded."""
    n = levels.shape[0]
    nb = (n + 3) // 4
    buf = np.zeros(nb * 4, dtype=np.uint8)
    buf[:n] = levels
    q = buf.reshape(nb, 4)
    return (q[:, 0] | (q[:, 1] << 2) | (q[:, 2] << 4) | (q[:, 3] << 6)).astype(np.uint8)


def unpack2(row: np.ndarray, nsamps: int) -> np.ndarray:
    """Inverse of :func:`pack2` (test helper; a layout statement, not the method)."""
    sh = np.arange(4, dtype=np.uint8) * 2
    return ((row[:, None] >> sh[None, :]) & 3).reshape(-1)[:nsamps].astype(np.uint8)


def pack_bits(levels: np.ndarray, nbits: int) -> np.ndarray:
    """Pack levels (1-D, values < 2**nbits, nbits in 1/2/4/8) LSB-first into bytes, zero padded:
    sample t occupies bits [t*nbits, (t+1)*nbits) of the row read as a little-endian bit string."""
    if nbits == 8:
        return levels.astype(np.uint8)
    per = 8 // nbits
    n = levels.shape[0]
    nb = (n + per - 1) // per
    buf = np.zeros(nb * per, dtype=np.uint8)
    buf[:n] = levels
    q = buf.reshape(nb, per)
    out = np.zeros(nb, dtype=np.uint8)
    for k in range(per):
        out |= (q[:, k] << (k * nbits)).astype(np.uint8)
    return out


def unpack_bits(row: np.ndarray, nbits: int, nsamps: int) -> np.ndarray:
    """Inverse of :func:`pack_bits` through numpy.unpackbits (a layout statement for tests)."""
    if nbits == 8:
        return row[:nsamps].astype(np.uint8)
    bits = np.unpackbits(row, bitorder="little")[: nsamps * nbits].reshape(nsamps, nbits)
    return (bits << np.arange(nbits, dtype=np.uint8)).sum(axis=1).astype(np.uint8)


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=np.array([seed, stream], dtype=np.uint64)))


@dataclass(frozen=True)
class Pulses:
    dm: np.ndarray        # float64 [npulses]
    width: np.ndarray     # int64   [npulses]
    t0: np.ndarray        # int64   [npulses]


def pulse_params(w: Workload) -> Pulses:
    """Seeded pulse list for the injected-pulse config: DM uniform 50..900, width
    1..64 samples, start uniform over the output span.  Stream key (seed, 1<<48)
    is used by no data row."""
    u = _rng(w.seed, 1 << 48).random((w.npulses, 3))
    dm = 50.0 + 850.0 * u[:, 0]
    width = 1 + np.floor(64.0 * u[:, 1]).astype(np.int64)
    t0 = np.floor(u[:, 2] * (w.nsamps_out - width)).astype(np.int64)
    return Pulses(dm, width, t0)


def generate(w: Workload, max_delay: int, beam: int = 0,
             pulse_sweep: np.ndarray | None = None, pulses: Pulses | None = None) -> np.ndarray:
    """Packed input of one beam: uint8 [nchans, row_stride], channel-major, tight rows.

    ``max_delay`` comes from the caller's delay table (nsamps_in = nsamps_out +
    max_delay).  For ``gauss2_pulses``, ``pulse_sweep[c][p]`` is the delay in
    samples of pulse p at channel c (same source) and ``pulses`` the output of
    :func:`pulse_params`.
    """
    nsamps_in = w.nsamps_out + int(max_delay)
    stride = row_stride_bytes(nsamps_in, w.nbits)
    out = np.zeros((w.nchans, stride), dtype=np.uint8)
    seed = w.seed + beam if w.nbeams > 1 else w.seed
    if w.kind == "gauss2_pulses":
        if pulse_sweep is None or pulses is None:
            raise ValueError("gauss2_pulses needs pulse_sweep and pulses")
        kmax = w.npulses
        thr_k = np.array([[_phi(j - k) for j in (-1.0, 0.0, 1.0)] for k in range(kmax + 1)])
    for c in range(w.nchans):
        g = _rng(seed, (beam << 32) | c)
        if w.kind == "uniform":
            out[c] = pack_bits((g.random(nsamps_in) * (1 << w.nbits)).astype(np.uint8), w.nbits)
        elif w.kind == "uniform2":
            u = g.random(nsamps_in)
            lev = (u * 4).astype(np.uint8)
            out[c] = pack2(lev)
        elif w.kind in ("gauss2", "gauss2_pulses"):
            u = g.random(nsamps_in)
            lev = np.searchsorted(_THR, u, side="right").astype(np.uint8)
            if w.kind == "gauss2_pulses":
                # k[t] = number of pulse sweeps covering sample t of this channel;
                # a +1 sigma shift per pulse before quantisation == thresholds Phi(j-k).
                diff = np.zeros(nsamps_in + 1, dtype=np.int32)
                for p in range(w.npulses):
                    a = int(pulses.t0[p]) + int(pulse_sweep[c, p])
                    b = a + int(pulses.width[p])
                    a, b = min(a, nsamps_in), min(b, nsamps_in)
                    diff[a] += 1
                    diff[b] -= 1
                k = np.cumsum(diff[:-1])
                idx = np.nonzero(k)[0]
                if idx.size:
                    t = thr_k[k[idx]]
                    uu = u[idx]
                    lev[idx] = ((uu >= t[:, 0]).astype(np.uint8) + (uu >= t[:, 1])
                                + (uu >= t[:, 2])).astype(np.uint8)
            out[c] = pack2(lev)
        elif w.kind == "gauss8":
            gs = g.standard_normal(nsamps_in)
            out[c] = np.clip(np.floor(128.0 + 16.0 * gs + 0.5), 0, 255).astype(np.uint8)
        else:
            raise ValueError(w.kind)
    return out


def generate_all_beams(w: Workload, max_delay: int, **kw) -> np.ndarray:
    """uint8 [nbeams, nchans, row_stride] -- beams contiguous."""
    return np.stack([generate(w, max_delay, beam=b, **kw) for b in range(w.nbeams)])


def random_small(seed: int, nchans: int, nsamps_in: int, nbits: int) -> np.ndarray:
    """Uniform random packed rows for the random-shape parity cases."""
    g = _rng(seed, 7)
    if nbits == 8:
        return g.integers(0, 256, size=(nchans, nsamps_in), dtype=np.uint8)
    lev = (g.random((nchans, nsamps_in)) * (1 << nbits)).astype(np.uint8)
    if nbits == 2:
        return np.stack([pack2(lev[c]) for c in range(nchans)])
    return np.stack([pack_bits(lev[c], nbits) for c in range(nchans)])


def dedispersed_like(seed: int, nrows: int, nsamps: int, mean: float = 1536.0, sigma: float = 30.1,
                     x_max: int = 3072, wiggle: float = 40.0, npulses: int = 3) -> np.ndarray:
    """Seeded stand-in for dedispersed time series (input of the matched-filter row f1):
    uint32 [nrows, nsamps] = Gaussian noise (mean, sigma: the HTRU-gulp output statistics)
    + a slow baseline wiggle (two sinusoids with periods of ~nsamps/3 and ~nsamps/11, the
    "red noise" of PAPER.md:52) + npulses boxcar pulses per row (width 1..64, height
    3..8 sigma/sqrt(width)), rounded and clipped to [0, x_max]."""
    out = np.empty((nrows, nsamps), dtype=np.uint32)
    t = np.arange(nsamps, dtype=np.float64)
    for r in range(nrows):
        g = _rng(seed, (3 << 48) | r)
        v = mean + sigma * g.standard_normal(nsamps)
        ph = g.random(2) * 2 * np.pi
        v += wiggle * np.sin(2 * np.pi * 3 * t / nsamps + ph[0]) + 0.5 * wiggle * np.sin(2 * np.pi * 11 * t / nsamps + ph[1])
        u = g.random((npulses, 3))
        for k in range(npulses):
            wd = 1 + int(64 * u[k, 0])
            if wd >= nsamps:
                continue
            t0 = int(u[k, 1] * (nsamps - wd))
            v[t0:t0 + wd] += (3.0 + 5.0 * u[k, 2]) * sigma / np.sqrt(wd)
        out[r] = np.clip(np.floor(v + 0.5), 0, x_max).astype(np.uint32)
    return out


def filtered_like(seed: int, nseries: int, nsamps: int, sigma: float = 30.1, npulses: int = 4,
                  max_width: int = 3000) -> np.ndarray:
    """Seeded stand-in for matched-filter output (input of the peak-finding row f2):
    float32 [nseries, nsamps] = zero-mean Gaussian noise of the given sigma + npulses flat-topped
    pulses per series (width 1..max_width, log-uniform, so that runs cross 32-sample words and
    1024-sample chunks; height 6..12 sigma with a small seeded ripple so maxima are unique)."""
    out = np.empty((nseries, nsamps), dtype=np.float32)
    for r in range(nseries):
        g = _rng(seed, (5 << 48) | r)
        v = sigma * g.standard_normal(nsamps)
        u = g.random((npulses, 3))
        for k in range(npulses):
            wd = min(nsamps, int(np.exp(u[k, 0] * np.log(max_width))))
            t0 = int(u[k, 1] * (nsamps - wd + 1))
            v[t0:t0 + wd] += (6.0 + 6.0 * u[k, 2]) * sigma
        out[r] = v.astype(np.float32)
    return out


def sha256(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
