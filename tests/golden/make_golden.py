"""Writes tests/golden/full_size.json: sha256 / sum / spot values of the ORACLE's
output on the five BASELINE.json configs (full size), plus sha256 of each packed
input.  Calls only ``oracle/`` and the seeded generators -- never the CUDA path.

    python tests/golden/make_golden.py            # all five (~3 min on 8 cores)
    python tests/golden/make_golden.py tiny htru_gulp
"""
import hashlib
import json
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))
import oracle  # noqa: E402
import workloads as W  # noqa: E402

OUT = Path(__file__).resolve().parent / "full_size.json"


def oracle_inputs(w):
    """Delay table, max_delay and the packed input [nbeams, nchans, stride] of a config."""
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    kw = {}
    if w.kind == "gauss2_pulses":
        p = W.pulse_params(w)
        sweep, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, p.dm)
        kw = dict(pulse_sweep=sweep, pulses=p)
    return delay, md, W.generate_all_beams(w, md, **kw)


def spot_index(w):
    """Fixed (beam, d, t) sample points recorded per config."""
    return [(0, 0, 0), (0, 0, 1), (0, w.ndm // 2, w.nsamps_out // 2),
            (w.nbeams - 1, w.ndm - 1, w.nsamps_out - 1), (w.nbeams - 1, w.ndm - 1, w.nsamps_out - 2)]


def main(names):
    res = json.loads(OUT.read_text()) if OUT.exists() else {}
    for name in names:
        w = W.CONFIGS[name]
        t0 = time.time()
        delay, md, x = oracle_inputs(w)
        h = hashlib.sha256()
        total = 0
        spots = {}
        omin, omax = None, None
        for b in range(w.nbeams):
            o = oracle.dedisperse(delay, x[b], w.nbits, w.nsamps_out)
            total += int(o.sum(dtype=np.uint64))
            omin = int(o.min()) if omin is None else min(omin, int(o.min()))
            omax = int(o.max()) if omax is None else max(omax, int(o.max()))
            for (bb, d, t) in spot_index(w):
                if bb == b:
                    spots[f"{bb},{d},{t}"] = int(o[d, t])
            view = oracle.to_f32(o) if w.out_dtype == "f32" else o
            h.update(view.tobytes())      # little-endian, [beam][d][t]
        res[name] = dict(max_delay=md, in_sha256=W.sha256(x), in_shape=list(x.shape),
                         out_dtype=w.out_dtype, out_sha256=h.hexdigest(), out_sum=total,
                         out_min=omin, out_max=omax, spots=spots)
        print(name, res[name], f"{time.time() - t0:.1f}s", flush=True)
        OUT.write_text(json.dumps(res, indent=1, sort_keys=True) + "\n")


if __name__ == "__main__":
    main(sys.argv[1:] or W.CONFIG_ORDER)
