"""Oracle + generator vs the stored goldens (no GPU).

tests/golden/full_size.json is written by tests/golden/make_golden.py, which
calls only oracle/.  The tiny and HTRU-gulp entries are ALSO pinned to values
that SURVEY.md Sec. 8(d) ("Generator goldens") obtained with an independent NumPy
slice-sum over exact-rational delay tables -- a third implementation.
"""
import json

import numpy as np
import pytest

import oracle
import workloads as W

SURVEY_GOLDENS = {  # SURVEY.md Sec. 8(d), table "Generator goldens"
    "tiny": dict(in_sha256="7c2cb4eae172d38b5f530334bacd060ab05ae221251e3c999c7fbdcc82eeb8c1",
                 out_sha256="60aa84d194809b1c7df309c9733a26dd8f8be87252e956345d3ffdda962df222",
                 out_sum=12574321, head=[86, 99, 99, 105], tail=[89, 95, 105, 92]),
    "htru_gulp": dict(in_sha256="e95970ababa0675d397fd110b76fbefc2ae1a168efe01607d8c2a845072920b9",
                      out_sha256="2aafd6bddfd4533d491b0a92d15f64c0317b5f8de2318d1694e6638022f7e9ec",
                      out_sum=120803264979, head=[1507, 1538, 1558, 1534],
                      tail=[1576, 1479, 1535, 1558]),
}


@pytest.mark.parametrize("name", ["tiny", "htru_gulp"])
def test_oracle_matches_goldens(name, golden_dir):
    stored = json.loads((golden_dir / "full_size.json").read_text())[name]
    w = W.CONFIGS[name]
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    x = W.generate(w, md)
    o = oracle.dedisperse(delay, x, w.nbits, w.nsamps_out)
    s = SURVEY_GOLDENS[name]
    assert W.sha256(x) == s["in_sha256"] == stored["in_sha256"]
    assert W.sha256(o) == s["out_sha256"] == stored["out_sha256"]
    assert int(o.sum(dtype=np.uint64)) == s["out_sum"] == stored["out_sum"]
    assert o[0, :4].tolist() == s["head"] and o[-1, -4:].tolist() == s["tail"]
    assert md == stored["max_delay"]
    # quantised-Gaussian / uniform statistics (SURVEY.md Sec. 8(c) "Bounds / statistics")
    if name == "htru_gulp":
        assert abs(o.mean() - 1536.0) < 0.5 and abs(o.std() - 30.10) < 0.1
        # literal loop on a few whole trials of the big config
        part = np.ascontiguousarray(delay[:, [0, 599, 1199]])
        lit = oracle.dedisperse_literal(part, x, w.nbits, 2048)
        assert np.array_equal(lit, o[[0, 599, 1199], :2048])


def test_all_five_configs_have_goldens(golden_dir):
    stored = json.loads((golden_dir / "full_size.json").read_text())
    assert sorted(stored) == sorted(W.CONFIG_ORDER)
    assert stored["wide8"]["max_delay"] == 49508 and stored["beams13"]["in_shape"][0] == 13


def test_generators_are_seeded_and_shaped():
    w = W.CONFIGS["tiny"]
    a, b = W.generate(w, 4004), W.generate(w, 4004)
    assert np.array_equal(a, b) and a.shape == (64, 2025)
    w13 = W.CONFIGS["beams13"].scaled(nsamps_out=512, nchans=8)
    x = W.generate_all_beams(w13, 100)
    assert x.shape == (13, 8, 153) and len({W.sha256(x[i]) for i in range(13)}) == 13
    w8 = W.CONFIGS["wide8"].scaled(nsamps_out=20000, nchans=4)
    x8 = W.generate(w8, 0)
    assert abs(x8.mean() - 128) < 0.5 and abs(x8.std() - 16) < 0.3
    # quantised Gaussian level probabilities .1587/.3413/.3413/.1587
    wg = W.CONFIGS["htru_gulp"].scaled(nsamps_out=40000, nchans=4)
    lev = np.stack([W.unpack2(r, 40000) for r in W.generate(wg, 0)])
    p = np.bincount(lev.ravel(), minlength=4) / lev.size
    assert np.allclose(p, [0.1587, 0.3413, 0.3413, 0.1587], atol=0.005)


def test_pulse_injection_raises_level_along_sweep():
    w = W.CONFIGS["htru_long_pulses"].scaled(nsamps_out=8192, nchans=32, df=-12.5)
    p = W.pulse_params(w)
    assert p.dm.shape == (16,) and (p.dm >= 50).all() and (p.dm <= 900).all()
    assert (p.width >= 1).all() and (p.width <= 64).all() and (p.t0 + p.width <= w.nsamps_out).all()
    delay, md = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, w.dms())
    sweep, _ = oracle.delay_table(w.nchans, w.dt, w.f_top, w.df, p.dm)
    x = W.generate(w, md, pulse_sweep=sweep, pulses=p)
    x0 = W.generate(w.scaled(kind="gauss2"), md)
    lev = np.stack([W.unpack2(r, w.nsamps_out + md) for r in x]).astype(int)
    lev0 = np.stack([W.unpack2(r, w.nsamps_out + md) for r in x0]).astype(int)
    diff = lev - lev0
    assert (diff >= 0).all() and diff.sum() > 0
    # every changed sample lies on some pulse's sweep
    on = np.zeros_like(diff, dtype=bool)
    for c in range(w.nchans):
        for k in range(16):
            a = p.t0[k] + sweep[c, k]
            on[c, a:a + p.width[k]] = True
    assert not diff[~on].any()
    # mean level shift of a +1 sigma pulse is 0.8186 per covered sample
    assert abs(diff[on].mean() - 0.8186) < 0.08
