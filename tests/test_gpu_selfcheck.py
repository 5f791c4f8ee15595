"""-m gpu: the hazard cases of tests/hazard_cases.py (SURVEY.md Sec. 4 tier T3) through both builds of the library --
the product build (parity + output guard zones + scratch poisoning) and the -DDEDISP_CHECKS build (in-kernel range /
ring-stage checks must count zero failures).  compute-sanitizer itself is closed on this GPU pool; see
profiles/r2_sanitizer.md."""
import os
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent
CHECKS_LIB = ROOT / "paper_1112_0065_b200" / "libdedisp_b200_checks.so"
NCASES = 10      # tests/hazard_cases.py::CASES


def _run_cases(env_extra):
    env = dict(os.environ, **env_extra)
    r = subprocess.run([sys.executable, str(ROOT / "tests" / "hazard_cases.py")], capture_output=True, text=True,
                       env=env, timeout=1500)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    return r.stdout


def test_hazard_cases_product_build():
    out = _run_cases({"DEDISP_B200_LIB": ""})
    assert f"{NCASES} cases ok" in out and "checks compiled: False" in out


def test_hazard_cases_with_in_kernel_checks():
    from paper_1112_0065_b200 import build
    if not CHECKS_LIB.exists() or build.stale(CHECKS_LIB):
        build.build(defs=["DEDISP_CHECKS"], out=CHECKS_LIB)
    out = _run_cases({"DEDISP_B200_LIB": str(CHECKS_LIB)})
    assert f"{NCASES} cases ok" in out and "checks compiled: True" in out
