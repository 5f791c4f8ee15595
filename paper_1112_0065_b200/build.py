"""Builds libdedisp_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch).

    python -m paper_1112_0065_b200.build [--force] [--verbose]

Every translation unit is compiled to an object file (in parallel) and the objects are linked into
the shared library.  Objects are cached by CONTENT -- the file name carries a hash of the source, of
every header and of the flags -- so a cache left behind by another checkout or an older snapshot
can never be linked by mistake, whatever the file times say.  The cache lives in the system temp
directory (DEDISP_B200_OBJDIR overrides it): it is a few hundred MB and must not travel with the
source tree.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libdedisp_b200.so"
OBJDIR = Path(os.environ.get("DEDISP_B200_OBJDIR") or
              Path(tempfile.gettempdir()) / ("dedisp_b200_obj_" + hashlib.sha1(str(PKG).encode()).hexdigest()[:10]))
SOURCES = ["dedisp_api.cu", "delay_table.cu", "direct_kernel.cu", "bitslice_prepare.cu", "bitslice_kernel.cu",
           "bitslice_inst_cfg1.cu", "bitslice_inst_cfg2.cu", "bitslice_inst_cfg3.cu", "bitslice_inst_cfg4.cu",
           "bitslice_inst_cfg5.cu", "bitslice_inst_cfg6.cu", "bitslice_inst_cfg8.cu", "bitslice_inst_pairs2.cu",
           "bitslice_inst_pairs4.cu", "bitslice_inst_pairs8.cu", "bitslice_inst_quads8.cu", "pair_rows.cu", "quad_rows.cu", "static_scratch.cu", "matched_filter.cu", "matched_filter_warp.cu", "peak_finding.cu", "rfi_mask.cu", "time_major.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--fmad=false", "-Xptxas", "-v"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    raise RuntimeError("nvcc not found")


def _headers() -> list[Path]:
    return sorted(CSRC.glob("*.h")) + sorted(CSRC.glob("*.cuh")) + [INCLUDE / "dedisp.h"]


def stale(lib: Path | None = None) -> bool:
    lib = lib or LIB
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    return any(d.stat().st_mtime > t for d in [CSRC / s for s in SOURCES] + _headers())


def _compile(src: Path, obj: Path, defs: list[str]) -> tuple[int, str]:
    tmp = obj.with_suffix(f".tmp{os.getpid()}.o")
    cmd = [_nvcc(), *NVCC_FLAGS, *[f"-D{d}" for d in defs], f"-I{INCLUDE}", f"-I{CSRC}", "-c", "-o", str(tmp), str(src)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode == 0:
        os.replace(tmp, obj)
    else:
        tmp.unlink(missing_ok=True)
    return r.returncode, r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False, defs: list[str] | None = None,
          out: Path | None = None, sources: list[str] | None = None) -> Path:
    """defs/out: tuning variants for A/B runs (e.g. defs=["BS_NW=20"], out=Path("x.so"))."""
    target = Path(out) if out else LIB
    defs = list(defs or [])
    sources = list(sources or SOURCES)
    if not force and not defs and not out and sources == SOURCES and not stale():
        return LIB
    objdir = OBJDIR
    objdir.mkdir(parents=True, exist_ok=True)
    hh = hashlib.sha1()
    for h in _headers():
        hh.update(h.name.encode() + b"\0" + h.read_bytes())
    hh.update(" ".join(NVCC_FLAGS + sorted(defs)).encode())
    common = hh.digest()
    objs, jobs = {}, []
    for s in sources:
        src = CSRC / s
        key = hashlib.sha1(common + src.read_bytes()).hexdigest()[:16]
        obj = objdir / f"{Path(s).stem}.{key}.o"
        objs[s] = obj
        if force or not obj.exists():
            jobs.append((src, obj))
    logs = []
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        for (src, obj), (rc, text) in zip(jobs, ex.map(lambda j: _compile(j[0], j[1], defs), jobs)):
            logs.append(f"==== {src.name}\n{text}")
            if verbose or rc != 0:
                sys.stderr.write(text)
            if rc != 0:
                obj.unlink(missing_ok=True)
                raise RuntimeError(f"nvcc failed compiling {src.name}")
    for src, obj in jobs:      # older objects of the same translation unit are of no use any more
        for old in objdir.glob(f"{src.stem}.*.o"):
            if old != obj and not force and old.stat().st_mtime < obj.stat().st_mtime - 6 * 3600:
                old.unlink(missing_ok=True)
    tmp = target.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", str(tmp)] + \
          [str(objs[s]) for s in sources]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError(f"nvcc failed linking {target.name}")
    logp = target.parent / (target.stem + "_ptxas.log")
    if jobs:
        old = logp.read_text() if logp.exists() and not force else ""
        keep = [blk for blk in old.split("==== ")[1:] if not any(blk.startswith(j[0].name) for j in jobs)]
        logp.write_text("".join("==== " + b for b in keep) + "".join(logs))
    os.replace(tmp, target)
    return target


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
