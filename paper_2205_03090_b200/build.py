"""Build libptflash.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

One translation unit per component count (ptflash_nc.cu with -DPTF_NC=k) so the 15 kernel variants compile in
parallel; objects land in csrc/build/, the shared library next to this file.  Usage:
    python -m paper_2205_03090_b200.build [--force] [--nc 2,8,10]
"""
from __future__ import annotations

import argparse
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = CSRC / "build"
LIB = HERE / "libptflash.so"
ALL_NC = list(range(2, 17))
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "--std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (Path(c).exists() or c == "nvcc"):
            return c
    raise RuntimeError("nvcc not found")


def _newest_src() -> float:
    return max(p.stat().st_mtime for p in list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h"))
               + [HERE.parent / "include" / "ptflash.h"])


def _compile(src: Path, obj: Path, extra: list) -> str:
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-c", str(src), "-o", str(obj)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
    (obj.with_suffix(".ptxas.txt")).write_text(r.stderr)
    return r.stderr


def build(force: bool = False, ncs=None, verbose: bool = False) -> Path:
    ncs = list(ncs or ALL_NC)
    stamp = OBJ / "stamp.txt"
    want = ",".join(map(str, ncs))
    if (not force and LIB.exists() and stamp.exists() and stamp.read_text() == want
            and LIB.stat().st_mtime >= _newest_src()):
        return LIB
    OBJ.mkdir(parents=True, exist_ok=True)
    jobs = [(CSRC / "ptflash_api.cu", OBJ / "api.o", []), (CSRC / "ptflash_peak.cu", OBJ / "peak.o", [])]
    for k in ALL_NC:
        # variants left out of a partial (development) build fall back to a stub that reports "not built"
        extra = [f"-DPTF_NC={k}"] + ([] if k in ncs else ["-DPTF_STUB"])
        jobs.append((CSRC / "ptflash_nc.cu", OBJ / f"nc{k}.o", extra))
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        outs = list(ex.map(lambda j: _compile(*j), jobs))
    if verbose:
        for (src, obj, extra), o in zip(jobs, outs):
            print(obj.name, "\n".join(l for l in o.splitlines() if "registers" in l or "spill" in l))
    objs = [str(j[1]) for j in jobs]
    cmd = [_nvcc(), "-shared", "-o", str(LIB), *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed: {r.stdout}\n{r.stderr}")
    stamp.write_text(want)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--nc", default="")
    ap.add_argument("-v", "--verbose", action="store_true")
    a = ap.parse_args()
    print(build(a.force, [int(x) for x in a.nc.split(",")] if a.nc else None, a.verbose))
