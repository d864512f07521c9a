"""Build the CUDA C-ABI library in-tree (paper_2203_02293_b200/libhelios_rt.so) for sm_100a.

Every csrc/*.cu is compiled to an object (cached by mtime under csrc/build/) and linked into one shared
library.  nvcc cross-compiles without a GPU.  `python -m paper_2203_02293_b200.build [--force] [--verbose]`.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
OBJ = CSRC / "build"
HDR = ROOT / "include" / "helios_rt.h"
LIB = PKG / "libhelios_rt.so"

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return "nvcc"


def _run(cmd, verbose):
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed ({res.returncode}): {' '.join(cmd)}")


def build(force: bool = False, verbose: bool = False) -> Path:
    sources = sorted(CSRC.glob("*.cu"))
    deps = [HDR, *CSRC.glob("*.cuh")]
    dep_time = max(d.stat().st_mtime for d in deps)
    OBJ.mkdir(exist_ok=True)
    todo, objs = [], []
    for src in sources:
        obj = OBJ / (src.stem + ".o")
        objs.append(obj)
        if force or not obj.exists() or obj.stat().st_mtime < max(src.stat().st_mtime, dep_time):
            todo.append((src, obj))
    if not todo and LIB.exists() and all(LIB.stat().st_mtime >= o.stat().st_mtime for o in objs):
        return LIB
    def compile_one(job):
        src, obj = job
        tmp = obj.with_suffix(f".tmp{os.getpid()}.o")
        _run([nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", "-o", str(tmp), str(src)], verbose)
        os.replace(tmp, obj)
    with ThreadPoolExecutor(max_workers=4) as ex:
        list(ex.map(compile_one, todo))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    _run([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, objs)], verbose)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
