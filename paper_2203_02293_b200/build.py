"""Build the CUDA C-ABI libraries in-tree for sm_100a:

    paper_2203_02293_b200/libhelios_rt.so            the product (include/helios_rt.h, helios_rt_debug.h)
    paper_2203_02293_b200/libhelios_rt_selftest.so   test / benchmark hooks only (include/helios_rt_selftest.h)

Every csrc/*.cu is compiled to an object (cached by mtime under csrc/build/).  nvcc cross-compiles without a GPU.
`python -m paper_2203_02293_b200.build [--force] [--verbose]`.
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
INC = ROOT / "include"
LIB = PKG / "libhelios_rt.so"
LIB_SELFTEST = PKG / "libhelios_rt_selftest.so"
LIBS = {LIB: ("helios_rt", "helios_rt_k_iso", "helios_rt_k_toa", "helios_rt_k_noniso", "helios_rt_k_sampling", "helios_post"),
        LIB_SELFTEST: ("helios_rt_selftest",)}

# -split-compile 1 (no parallel split of a translation unit): with any larger value -- and with 0, "as many as there are
# host threads" -- nvcc's code for the kernels differs from one build of the SAME source to the next (measured: three
# builds in a row, two different binaries, 3 % apart in step time).  Parallelism comes from compiling
# the translation units side by side instead.
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-split-compile", "1"]


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
    deps = [*INC.glob("*.h"), *CSRC.glob("*.cuh"), *CSRC.glob("*.inc")]
    dep_time = max(d.stat().st_mtime for d in deps)
    OBJ.mkdir(exist_ok=True)
    todo, objs = [], {}
    for src in sources:
        obj = OBJ / (src.stem + ".o")
        objs[src.stem] = obj
        if force or not obj.exists() or obj.stat().st_mtime < max(src.stat().st_mtime, dep_time):
            todo.append((src, obj))

    def compile_one(job):
        src, obj = job
        tmp = obj.with_suffix(f".tmp{os.getpid()}.o")
        _run([nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", "-o", str(tmp), str(src)], verbose)
        os.replace(tmp, obj)

    with ThreadPoolExecutor(max_workers=6) as ex:
        list(ex.map(compile_one, todo))
    for lib, stems in LIBS.items():
        members = [objs[s] for s in stems]
        if lib.exists() and all(lib.stat().st_mtime >= o.stat().st_mtime for o in members):
            continue
        tmp = lib.with_suffix(f".tmp{os.getpid()}.so")
        _run([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, members)], verbose)
        os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
