"""Audit of the oracle's floating-point operation mix per layer.point ("the
definitive count comes from running the oracle with an op-counting scalar type").

    python -m oracle.opcount            # one JSON line per (config, dayside / nightside)

helios_oracle.c is compiled UNCHANGED as C++ with ORACLE_REAL = Counted (opcount.hpp: a long double that counts every
+ - * / comparison, sqrt, exp and log it takes part in) and run on four dayside and four nightside columns of configs 2
and 3.  Test infrastructure like the rest of oracle/: nothing here is used by the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import json
import os
import subprocess
import sys
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
if str(_HERE.parent) not in sys.path:
    sys.path.insert(0, str(_HERE.parent))

import oracle  # noqa: E402


def build() -> Path:
    out = _HERE / "build"
    out.mkdir(exist_ok=True)
    so = out / "libhelios_oracle_opcount.so"
    src = _HERE / "helios_oracle.c"
    if so.exists() and so.stat().st_mtime >= max(src.stat().st_mtime, (_HERE / "opcount.hpp").stat().st_mtime):
        return so
    body = out / "opcount_body.c"
    body.write_text(src.read_text().replace("#include <tgmath.h>", ""))      # math calls resolve to opcount.hpp's overloads
    wrap = out / "opcount_wrap.cpp"
    wrap.write_text('#include "../opcount.hpp"\nthread_local OpCounts g_ops;\nextern "C" {\n#include "opcount_body.c"\n}\n'
                    'extern "C" void opc_reset(void) { g_ops = OpCounts(); }\n'
                    'extern "C" void opc_get(long long *o) { o[0] = g_ops.add; o[1] = g_ops.mul; o[2] = g_ops.div; '
                    'o[3] = g_ops.sqrt_; o[4] = g_ops.exp_; o[5] = g_ops.log_; o[6] = g_ops.cmp; }\n')
    tmp = so.with_suffix(f".tmp{os.getpid()}.so")
    subprocess.run(["g++", "-std=c++17", "-fpermissive", "-w", "-O1", "-shared", "-fPIC", "-DORACLE_REAL=Counted",
                    "-o", str(tmp), str(wrap)], check=True)
    os.replace(tmp, so)
    return so


NAMES = ("add_sub", "mul", "div", "sqrt", "exp", "log", "compare")


def count(config: int, dayside: bool, n_cols: int = 4) -> dict:
    from paper_2203_02293_b200 import workloads as W
    L = C.CDLL(str(build()))
    L.oracle_rt_step.restype = C.c_int
    L.oracle_rt_step.argtypes = [C.POINTER(oracle._Config), C.POINTER(oracle._Inputs), C.POINTER(oracle._Outputs)]
    oracle._libs["opcount"] = L
    cfg, inp, meta = W.make(config)
    mu = inp["mu_star"]
    idx = np.flatnonzero((mu > 0) == dayside)[:n_cols]
    sub = dict(inp, p=inp["p"][idx], T=inp["T"][idx], mu_star=mu[idx])
    L.opc_reset()
    oracle.rt_step(cfg, sub, real="opcount", want=("F_net",))
    o = (C.c_longlong * 7)()
    L.opc_get(o)
    per = np.array(list(o), dtype=float) / (len(idx) * meta["n_layers"] * meta["n_bins"] * meta["n_gauss"])
    return dict(zip(NAMES, (round(float(x), 1) for x in per)))


if __name__ == "__main__":
    for config in (2, 3):
        for day in (True, False):
            print(json.dumps({"config": config, "side": "day" if day else "night", "per_layer_point": count(config, day)}))
