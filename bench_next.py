"""Measurements of the NEXT rows on one B200: `python bench_next.py
[--what postproc|onedim|iterative|all] [--steps K]`.  One JSON line per row; CUDA-event times on the launching
stream after warm-up, inputs resident on the device, L2 flushed between timed repetitions.

  postproc   config 6: helios_rt_extend_top -> helios_rt_step (R=500 opacity sampling, 3255 wavelengths, 60 layers,
             TOA spectrum) -> helios_rt_phase_curve (64 phases + HST-WFC3 band), Eqs. 23-26
  onedim     Sec. 3 "1-D mode": (helios_rt_step -> helios_rt_advance_1d) per time step, plain launches and one
             CUDA graph of the pair replayed; 4 zenith angles (config-1 sized columns) and the config-2 grid; then the
             four zenith angles run to radiative equilibrium (12000 / 36000 replays), residuals reported
  iterative  helios_rt_step_iterative (the scheme Thomas replaces, L258-270) against helios_rt_step on config 2:
             the paper's "about 2 orders of magnitude" (L13, L397) re-measured on B200
"""
from __future__ import annotations

import argparse
import json
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

L2_FLUSH_BYTES = 256 << 20


def _peaks() -> dict:
    f = ROOT / "MEASURED_PEAKS.json"
    return json.loads(f.read_text()) if f.exists() else {}


def _timed(torch, fn, steps, flush, stream):
    for _ in range(3):
        flush.fill_(1.0)
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    torch.cuda.synchronize()
    for a, b in ev:
        flush.fill_(1.0)
        a.record(stream)
        fn()
        b.record(stream)
    torch.cuda.synchronize()
    t = np.array([a.elapsed_time(b) for a, b in ev])
    return float(t.mean()), float(t.min())


def _postproc_cpu_baseline(cfg, inp, meta, n_cols: int = 12) -> dict:
    """The oracle (as it stands, double build) on a bounded sample of config 6: the RT step of `n_cols` evenly strided
    extended columns, then the phase curve of the whole grid from a synthetic spectrum of the right shape -- scaled to one
    pipeline pass.  A stated baseline, not a target."""
    import time
    import oracle
    from oracle import postproc
    n, N, ne = meta["n_columns"], meta["n_model_layers"], meta["n_extra"]
    idx = np.linspace(0, n - 1, n_cols).astype(int)
    p_ext, T_ext = postproc.extend_top(inp["p"][idx], inp["T"][idx], ne, meta["p_min"])
    sub = dict(inp, p=p_ext, T=T_ext, mu_star=inp["mu_star"][idx])
    t0 = time.perf_counter()
    ref = oracle.rt_step(cfg, sub, real="f64", want=("F_up_toa_bin",))
    t_step = (time.perf_counter() - t0) * n / n_cols
    F = np.tile(ref["F_up_toa_bin"], (n // n_cols + 1, 1))[:n]
    t0 = time.perf_counter()
    postproc.phase_curve(F, meta["lon"], meta["lat"], meta["area"], meta["alpha"], cfg["bin_edges"], *meta["band"])
    t_pc = time.perf_counter() - t0
    return {"value": (t_step + t_pc) * 1e3, "unit": "ms", "cores": oracle.max_threads(), "kind": "oracle",
            "sample": f"RT step of {n_cols} evenly strided extended columns scaled to {n}, + the phase curve of the whole grid",
            "rt_step_s": t_step, "phase_curve_s": t_pc}


def bench_postproc(torch, H, W, steps, cpu_baseline: bool = True):
    cfg, inp, meta = W.make(6)
    dev = torch.device("cuda", 0)
    t = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    n, N, ne, nb = meta["n_columns"], meta["n_model_layers"], meta["n_extra"], meta["n_bins"]
    na = meta["alpha"].size
    rt = H.HeliosRT(cfg, n)
    d = dict(p=t(inp["p"]), T=t(inp["T"]), mu=t(inp["mu_star"]), fs=t(inp["stellar_flux"]), lon=t(meta["lon"]),
             lat=t(meta["lat"]), area=t(meta["area"]), alpha=t(meta["alpha"]), edges=t(cfg["bin_edges"]))
    pe = torch.empty((n, N + ne), dtype=torch.float64, device=dev)
    Te = torch.empty_like(pe)
    spec = torch.empty((n, nb), dtype=torch.float64, device=dev)
    ph = torch.empty((na, nb), dtype=torch.float64, device=dev)
    band = torch.empty((na,), dtype=torch.float64, device=dev)
    pc_ws = H.phase_curve_workspace(n, nb, na, dev)
    flush = torch.empty(L2_FLUSH_BYTES // 8, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream()
    f_ext = lambda: H.extend_top(d["p"], d["T"], ne, meta["p_min"], pe, Te)
    f_step = lambda: rt.step(pe, Te, d["mu"], d["fs"], inp["f_internal"], {"F_up_toa_bin": spec})
    f_pc = lambda: H.phase_curve(spec, d["lon"], d["lat"], d["area"], d["alpha"], ph, bin_edges=d["edges"],
                                 lam1=meta["band"][0], lam2=meta["band"][1], F_phase_band=band, workspace=pc_ws)

    def pipeline():
        f_ext(); f_step(); f_pc()
    ms_all, ms_all_min = _timed(torch, pipeline, steps, flush, st)
    f_ext(); f_step()
    ms_ext, _ = _timed(torch, f_ext, steps, flush, st)
    ms_step, _ = _timed(torch, f_step, steps, flush, st)
    ms_pc, _ = _timed(torch, f_pc, steps, flush, st)
    peaks = _peaks()
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    pc_bytes = 8.0 * (n * nb + na * nb + 3 * n + na)       # F read once, phase spectra written once
    pc_flops = 2.0 * n * nb * na                           # one FMA per (column, bin, phase)
    solves = n * nb
    # fp64-ALU roofline of the opacity-sampling RT step: the locked TOA-mode slots of bench.py (138 day / 90 night per
    # layer.point) over the extended columns
    from bench import FP64_LANES_PER_SM, algorithmic_slots
    info = rt.launch_info()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    slots = algorithmic_slots(meta, cfg["flags"], inp["mu_star"])
    peak = info["sm_count"] * FP64_LANES_PER_SM * sm_max * 1e6
    rt_roofline = {"bound": "alu", "achieved": slots / (ms_step * 1e-3) * 1e-12, "peak": peak * 1e-12, "unit": "Tslot/s",
                   "frac": slots / (ms_step * 1e-3) / peak, "algorithmic_slots_per_step": slots,
                   "t_alu_ms": slots / peak * 1e3, "kernel_ms": ms_step,
                   "kernel": "rt_step_kernel<NONISO=0, TOA=1, BDIRECT=1> (one point per bin)",
                   "slot_lock": "BASELINE.md section 3 (TOA mode: 138 day / 90 night slots per layer.point)"}
    line = {"row": "NEXT-2 post-processing", "metric": "postproc_pipeline_ms", "value": ms_all, "unit": "ms",
            "higher_is_better": False, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config6 {meta['name']}: {n} columns x {N}+{ne} layers x {nb} wavelengths x 1, "
                                   f"TOA spectrum, {na} phases, band {meta['band'][0]*1e6:.1f}-{meta['band'][1]*1e6:.1f} um",
                       "launch": rt.launch_info()},
            "stages_ms": {"extend_top": ms_ext, "rt_step": ms_step, "phase_curve": ms_pc, "pipeline_min": ms_all_min},
            "rt_step_solves_per_s": solves / (ms_step * 1e-3),
            "roofline": rt_roofline,
            "cpu_baseline": _postproc_cpu_baseline(cfg, inp, meta) if cpu_baseline else None,
            "phase_curve": {"bound": "hbm", "algorithmic_bytes": pc_bytes, "achieved_gbs": pc_bytes / (ms_pc * 1e-3) * 1e-9,
                            "peak_gbs": hbm, "frac": pc_bytes / (ms_pc * 1e-3) * 1e-9 / hbm,
                            "fp64_gflops": pc_flops / (ms_pc * 1e-3) * 1e-9,
                            "note": "3 launches (phase_partial_kernel, phase_reduce_kernel, phase_band_kernel); F is read once "
                                    "per 32 phases; cold L2"},
            "gpu_launches": steps * 5}
    rt.close()
    return line


def bench_onedim(torch, H, W, steps):
    dev = torch.device("cuda", 0)
    t = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    out = []
    # dt: the paper's 300 s (L384) for the config-1 columns (top at 1e-4 bar); 10 s on the config-2 grid, whose 1e-6 bar
    # top layers (2e-3 kg m^-2) would overshoot with an explicit 300 s step
    for label, config, cols, dt in (("4 zenith angles (0/30/60/89 deg), config-1 column shape", 1, slice(0, 4), 300.0),
                                    ("config-2 grid, 2562 columns", 2, None, 10.0)):
        cfg, inp, meta = W.make(config, columns=cols)
        n, N = meta["n_columns"], meta["n_layers"]
        mu = inp["mu_star"] if config == 2 else np.cos(np.radians([0.0, 30.0, 60.0, 89.0]))
        g, R = cfg["gravity"], 3553.0
        z = (R * inp["T"].mean() / g) * np.log(inp["p"][0, 0] / inp["p"][0])
        pref = float(inp["p"][0, 0])
        rt = H.HeliosRT(cfg, n)
        dT, dz, dmu, dfs = t(inp["T"]), t(z), t(mu), t(inp["stellar_flux"])
        dp = torch.empty((n, N), dtype=torch.float64, device=dev)
        dh = torch.empty((n, N), dtype=torch.float64, device=dev)
        s = torch.cuda.Stream()
        K = max(steps, 20)
        with torch.cuda.stream(s):
            H.advance_1d(0.0, g, R, pref, dz, None, dT, dp, None, stream=s)

            def pair():
                rt.step(dp, dT, dmu, dfs, inp["f_internal"], {"dTdt": dh}, stream=s)
                H.advance_1d(dt, g, R, pref, dz, dh, dT, dp, None, stream=s)
            for _ in range(5):
                pair()
            s.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(s)
            for _ in range(K):
                pair()
            b.record(s)
            s.synchronize()
            ms_plain = a.elapsed_time(b) / K
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr, stream=s):
                pair()
            for _ in range(5):
                gr.replay()
            s.synchronize()
            a.record(s)
            for _ in range(K):
                gr.replay()
            b.record(s)
            s.synchronize()
            ms_graph = a.elapsed_time(b) / K
        finite = bool(torch.isfinite(dT).all().item())
        out.append({"row": "NEXT-3 1-D mode", "metric": "one_d_time_step_ms", "value": ms_graph, "unit": "ms",
                    "higher_is_better": False, "dtype": "f64", "data": "synthetic",
                    "config": {"workload": f"{label}: {n} columns x {N} layers x {meta['n_bins']}x{meta['n_gauss']}, "
                                           f"dt = {dt:.0f} s, RT step + T update + Eq. 20 per time step, warm L2"},
                    "plain_launch_ms": ms_plain, "cuda_graph_ms": ms_graph, "time_steps_timed": K, "state_finite": finite,
                    "launches_per_time_step": 3, "gpu_launches": 3 * K * 2})
        rt.close()
    return out


def bench_steady_state(torch, H, W):
    """NEXT-3: the Sec. 3 experiment -- the four zenith angles run to radiative equilibrium by replaying one captured time
    step (RT step + T update + Eq. 20); residuals at the end and time steps per second."""
    import time
    dev = torch.device("cuda", 0)
    t = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    out = []
    for zenith, cp, K in (((0.0, 30.0, 60.0), 2000.0, 12000), ((89.0,), 500.0, 36000)):
        cfg, inp, meta, ex = W.make_one_d(zenith, cp)
        n, N = inp["T"].shape
        g = cfg["gravity"]
        rt = H.HeliosRT(cfg, n)
        dT, dz, dmu, dfs = t(inp["T"]), t(ex["z"]), t(inp["mu_star"]), t(inp["stellar_flux"])
        dp = torch.empty((n, N), dtype=torch.float64, device=dev)
        dh = torch.empty((n, N), dtype=torch.float64, device=dev)
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            H.advance_1d(0.0, g, ex["R_d"], ex["p_ref"], dz, None, dT, dp, None, stream=s)

            def pair():
                rt.step(dp, dT, dmu, dfs, inp["f_internal"], {"dTdt": dh}, stream=s)
                H.advance_1d(ex["dt"], g, ex["R_d"], ex["p_ref"], dz, dh, dT, dp, None, stream=s)
            pair()
            s.synchronize()
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr, stream=s):
                pair()
            t0 = time.perf_counter()
            for _ in range(K - 1):
                gr.replay()
            s.synchronize()
            wall = time.perf_counter() - t0
            res = {k: torch.empty((n, N + 1) if k != "dTdt" else (n, N), dtype=torch.float64, device=dev) for k in ("F_net", "dTdt")}
            rt.step(dp, dT, dmu, dfs, inp["f_internal"], res, stream=s)
        torch.cuda.synchronize()
        F_net, dTdt = res["F_net"].cpu().numpy(), res["dTdt"].cpu().numpy()
        absorbed = inp["mu_star"] * meta["F_star_tot"]
        out.append({"row": "NEXT-3 steady state", "metric": "one_d_time_steps_per_s", "value": (K - 1) / wall, "unit": "steps/s",
                    "higher_is_better": True, "dtype": "f64", "data": "synthetic",
                    "config": {"workload": f"1-D mode, zenith angles {list(zenith)} deg, config-1 column shape, c_P = {cp:.0f} "
                                           f"(pseudo-time acceleration), dt = {ex['dt']:.0f} s, {K} time steps replayed from one "
                                           "CUDA graph"},
                    "max_abs_dTdt_times_dt_K": float(np.abs(dTdt).max() * ex["dt"]),
                    "max_F_net_spread_over_absorbed": float(np.max(np.abs(F_net - F_net[:, :1]) / absorbed[:, None])),
                    "F_net_boa": [float(x) for x in F_net[:, 0]], "T_range_K": [float(dT.min()), float(dT.max())],
                    "gpu_launches": 2 * K})
        rt.close()
    return out


def bench_iterative(torch, H, W, steps):
    dev = torch.device("cuda", 0)
    t = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    cfg, inp, meta = W.make(2)
    n = meta["n_columns"]
    rt = H.HeliosRT(cfg, n)
    shapes = rt.output_shapes(n)
    names = ("F_up", "F_down", "F_net", "dTdt")
    o1 = {k: torch.empty(shapes[k], dtype=torch.float64, device=dev) for k in names}
    o2 = {k: torch.empty(shapes[k], dtype=torch.float64, device=dev) for k in names}
    args = (t(inp["p"]), t(inp["T"]), t(inp["mu_star"]), t(inp["stellar_flux"]), inp["f_internal"])
    flush = torch.empty(L2_FLUSH_BYTES // 8, dtype=torch.float64, device=dev)
    st = torch.cuda.current_stream()
    ms_thomas, _ = _timed(torch, lambda: rt.step(*args, o1), steps, flush, st)
    res = {}
    for nit in (10, 200):
        k = max(3, steps // (1 if nit == 10 else 5))
        ms, _ = _timed(torch, lambda: rt.step_iterative(*args, o2, nit), k, flush, st)
        err = float(((o2["F_net"] - o1["F_net"]).abs() / (o1["F_net"].abs() + 1e-12 * meta["F_star_tot"])).max().item())
        res[str(nit)] = {"ms": ms, "slowdown_vs_thomas": ms / ms_thomas, "max_rel_diff_F_net_vs_thomas": err}
    rt.close()
    return {"row": "NEXT-4 iterative scheme", "metric": "iterative_over_thomas_time_ratio", "value": res["200"]["slowdown_vs_thomas"],
            "unit": "x", "higher_is_better": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config2 {meta['name']}: {n} columns x 40 layers x 30x20; N = 200 iterations (HELIOS, L270) "
                                   f"and N = 10 (Oreshenko et al., L270)"},
            "thomas_ms": ms_thomas, "iterative": res,
            "paper": "about 2 orders of magnitude (L13, L397); 'a factor of roughly N' (L397)",
            "gpu_launches": steps * 2 + (steps + max(3, steps // 5)) * 2}


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--what", default="all", choices=("postproc", "onedim", "iterative", "all"))
    ap.add_argument("--steps", type=int, default=20)
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench_next: no CUDA device -- the product path has no CPU fallback")
    from paper_2203_02293_b200 import build, helios_rt as H, workloads as W
    build.build()
    torch.cuda.set_device(0)
    if args.what in ("postproc", "all"):
        print(json.dumps(bench_postproc(torch, H, W, args.steps)), flush=True)
    if args.what in ("onedim", "all"):
        for line in bench_onedim(torch, H, W, args.steps):
            print(json.dumps(line), flush=True)
        for line in bench_steady_state(torch, H, W):
            print(json.dumps(line), flush=True)
    if args.what in ("iterative", "all"):
        print(json.dumps(bench_iterative(torch, H, W, args.steps)), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
