"""CPU oracle for the THOR+HELIOS RT step (arXiv 2203.02293) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2203_02293_b200 (the CUDA product path) and
must never be imported from it.

The arithmetic lives in helios_oracle.c (plain C, literal paper equations); this module only
compiles it with gcc and marshals numpy arrays through ctypes.

Two builds of the same source:
  real="ld"  -> long double  (truth for parity)
  real="f64" -> double       (timed CPU baseline)
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "helios_oracle.c"
_BUILD = _HERE / "build"

IMPROVED = 1
NONISOTHERMAL = 2
TOA_SPECTRUM = 4

_DEFAULTS = dict(eps2=2.0 / 3.0, e_tau=1e-4, gcrit_tol=1e-5, w0_transition=0.1, f_toa=0.0)


def build(force: bool = False) -> dict[str, Path]:
    """Compile both precisions of the oracle with gcc (-fopenmp; no fast-math)."""
    _BUILD.mkdir(exist_ok=True)
    out = {}
    for tag, real in (("ld", "long double"), ("f64", "double")):
        so = _BUILD / f"libhelios_oracle_{tag}.so"
        out[tag] = so
        if not force and so.exists() and so.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        tmp = so.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", f"-DORACLE_REAL={real}",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return out


_libs: dict[str, C.CDLL] = {}
_dp = C.POINTER(C.c_double)


class _Config(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "n_bins", "n_gauss", "n_ktab_p", "n_ktab_t")] + \
               [(n, _dp) for n in ("ktab_p", "ktab_t", "ktab", "bin_edges", "gauss_w", "scat_gas",
                                   "cloud_ext", "cloud_w0", "cloud_g0")] + \
               [(n, C.c_double) for n in ("cloud_p_top", "cloud_p_bot", "gravity", "cp", "eps2",
                                          "e_tau", "gcrit_tol", "w0_transition", "f_toa")] + \
               [("flags", C.c_uint32), ("n_iterations", C.c_int32)]


class _Inputs(C.Structure):
    _fields_ = [("n_columns", C.c_int32)] + [(n, _dp) for n in ("p", "T", "mu_star", "stellar_flux")] + \
               [("f_internal", C.c_double)]


class _Outputs(C.Structure):
    _fields_ = [(n, _dp) for n in ("F_up", "F_down", "F_net", "dTdt", "F_beam", "F_up_toa_bin")] + \
               [("dbg_column", C.c_int32), ("dbg_F_up_pt", _dp), ("dbg_F_dn_pt", _dp)]


def lib(real: str = "ld") -> C.CDLL:
    if real not in _libs:
        so = build()[real]
        L = C.CDLL(str(so))
        L.oracle_planck_G.restype = C.c_double
        L.oracle_planck_G.argtypes = [C.c_double]
        L.oracle_planck_bin_mean.restype = C.c_double
        L.oracle_planck_bin_mean.argtypes = [C.c_double] * 3
        L.oracle_kappa.restype = C.c_double
        L.oracle_kappa.argtypes = [C.c_int] * 4 + [_dp] * 3 + [C.c_double] * 2 + [C.c_int] * 2
        L.oracle_levels.restype = None
        L.oracle_levels.argtypes = [C.c_int, _dp, _dp, _dp, _dp]
        L.oracle_layer_coeffs.restype = None
        L.oracle_layer_coeffs.argtypes = [C.c_double] * 5 + [C.c_int] + [C.c_double] * 2 + [_dp]
        mono = [C.c_int] + [_dp] * 5 + [C.c_double] * 8 + [C.c_int] * 2
        L.oracle_column_mono.restype = None
        L.oracle_column_mono.argtypes = mono + [_dp] * 3
        L.oracle_column_mono_iter.restype = None
        L.oracle_column_mono_iter.argtypes = mono + [C.c_int] + [_dp] * 3
        L.oracle_assemble_blocks.restype = None
        L.oracle_assemble_blocks.argtypes = mono + [_dp] * 5
        L.oracle_rt_step.restype = C.c_int
        L.oracle_rt_step.argtypes = [C.POINTER(_Config), C.POINTER(_Inputs), C.POINTER(_Outputs)]
        L.oracle_level_optics.restype = None
        L.oracle_level_optics.argtypes = [C.POINTER(_Config), C.c_double, C.c_double, C.c_int, C.c_int, _dp]
        L.oracle_sizeof_real.restype = C.c_int
        _libs[real] = L
    return _libs[real]


def _a(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(a: np.ndarray | None):
    return a.ctypes.data_as(_dp) if a is not None else None


def planck_G(x: float, real: str = "ld") -> float:
    return lib(real).oracle_planck_G(float(x))


def planck_bin_mean(T: float, lam_lo: float, lam_hi: float, real: str = "ld") -> float:
    return lib(real).oracle_planck_bin_mean(float(T), float(lam_lo), float(lam_hi))


def kappa(ktab_p, ktab_t, ktab, p: float, T: float, b: int, g: int, real: str = "ld") -> float:
    ktab = _a(ktab)
    nP, nT, nb, ng = ktab.shape
    kp, ktt = _a(ktab_p), _a(ktab_t)
    return lib(real).oracle_kappa(nP, nT, nb, ng, _p(kp), _p(ktt), _p(ktab), float(p), float(T), int(b), int(g))


def levels(p, T, real: str = "ld"):
    p, T = _a(p), _a(T)
    N = p.shape[0]
    pi, ti = np.empty(N + 1), np.empty(N + 1)
    lib(real).oracle_levels(N, _p(p), _p(T), _p(pi), _p(ti))
    return pi, ti


_COEFF_NAMES = ("E", "zeta_p", "zeta_m", "trans", "chi", "xi", "psi", "Pi", "G_p", "G_m")


def layer_coeffs(w0, g0, dtau, mu, *, improved=True, real="ld", **opts) -> dict[str, float]:
    o = {**_DEFAULTS, **opts}
    out = np.empty(10)
    lib(real).oracle_layer_coeffs(float(w0), float(g0), float(dtau), float(mu), o["eps2"], int(improved),
                                  o["gcrit_tol"], o["w0_transition"], _p(out))
    return dict(zip(_COEFF_NAMES, out.tolist()))


def _mono_args(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, improved, linear_source, opts):
    o = {**_DEFAULTS, **opts}
    arrs = [_a(x) for x in (dtau, w0, g0, B_lo, B_hi)]
    L = arrs[0].shape[0]
    assert all(a.shape == (L,) for a in arrs)
    args = [L] + [_p(a) for a in arrs] + [float(mu), float(Fstar), float(F_boa), o["eps2"], o["e_tau"],
                                          o["gcrit_tol"], o["w0_transition"], o["f_toa"],
                                          int(improved), int(linear_source)]
    return L, arrs, args


def column_mono(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, *, improved=True, linear_source=False,
                real="ld", **opts):
    """One monochromatic column of L system layers (index 0 = bottom). Returns F_up, F_dn (diffuse),
    F_beam at the L+1 levels."""
    L, keep, args = _mono_args(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, improved, linear_source, opts)
    fu, fd, fb = np.empty(L + 1), np.empty(L + 1), np.empty(L + 1)
    lib(real).oracle_column_mono(*args, _p(fu), _p(fd), _p(fb))
    return fu, fd, fb


def column_mono_iter(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, n_iter, *, improved=True, linear_source=False,
                     real="ld", **opts):
    """The pair-wise iterative scheme Thomas replaces, n_iter iterations from zero fluxes."""
    L, keep, args = _mono_args(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, improved, linear_source, opts)
    fu, fd, fb = np.empty(L + 1), np.empty(L + 1), np.empty(L + 1)
    lib(real).oracle_column_mono_iter(*args, int(n_iter), _p(fu), _p(fd), _p(fb))
    return fu, fd, fb


def assemble_blocks(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, *, improved=True, linear_source=False,
                    real="ld", **opts):
    """The 2x2 blocks A, B, C [L+1,2,2], D [L+1,2] of Eq.(12) and F_beam [L+1]."""
    L, keep, args = _mono_args(dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, improved, linear_source, opts)
    n = L + 1
    A, B, Cm, D, fb = np.empty(4 * n), np.empty(4 * n), np.empty(4 * n), np.empty(2 * n), np.empty(n)
    lib(real).oracle_assemble_blocks(*args, _p(A), _p(B), _p(Cm), _p(D), _p(fb))
    return A.reshape(n, 2, 2), B.reshape(n, 2, 2), Cm.reshape(n, 2, 2), D.reshape(n, 2), fb


def level_optics(cfg: dict, p: float, T: float, b: int, g: int, real: str = "ld"):
    """(kappa_ext, omega0, g0) at one level for (bin b, Gauss point g): Eqs.(17)-(18) in per-mass units, the
    function the step itself calls.  cfg as for rt_step."""
    o = {**_DEFAULTS, **{k: cfg[k] for k in _DEFAULTS if k in cfg}}
    ktab = _a(cfg["ktab"])
    nP, nT, nb, ng = ktab.shape
    keep = {k: _a(cfg[k]) for k in ("ktab_p", "ktab_t", "bin_edges", "gauss_w", "scat_gas", "cloud_ext", "cloud_w0",
                                    "cloud_g0")}
    c = _Config(1, nb, ng, nP, nT, _p(keep["ktab_p"]), _p(keep["ktab_t"]), _p(ktab), _p(keep["bin_edges"]),
                _p(keep["gauss_w"]), _p(keep["scat_gas"]), _p(keep["cloud_ext"]), _p(keep["cloud_w0"]),
                _p(keep["cloud_g0"]), float(cfg["cloud_p_top"]), float(cfg["cloud_p_bot"]),
                float(cfg["gravity"]), float(cfg["cp"]), o["eps2"], o["e_tau"], o["gcrit_tol"],
                o["w0_transition"], o["f_toa"], int(cfg["flags"]), 0)
    out = np.empty(3)
    lib(real).oracle_level_optics(C.byref(c), float(p), float(T), int(b), int(g), _p(out))
    return tuple(out.tolist())


def rt_step(cfg: dict, inp: dict, *, real: str = "ld", threads: int | None = None,
            want=("F_up", "F_down", "F_net", "dTdt", "F_beam", "F_up_toa_bin"), dbg_column: int | None = None):
    """Full RT step on host arrays.

    cfg keys: ktab_p, ktab_t, ktab[nP,nT,nb,ng], bin_edges, gauss_w, scat_gas, cloud_ext, cloud_w0,
      cloud_g0, cloud_p_top, cloud_p_bot, gravity, cp, flags (+ optional eps2, e_tau, gcrit_tol,
      w0_transition, f_toa).
    inp keys: p[ncol,N], T[ncol,N], mu_star[ncol], stellar_flux[nb], f_internal.
    """
    o = {**_DEFAULTS, **{k: cfg[k] for k in _DEFAULTS if k in cfg}}
    ktab = _a(cfg["ktab"])
    nP, nT, nb, ng = ktab.shape
    p, T = _a(inp["p"]), _a(inp["T"])
    ncol, N = p.shape
    keep = dict(ktab=ktab, p=p, T=T)
    for k in ("ktab_p", "ktab_t", "bin_edges", "gauss_w", "scat_gas", "cloud_ext", "cloud_w0", "cloud_g0"):
        keep[k] = _a(cfg[k])
    keep["mu_star"] = _a(inp["mu_star"])
    keep["stellar_flux"] = _a(inp["stellar_flux"])
    assert keep["ktab_p"].shape == (nP,) and keep["ktab_t"].shape == (nT,)
    assert keep["bin_edges"].shape == (nb + 1,) and keep["gauss_w"].shape == (ng,)
    assert T.shape == (ncol, N) and keep["mu_star"].shape == (ncol,) and keep["stellar_flux"].shape == (nb,)
    c = _Config(N, nb, ng, nP, nT, _p(keep["ktab_p"]), _p(keep["ktab_t"]), _p(ktab), _p(keep["bin_edges"]),
                _p(keep["gauss_w"]), _p(keep["scat_gas"]), _p(keep["cloud_ext"]), _p(keep["cloud_w0"]),
                _p(keep["cloud_g0"]), float(cfg["cloud_p_top"]), float(cfg["cloud_p_bot"]),
                float(cfg["gravity"]), float(cfg["cp"]), o["eps2"], o["e_tau"], o["gcrit_tol"],
                o["w0_transition"], o["f_toa"], int(cfg["flags"]), int(cfg.get("n_iterations", 0)))
    i = _Inputs(ncol, _p(p), _p(T), _p(keep["mu_star"]), _p(keep["stellar_flux"]), float(inp["f_internal"]))
    shapes = dict(F_up=(ncol, N + 1), F_down=(ncol, N + 1), F_net=(ncol, N + 1), dTdt=(ncol, N),
                  F_beam=(ncol, N + 1), F_up_toa_bin=(ncol, nb))
    res = {k: np.zeros(shapes[k]) for k in want}
    dbg_u = dbg_d = None
    if dbg_column is not None:
        dbg_u, dbg_d = np.zeros((N + 1, nb * ng)), np.zeros((N + 1, nb * ng))
        res["dbg_F_up_pt"], res["dbg_F_dn_pt"] = dbg_u, dbg_d
    out = _Outputs(*[_p(res.get(k)) for k in ("F_up", "F_down", "F_net", "dTdt", "F_beam", "F_up_toa_bin")],
                   -1 if dbg_column is None else int(dbg_column), _p(dbg_u), _p(dbg_d))
    old = os.environ.get("OMP_NUM_THREADS")
    L = lib(real)
    if threads is not None:
        # libgomp honours omp_set_num_threads at run time
        gomp = C.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(int(threads))
    rc = L.oracle_rt_step(C.byref(c), C.byref(i), C.byref(out))
    if rc != 0:
        raise RuntimeError(f"oracle_rt_step failed: {rc}")
    del old
    return res


def max_threads() -> int:
    gomp = C.CDLL("libgomp.so.1")
    return int(gomp.omp_get_max_threads())
