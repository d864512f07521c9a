"""Thin ctypes binding of include/helios_rt.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libhelios_rt.so.  There is no CPU fallback: if
the library is missing or no sm_100 device is present, construction raises.
PyTorch is used only for device memory and streams.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from .workloads import IMPROVED, NONISOTHERMAL, TOA_SPECTRUM  # noqa: F401

_LIB_PATH = Path(__file__).resolve().parent / "libhelios_rt.so"
_SELFTEST_PATH = Path(__file__).resolve().parent / "libhelios_rt_selftest.so"   # test / benchmark hooks, not the product
_dp = C.POINTER(C.c_double)

# symbols declared in include/helios_rt.h + include/helios_rt_debug.h (libhelios_rt.so) ...
EXPORTS = ("helios_rt_create", "helios_rt_step", "helios_rt_step_host", "helios_rt_destroy",
           "helios_rt_strerror", "helios_rt_last_cuda_error", "helios_rt_launch_info", "helios_rt_step_iterative",
           "helios_rt_extend_top", "helios_rt_phase_curve", "helios_rt_phase_curve_workspace_bytes",
           "helios_rt_phase_curve_noalloc",
           "helios_rt_advance_1d", "helios_rt_debug_set_launch", "helios_rt_debug_get_launch",
           "helios_rt_debug_force_two_launches", "helios_rt_debug_set_workers", "helios_rt_debug_force_stuck")
# ... and in include/helios_rt_selftest.h (libhelios_rt_selftest.so)
SELFTEST_EXPORTS = ("helios_rt_selftest_math", "helios_rt_selftest_planck", "helios_rt_selftest_planck_G",
                    "helios_rt_measure_dfma_peak", "helios_rt_measure_latencies")


class Config(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "n_bins", "n_gauss", "n_ktab_p", "n_ktab_t", "max_columns")] + \
               [(n, _dp) for n in ("ktab_p", "ktab_t", "ktab", "bin_edges", "gauss_w", "scat_gas", "cloud_ext",
                                   "cloud_w0", "cloud_g0")] + \
               [(n, C.c_double) for n in ("cloud_p_top", "cloud_p_bot", "gravity", "cp", "eps2", "e_tau",
                                          "gcrit_tol", "w0_transition", "f_toa")] + \
               [("flags", C.c_uint32)]


class Inputs(C.Structure):
    _fields_ = [("n_columns", C.c_int32)] + [(n, C.c_void_p) for n in ("p", "T", "mu_star", "stellar_flux")] + \
               [("f_internal", C.c_double)]


class Outputs(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("F_up", "F_down", "F_net", "dTdt", "F_beam", "F_up_toa_bin")]


OUTPUT_NAMES = tuple(n for n, _ in Outputs._fields_)
_lib = None
_selftest = None


class HeliosRTError(RuntimeError):
    pass


def load_library() -> C.CDLL:
    """dlopen the in-tree CUDA library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise HeliosRTError(f"{_LIB_PATH} is missing: run `python -m paper_2203_02293_b200.build` "
                                "(there is no CPU fallback)")
        L = C.CDLL(str(_LIB_PATH))
        L.helios_rt_create.restype = C.c_int
        L.helios_rt_create.argtypes = [C.POINTER(Config), C.POINTER(C.c_void_p)]
        L.helios_rt_step.restype = C.c_int
        L.helios_rt_step.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Outputs), C.c_void_p]
        L.helios_rt_step_host.restype = C.c_int
        L.helios_rt_step_host.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Outputs)]
        L.helios_rt_destroy.restype = C.c_int
        L.helios_rt_destroy.argtypes = [C.c_void_p]
        L.helios_rt_strerror.restype = C.c_char_p
        L.helios_rt_strerror.argtypes = [C.c_int]
        L.helios_rt_last_cuda_error.restype = C.c_char_p
        L.helios_rt_last_cuda_error.argtypes = [C.c_void_p]
        L.helios_rt_launch_info.restype = C.c_int
        L.helios_rt_launch_info.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.helios_rt_step_iterative.restype = C.c_int
        L.helios_rt_step_iterative.argtypes = [C.c_void_p, C.POINTER(Inputs), C.POINTER(Outputs), C.c_int32, C.c_void_p]
        L.helios_rt_extend_top.restype = C.c_int
        L.helios_rt_extend_top.argtypes = [C.c_int32] * 3 + [C.c_double] + [C.c_void_p] * 5
        L.helios_rt_phase_curve.restype = C.c_int
        L.helios_rt_phase_curve.argtypes = [C.c_int32] * 3 + [C.c_void_p] * 6 + [C.c_double] * 2 + [C.c_void_p] * 4
        L.helios_rt_phase_curve_noalloc.restype = C.c_int
        L.helios_rt_phase_curve_noalloc.argtypes = [C.c_int32] * 3 + [C.c_void_p] * 6 + [C.c_double] * 2 + [C.c_void_p] * 3
        L.helios_rt_phase_curve_workspace_bytes.restype = C.c_int64
        L.helios_rt_phase_curve_workspace_bytes.argtypes = [C.c_int32] * 3
        L.helios_rt_advance_1d.restype = C.c_int
        L.helios_rt_advance_1d.argtypes = [C.c_int32] * 2 + [C.c_double] * 4 + [C.c_void_p] * 6
        L.helios_rt_debug_force_two_launches.restype = C.c_int
        L.helios_rt_debug_force_two_launches.argtypes = [C.c_void_p, C.c_int32]
        L.helios_rt_debug_force_stuck.restype = C.c_int
        L.helios_rt_debug_force_stuck.argtypes = [C.c_void_p, C.c_int32]
        L.helios_rt_debug_set_workers.restype = C.c_int
        L.helios_rt_debug_set_workers.argtypes = [C.c_void_p, C.c_int32]
        L.helios_rt_debug_set_launch.restype = C.c_int
        L.helios_rt_debug_set_launch.argtypes = [C.c_void_p] + [C.c_int32] * 5
        L.helios_rt_debug_get_launch.restype = C.c_int
        L.helios_rt_debug_get_launch.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        _lib = L
    return _lib


def load_selftest_library() -> C.CDLL:
    """dlopen the test / benchmark hooks (include/helios_rt_selftest.h)."""
    global _selftest
    if _selftest is None:
        if not _SELFTEST_PATH.exists():
            raise HeliosRTError(f"{_SELFTEST_PATH} is missing: run `python -m paper_2203_02293_b200.build`")
        L = C.CDLL(str(_SELFTEST_PATH))
        L.helios_rt_selftest_math.restype = C.c_int
        L.helios_rt_selftest_math.argtypes = [C.c_int32] + [_dp] * 5
        L.helios_rt_selftest_planck.restype = C.c_int
        L.helios_rt_selftest_planck.argtypes = [C.c_int32] + [_dp] * 4
        L.helios_rt_selftest_planck_G.restype = C.c_int
        L.helios_rt_selftest_planck_G.argtypes = [C.c_int32] + [_dp] * 2
        L.helios_rt_measure_dfma_peak.restype = C.c_int
        L.helios_rt_measure_dfma_peak.argtypes = [C.c_int32, _dp, _dp]
        L.helios_rt_measure_latencies.restype = C.c_int
        L.helios_rt_measure_latencies.argtypes = [_dp]
        _selftest = L
    return _selftest


def _check(rc: int, handle=None):
    if rc != 0:
        L = load_library()
        msg = L.helios_rt_strerror(rc).decode()
        if handle:
            extra = L.helios_rt_last_cuda_error(handle).decode()
            if extra:
                msg += f": {extra}"
        raise HeliosRTError(f"helios_rt error {rc}: {msg}")


def _np(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_dp)


class HeliosRT:
    """Handle around helios_rt_create / helios_rt_step / helios_rt_destroy.

    cfg: dict of host arrays/scalars with the field names of helios_rt_config (see workloads.make);
    n_layers is taken from cfg["n_layers"] or passed explicitly.
    """

    def __init__(self, cfg: dict, max_columns: int, n_layers: int | None = None):
        L = load_library()
        ktab = _np(cfg["ktab"])
        if ktab.ndim != 4:
            raise HeliosRTError("helios_rt error -1: ktab must be [nP, nT, n_bins, n_gauss]")
        nP, nT, nb, ng = ktab.shape
        keep = {k: _np(cfg[k]) for k in ("ktab_p", "ktab_t", "bin_edges", "gauss_w", "scat_gas", "cloud_ext",
                                         "cloud_w0", "cloud_g0")}
        if keep["ktab_p"].shape != (nP,) or keep["ktab_t"].shape != (nT,) or keep["bin_edges"].shape != (nb + 1,) \
                or keep["gauss_w"].shape != (ng,) or any(keep[k].shape != (nb,) for k in
                                                         ("scat_gas", "cloud_ext", "cloud_w0", "cloud_g0")):
            raise HeliosRTError("helios_rt error -1: array shapes inconsistent with ktab[nP,nT,n_bins,n_gauss]")
        self.n_layers = int(n_layers if n_layers is not None else cfg["n_layers"])
        self.n_bins, self.n_gauss = nb, ng
        self.max_columns, self.flags = int(max_columns), int(cfg["flags"])
        c = Config(self.n_layers, nb, ng, nP, nT, self.max_columns, _ptr(keep["ktab_p"]), _ptr(keep["ktab_t"]),
                   _ptr(ktab), _ptr(keep["bin_edges"]), _ptr(keep["gauss_w"]), _ptr(keep["scat_gas"]),
                   _ptr(keep["cloud_ext"]), _ptr(keep["cloud_w0"]), _ptr(keep["cloud_g0"]),
                   float(cfg["cloud_p_top"]), float(cfg["cloud_p_bot"]), float(cfg["gravity"]), float(cfg["cp"]),
                   float(cfg.get("eps2", 2.0 / 3.0)), float(cfg.get("e_tau", 1e-4)), float(cfg.get("gcrit_tol", 1e-5)),
                   float(cfg.get("w0_transition", 0.1)), float(cfg.get("f_toa", 0.0)), self.flags)
        h = C.c_void_p()
        _check(L.helios_rt_create(C.byref(c), C.byref(h)))
        self._h = h

    def output_shapes(self, n: int) -> dict:
        N, nb = self.n_layers, self.n_bins
        return dict(F_up=(n, N + 1), F_down=(n, N + 1), F_net=(n, N + 1), dTdt=(n, N), F_beam=(n, N + 1),
                    F_up_toa_bin=(n, nb))

    def launch_info(self) -> dict:
        info = (C.c_int32 * 8)()
        _check(load_library().helios_rt_launch_info(self._h, info))
        keys = ("block", "tiles", "smem_bytes", "registers", "blocks_per_sm", "local_bytes", "launches_per_step",
                "sm_count")
        return dict(zip(keys, list(info)))

    def debug_set_launch(self, warps: int = 0, ppt: int = 0, rows: int = -1, maxt: int = -1, minb: int = -1) -> None:
        """helios_rt_debug_set_launch (include/helios_rt_debug.h; tests and tuning only)."""
        _check(load_library().helios_rt_debug_set_launch(self._h, int(warps), int(ppt), int(rows), int(maxt), int(minb)),
               self._h)

    def debug_force_stuck(self, on: bool = True) -> None:
        """Tests only (helios_rt_debug.h): later steps never see their columns published and must report error -6."""
        _check(load_library().helios_rt_debug_force_stuck(self._h, int(bool(on))), self._h)

    def debug_set_workers(self, workers: int) -> None:
        """helios_rt_debug_set_workers (helios_rt_debug.h; tuning only): cap the persistent workers per tile (0 = no cap)."""
        _check(load_library().helios_rt_debug_set_workers(self._h, int(workers)), self._h)

    def debug_force_two_launches(self, on: bool = True) -> None:
        """Tests only (helios_rt_debug.h): take the non-cooperative fallback path (rt_prep_kernel + plain launch)."""
        _check(load_library().helios_rt_debug_force_two_launches(self._h, int(bool(on))), self._h)

    def debug_get_launch(self) -> dict:
        info = (C.c_int32 * 16)()
        _check(load_library().helios_rt_debug_get_launch(self._h, info))
        keys = ("warps", "ppt", "rows", "unused", "maxt", "minb", "tiles", "workers", "blocks_per_sm", "registers",
                "local_bytes", "smem_bytes", "stack_mib", "variant", "n_variants")
        return dict(zip(keys, list(info)))

    def step_iterative(self, p, T, mu_star, stellar_flux, f_internal: float, out: dict, n_iterations: int,
                       stream=None) -> None:
        """The pair-wise iterative scheme Thomas replaces (helios_rt_step_iterative); arguments as `step`."""
        self.step(p, T, mu_star, stellar_flux, f_internal, out, stream=stream, _n_iter=int(n_iterations))

    def step(self, p, T, mu_star, stellar_flux, f_internal: float, out: dict, stream=None, _n_iter=None) -> None:
        """Device step: torch CUDA float64 contiguous tensors; `out` maps output names to pre-allocated
        tensors (omitted = not wanted).  Asynchronous on `stream` (default: torch's current stream)."""
        import torch
        n = int(p.shape[0])
        for name, t, shape in (("p", p, (n, self.n_layers)), ("T", T, (n, self.n_layers)), ("mu_star", mu_star, (n,)),
                               ("stellar_flux", stellar_flux, (self.n_bins,))):
            if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shape):
                raise HeliosRTError(f"helios_rt error -1: {name} must be a contiguous CUDA float64 tensor {shape}")
        shapes = self.output_shapes(n)
        ptrs = {}
        for k, t in out.items():
            if k not in shapes:
                raise HeliosRTError(f"helios_rt error -1: unknown output {k}")
            if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shapes[k]):
                raise HeliosRTError(f"helios_rt error -1: output {k} must be a contiguous CUDA float64 tensor {shapes[k]}")
            ptrs[k] = t.data_ptr()
        i = Inputs(n, p.data_ptr(), T.data_ptr(), mu_star.data_ptr(), stellar_flux.data_ptr(), float(f_internal))
        o = Outputs(*[ptrs.get(k) for k in OUTPUT_NAMES])
        st = (stream if stream is not None else torch.cuda.current_stream()).cuda_stream
        if _n_iter is None:
            _check(load_library().helios_rt_step(self._h, C.byref(i), C.byref(o), C.c_void_p(st)), self._h)
        else:
            _check(load_library().helios_rt_step_iterative(self._h, C.byref(i), C.byref(o), _n_iter, C.c_void_p(st)),
                   self._h)

    def step_host(self, p, T, mu_star, stellar_flux, f_internal: float, out: dict) -> None:
        """Host step (end-to-end path): numpy arrays or CPU (ideally pinned) torch tensors, float64 contiguous.
        Copies in, runs, copies the requested outputs back, synchronises."""
        def addr(x):
            if isinstance(x, np.ndarray):
                if x.dtype != np.float64 or not x.flags.c_contiguous:
                    raise HeliosRTError("helios_rt error -1: host arrays must be contiguous float64")
                return x.ctypes.data
            return x.data_ptr()
        n = int(p.shape[0])
        shapes = self.output_shapes(n)
        for k, t in out.items():
            if k not in shapes or tuple(t.shape) != shapes[k]:
                raise HeliosRTError(f"helios_rt error -1: bad output {k}")
        if tuple(p.shape) != (n, self.n_layers) or tuple(T.shape) != (n, self.n_layers) or \
                tuple(mu_star.shape) != (n,) or tuple(stellar_flux.shape) != (self.n_bins,):
            raise HeliosRTError("helios_rt error -1: bad input shape")
        i = Inputs(n, addr(p), addr(T), addr(mu_star), addr(stellar_flux), float(f_internal))
        o = Outputs(*[addr(out[k]) if k in out else None for k in OUTPUT_NAMES])
        _check(load_library().helios_rt_step_host(self._h, C.byref(i), C.byref(o)), self._h)

    def close(self) -> None:
        if getattr(self, "_h", None):
            load_library().helios_rt_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _dev(t, shape, name):
    import torch
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise HeliosRTError(f"helios_rt error -1: {name} must be a contiguous CUDA float64 tensor {tuple(shape)}")
    return t.data_ptr()


def _stream(stream):
    import torch
    return C.c_void_p((stream if stream is not None else torch.cuda.current_stream()).cuda_stream)


def extend_top(p, T, n_extra: int, p_min: float, p_ext, T_ext, stream=None) -> None:
    """helios_rt_extend_top on CUDA tensors: p, T [n, N] -> p_ext, T_ext [n, N + n_extra] (pre-allocated)."""
    n, N = p.shape
    _check(load_library().helios_rt_extend_top(n, N, int(n_extra), float(p_min), _dev(p, (n, N), "p"), _dev(T, (n, N), "T"),
                                               _dev(p_ext, (n, N + n_extra), "p_ext"),
                                               _dev(T_ext, (n, N + n_extra), "T_ext"), _stream(stream)))


def phase_curve_workspace(n_columns: int, n_bins: int, n_phases: int, device="cuda"):
    """A scratch tensor of the size helios_rt_phase_curve needs."""
    import torch
    nbytes = load_library().helios_rt_phase_curve_workspace_bytes(int(n_columns), int(n_bins), int(n_phases))
    if nbytes < 0:
        _check(int(nbytes))
    return torch.empty(max(nbytes // 8, 1), dtype=torch.float64, device=device)


def phase_curve(F_toa_bin, lon, lat, area, alpha, F_phase_bin, bin_edges=None, lam1=0.0, lam2=0.0, F_phase_band=None,
                workspace=None, stream=None) -> None:
    """helios_rt_phase_curve on CUDA tensors (Eqs. 25-26; band integral of Eq. 23 if F_phase_band is given).
    `workspace`: tensor from phase_curve_workspace (allocated here if omitted -- pass it to stay allocation-free)."""
    n, nb = F_toa_bin.shape
    na = alpha.shape[0]
    if workspace is None:
        workspace = phase_curve_workspace(n, nb, na, F_toa_bin.device)
    need = load_library().helios_rt_phase_curve_workspace_bytes(n, nb, na)
    if not (workspace.is_cuda and workspace.is_contiguous() and workspace.numel() * workspace.element_size() >= need):
        raise HeliosRTError("helios_rt error -1: workspace too small")
    _check(load_library().helios_rt_phase_curve(
        n, nb, na, _dev(F_toa_bin, (n, nb), "F_toa_bin"), _dev(lon, (n,), "lon"), _dev(lat, (n,), "lat"),
        _dev(area, (n,), "area"), _dev(alpha, (na,), "alpha"),
        None if bin_edges is None else _dev(bin_edges, (nb + 1,), "bin_edges"), float(lam1), float(lam2),
        _dev(F_phase_bin, (na, nb), "F_phase_bin"),
        None if F_phase_band is None else _dev(F_phase_band, (na,), "F_phase_band"), workspace.data_ptr(),
        _stream(stream)))


PHASE_CURVE_NOALLOC_MAX_BYTES = 8 << 20   # HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES of include/helios_rt.h


def phase_curve_noalloc(F_toa_bin, lon, lat, area, alpha, F_phase_bin, bin_edges=None, lam1=0.0, lam2=0.0,
                        F_phase_band=None, stream=None) -> None:
    """helios_rt_phase_curve_noalloc on CUDA tensors: the phase curve (same arguments and bit-identical results as
    `phase_curve`) for code that is not allowed to allocate device memory where it runs -- a plug-in inside an
    application that owns the whole GPU, a latency-critical path that must not enter the CUDA allocator, a worker
    whose memory budget is already spent.  The scratch that `phase_curve` takes as `workspace` is a fixed 8 MiB array
    inside libhelios_rt.so instead, so:

    * problems needing more than PHASE_CURVE_NOALLOC_MAX_BYTES of scratch (ceil(n/128) * n_phases * n_bins * 8
      bytes) raise HeliosRTError with code -5; use `phase_curve` with your own workspace for those;
    * make the first call on each device at start-up, outside any stream capture (it looks up the array's address
      on that device, once), with the tensors' device as the current device;
    * every call on a device shares that one array: keep the calls stream-ordered -- two that overlap on the GPU
      corrupt each other.

    This wrapper creates no tensor either (it passes the pointers of the ones it is given)."""
    n, nb = F_toa_bin.shape
    na = alpha.shape[0]
    _check(load_library().helios_rt_phase_curve_noalloc(
        n, nb, na, _dev(F_toa_bin, (n, nb), "F_toa_bin"), _dev(lon, (n,), "lon"), _dev(lat, (n,), "lat"),
        _dev(area, (n,), "area"), _dev(alpha, (na,), "alpha"),
        None if bin_edges is None else _dev(bin_edges, (nb + 1,), "bin_edges"), float(lam1), float(lam2),
        _dev(F_phase_bin, (na, nb), "F_phase_bin"),
        None if F_phase_band is None else _dev(F_phase_band, (na,), "F_phase_band"), _stream(stream)))


def advance_1d(dt: float, gravity: float, R_d: float, p_ref: float, z, dTdt, T, p, rho=None, stream=None) -> None:
    """helios_rt_advance_1d on CUDA tensors: T [n, N] updated in place, p (and rho) written."""
    n, N = T.shape
    _check(load_library().helios_rt_advance_1d(
        n, N, float(dt), float(gravity), float(R_d), float(p_ref), _dev(z, (N,), "z"),
        None if dTdt is None else _dev(dTdt, (n, N), "dTdt"), _dev(T, (n, N), "T"), _dev(p, (n, N), "p"),
        None if rho is None else _dev(rho, (n, N), "rho"), _stream(stream)))


# ---- include/helios_rt_selftest.h (libhelios_rt_selftest.so): test / benchmark hooks ----
def selftest_math(x):
    x = _np(x)
    outs = [np.empty_like(x) for _ in range(4)]
    _check(load_selftest_library().helios_rt_selftest_math(x.size, _ptr(x), *[_ptr(o) for o in outs]))
    return tuple(outs)  # rcp, rsqrt, exp(-|x|), 1-exp(-|x|)


def selftest_planck(T, lam_lo, lam_hi) -> np.ndarray:
    T, lo, hi = _np(T), _np(lam_lo), _np(lam_hi)
    out = np.empty_like(T)
    _check(load_selftest_library().helios_rt_selftest_planck(T.size, _ptr(T), _ptr(lo), _ptr(hi), _ptr(out)))
    return out


def selftest_planck_G(x) -> np.ndarray:
    x = _np(x)
    out = np.empty_like(x)
    _check(load_selftest_library().helios_rt_selftest_planck_G(x.size, _ptr(x), _ptr(out)))
    return out


def measure_dfma_peak(iters: int = 1 << 16) -> tuple[float, float]:
    a, b = C.c_double(), C.c_double()
    _check(load_selftest_library().helios_rt_measure_dfma_peak(int(iters), C.byref(a), C.byref(b)))
    return a.value, b.value


def measure_latencies() -> dict:
    lat = (C.c_double * 4)()
    _check(load_selftest_library().helios_rt_measure_latencies(lat))
    return dict(zip(("dfma", "rcp_link", "lds_f2i_link", "dadd"), list(lat)))
