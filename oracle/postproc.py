"""CPU oracle for the post-processing side of THOR+HELIOS -- TEST INFRASTRUCTURE ONLY.

Plain numpy, fp64, written out from /root/reference/PAPER.md; shares nothing with the CUDA path.

  extend_top   -- PAPER.md L385: "we extend the top altitude of the simulation, extrapolating the temperatures
                  down to pressures of <= 1 ubar ... the temperatures of each column are isothermal above the
                  original model top and take on the value of the top-most layer ... Users of the code can
                  specify the desired lowest pressure level of the extrapolation."
  band_weights -- the wavelength integral of Eq.(23) (L521) over [lam1, lam2] on the k-table bins.
  phase_curve  -- Eqs.(25)-(26) (L546-552): F = sum_i F_TOA,i / pi * mu_i * A_i / R_p^2 with
                  mu_i = cos(theta_i) cos(phi_i - alpha) on the visible hemisphere, 0 elsewhere.

Readings: R21 the paper does not say how the added levels are spaced: n_extra layers equally spaced
in ln p above the top layer, with the per-layer pressure ratio q = min(p[N-1]/p[N-2], (p_min/p[N-1])^(1/n_extra)),
i.e. the column's own top spacing, stretched if that would not reach p_min; so the new top is always <= p_min.
R22 the visibility test of Eq.(26), alpha - pi/2 < phi < alpha + pi/2, is taken modulo 2 pi (the GCM's longitudes
run over 0..2 pi, L533): visible iff cos(phi - alpha) > 0.  R24 a bin that straddles lam1 or lam2 contributes
the length of its overlap with [lam1, lam2] (F_TOA is per unit wavelength and constant over a bin).
"""
from __future__ import annotations

import numpy as np


def extend_top(p: np.ndarray, T: np.ndarray, n_extra: int, p_min: float):
    """p, T [ncol, N] (layer 0 = bottom) -> p_ext, T_ext [ncol, N + n_extra]."""
    p = np.asarray(p, dtype=np.float64)
    T = np.asarray(T, dtype=np.float64)
    ncol, N = p.shape
    p_ext = np.empty((ncol, N + n_extra))
    T_ext = np.empty((ncol, N + n_extra))
    for c in range(ncol):
        p_ext[c, :N] = p[c]
        T_ext[c, :N] = T[c]
        if n_extra == 0:
            continue
        p_top = p[c, N - 1]
        q_own = p[c, N - 1] / p[c, N - 2] if N > 1 else 0.1 ** 0.5
        q_need = (p_min / p_top) ** (1.0 / n_extra)
        q = min(q_own, q_need)
        for k in range(1, n_extra + 1):
            p_ext[c, N - 1 + k] = p_top * q ** k
            T_ext[c, N - 1 + k] = T[c, N - 1]          # isothermal above the model top (L385)
    return p_ext, T_ext


def band_weights(bin_edges: np.ndarray, lam1: float, lam2: float) -> np.ndarray:
    """Length of the overlap of every bin [edges[b], edges[b+1]] with [lam1, lam2] (metres)."""
    e = np.asarray(bin_edges, dtype=np.float64)
    w = np.zeros(e.size - 1)
    for b in range(e.size - 1):
        lo, hi = max(e[b], lam1), min(e[b + 1], lam2)
        w[b] = hi - lo if hi > lo else 0.0
    return w


def phase_curve(F_toa_bin: np.ndarray, lon: np.ndarray, lat: np.ndarray, area: np.ndarray, alpha: np.ndarray,
                bin_edges: np.ndarray | None = None, lam1: float | None = None, lam2: float | None = None):
    """Eq.(25): F[alpha, b] = sum_i F_TOA[i, b] / pi * mu_i(alpha) * area_i, area_i = A_i / R_p^2, mu_i from Eq.(26).
    With bin_edges, lam1, lam2 also the band integral of Eq.(23): F_band[alpha] = sum_b w_b F[alpha, b].
    Returns (F [n_alpha, n_bins], F_band [n_alpha] or None)."""
    F_toa_bin = np.asarray(F_toa_bin, dtype=np.float64)
    ncol, nb = F_toa_bin.shape
    alpha = np.atleast_1d(np.asarray(alpha, dtype=np.float64))
    out = np.zeros((alpha.size, nb))
    for a in range(alpha.size):
        for i in range(ncol):
            c = np.cos(lon[i] - alpha[a])
            mu_i = np.cos(lat[i]) * c if c > 0.0 else 0.0              # Eq.(26)
            out[a] += F_toa_bin[i] / np.pi * mu_i * area[i]            # Eq.(25)
    band = None
    if bin_edges is not None:
        w = band_weights(bin_edges, lam1, lam2)
        band = out @ w
    return out, band
