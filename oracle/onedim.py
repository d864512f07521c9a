"""CPU oracle for the "1-D mode" of THOR+HELIOS (Sec. 3) -- TEST
INFRASTRUCTURE ONLY.  Plain numpy, fp64; shares nothing with the CUDA path.

"The only physical processes acting on the column are the radiative-transfer followed by an adjustment to the
pressure and density in each layer to preserve hydrostatic balance" (L403).  After the RT module has updated the
layer temperatures, "the pressure in the lowest layer is held at the reference pressure, P_ref.  The pressure in
each layer, i, above is set based on the layer below, i-1, according to" Eq.(20) (L405-408); "the density is
calculated from the ideal gas law".

Reading R25 (garbled sign): as extracted, Eq.(20) has "-" in front of g/(2 R_d T) in BOTH numerator and
denominator, which makes an isothermal column isobaric.  The text says the relation "is derived from the discrete
equation for hydrostatic balance and the ideal gas law": (P_i - P_{i-1})/(z_i - z_{i-1}) = -g (rho_i + rho_{i-1})/2,
rho = P/(R_d T), which gives
    P_i = P_{i-1} [1/(z_i - z_{i-1}) - g/(2 R_d T_{i-1})] / [1/(z_i - z_{i-1}) + g/(2 R_d T_i)];
that form (denominator "+") is taken.  Reading R26: the temperature update is the explicit step
T <- T + dt dT/dt with the heating rate of the RT step (L127 "heating rates", constant time step L384).
"""
from __future__ import annotations

import numpy as np


def advance_temperature(T: np.ndarray, dTdt: np.ndarray, dt: float) -> np.ndarray:
    return np.asarray(T, dtype=np.float64) + dt * np.asarray(dTdt, dtype=np.float64)


def hydrostatic_rebalance(z: np.ndarray, T: np.ndarray, p_ref: float, gravity: float, R_d: float):
    """z [N] layer-centre altitudes (m, ascending), T [ncol, N] -> (p [ncol, N], rho [ncol, N])."""
    z = np.asarray(z, dtype=np.float64)
    T = np.asarray(T, dtype=np.float64)
    ncol, N = T.shape
    p = np.empty_like(T)
    for c in range(ncol):
        p[c, 0] = p_ref
        for i in range(1, N):
            inv_dz = 1.0 / (z[i] - z[i - 1])
            p[c, i] = p[c, i - 1] * (inv_dz - gravity / (2.0 * R_d * T[c, i - 1])) / (inv_dz + gravity / (2.0 * R_d * T[c, i]))
    rho = p / (R_d * T)
    return p, rho


def run(rt_step, z, T0, p_ref, gravity, R_d, dt, n_steps):
    """n_steps of: p <- rebalance(T); dT/dt <- rt_step(p, T); T <- T + dt dT/dt.  `rt_step(p, T) -> dTdt` is the
    RT oracle bound to its configuration.  Returns (p, T) after the last step (p consistent with T)."""
    T = np.asarray(T0, dtype=np.float64).copy()
    p, _ = hydrostatic_rebalance(z, T, p_ref, gravity, R_d)
    for _ in range(n_steps):
        dTdt = rt_step(p, T)
        T = advance_temperature(T, dTdt, dt)
        p, _ = hydrostatic_rebalance(z, T, p_ref, gravity, R_d)
    return p, T
