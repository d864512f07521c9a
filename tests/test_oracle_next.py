"""Pins of the oracle's NEXT-row functions: post-processing (column extension, phase curve),
1-D mode (hydrostatic re-balance, explicit temperature step) and the pair-wise iterative scheme.  Each is
checked against something other than itself: closed forms, the continuous integral by brute-force quadrature,
the discrete relation the paper says the formula is derived from, hand-computed values.  CPU only."""
from __future__ import annotations

import numpy as np
import pytest


@pytest.fixture(scope="module")
def geo():
    from paper_2203_02293_b200 import workloads as W
    return W.grid_geometry(4)


# ------------------------------------------------------------------------------------ phase curve, Eqs. 23-26
def test_control_volumes_tile_the_sphere(geo):
    lon, lat, area = geo
    assert area.shape == (2562,) and abs(area.sum() - 4 * np.pi) < 1e-10
    assert lon.min() >= 0 and lon.max() < 2 * np.pi


def test_phase_curve_uniform_emission_returns_the_flux(geo):
    """A planet emitting F0 everywhere: Eq.(23) = F0/pi x (projected area of the unit disc = pi) = F0 at every phase."""
    from oracle import postproc
    lon, lat, area = geo
    F = np.full((lon.size, 3), 7.5)
    out, _ = postproc.phase_curve(F, lon, lat, area, np.array([-3.0, -1.0, 0.0, 0.4, 2.5]))
    assert out.shape == (5, 3)
    assert np.allclose(out, 7.5, rtol=2e-3)


def test_phase_curve_lambert_hot_spot_closed_form_and_sign_of_alpha(geo):
    """F_TOA = F0 max(n.s, 0) with the hot spot s at longitude phi0 on the equator: the disc integral is the Lambert
    phase function, F(alpha) = F0/pi * 2/3 (sin g + (pi - g) cos g), g = |alpha - phi0|.  Peaks at alpha = +phi0:
    pins the sign convention of alpha in Eq.(26)."""
    from oracle import postproc
    lon, lat, area = geo
    phi0, F0 = 0.7, 3.0
    n_dot_s = np.cos(lat) * np.cos(lon - phi0)
    F = (F0 * np.maximum(n_dot_s, 0.0))[:, None]
    alpha = np.array([0.7, -0.7, 0.2, 1.5, -2.0, 0.7 + np.pi])
    out, _ = postproc.phase_curve(F, lon, lat, area, alpha)
    g = np.abs(np.angle(np.exp(1j * (alpha - phi0))))
    exact = F0 / np.pi * (2.0 / 3.0) * (np.sin(g) + (np.pi - g) * np.cos(g))
    assert np.allclose(out[:, 0], exact, atol=3e-3 * exact.max())
    assert out[0, 0] > out[1, 0] and abs(out[5, 0]) < 1e-12


def test_phase_curve_matches_brute_force_quadrature_of_eq23(geo):
    """Eq.(25) on the icosahedral grid against the continuous Eq.(23) by a midpoint rule on a fine lat-lon grid."""
    from oracle import postproc
    lon, lat, area = geo
    field = lambda th, ph: 2.0 + 0.8 * np.sin(th) + 0.5 * np.cos(2 * ph + 0.3) * np.cos(th) ** 2
    F = field(lat, lon)[:, None]
    nth, nph = 600, 1200
    th = (np.arange(nth) + 0.5) / nth * np.pi - np.pi / 2
    for alpha in (0.0, 1.1, -2.3):
        ph = alpha - np.pi / 2 + (np.arange(nph) + 0.5) / nph * np.pi       # Eq.(24) limits, phi - alpha in (-pi/2, pi/2)
        TH, PH = np.meshgrid(th, ph, indexing="ij")
        integrand = field(TH, PH) / np.pi * np.cos(TH) ** 2 * np.cos(PH - alpha)
        exact = integrand.sum() * (np.pi / nth) * (np.pi / nph)
        out, _ = postproc.phase_curve(F, lon, lat, area, np.array([alpha]))
        assert out[0, 0] == pytest.approx(exact, rel=3e-3)


def test_phase_curve_visibility_mask_and_single_column():
    from oracle import postproc
    F = np.array([[4.0, 8.0]])
    a = 0.3
    out, _ = postproc.phase_curve(F, np.array([a]), np.array([0.5]), np.array([0.01]), np.array([a]))
    assert np.allclose(out[0], F[0] / np.pi * np.cos(0.5) * 0.01, rtol=1e-15)
    for dphi in (np.pi / 2 + 0.01, -np.pi / 2 - 0.01, np.pi):
        out, _ = postproc.phase_curve(F, np.array([a + dphi]), np.array([0.5]), np.array([0.01]), np.array([a]))
        assert np.all(out == 0.0)
    # longitudes are periodic (reading R22): phi = 6.2 is visible from alpha = 0
    out, _ = postproc.phase_curve(F, np.array([6.2]), np.array([0.0]), np.array([1.0]), np.array([0.0]))
    assert out[0, 0] == pytest.approx(4.0 / np.pi * np.cos(6.2 - 2 * np.pi), rel=1e-14)


def test_band_weights_hand_values():
    from oracle import postproc
    e = np.array([1.0, 2.0, 3.0, 4.0])
    assert np.allclose(postproc.band_weights(e, 1.5, 3.2), [0.5, 1.0, 0.2], atol=1e-15)
    assert np.all(postproc.band_weights(e, 5.0, 6.0) == 0)
    assert np.allclose(postproc.band_weights(e, 0.0, 10.0), [1, 1, 1])
    # a flat spectrum integrates to F (lam2 - lam1)
    out, band = postproc.phase_curve(np.full((1, 3), 2.0), np.array([0.0]), np.array([0.0]), np.array([np.pi]),
                                     np.array([0.0]), e, 1.25, 3.75)
    assert band[0] == pytest.approx(2.0 * 2.5, rel=1e-14)


# ------------------------------------------------------------------------------------ column extension, L385
def test_extend_top_hand_values():
    from oracle import postproc
    p = np.array([[1e5, 1e4, 1e3]])
    T = np.array([[1500.0, 1200.0, 900.0]])
    pe, Te = postproc.extend_top(p, T, 3, 1.0)       # own ratio 0.1 reaches 1 Pa exactly
    assert np.allclose(pe[0], [1e5, 1e4, 1e3, 1e2, 1e1, 1e0], rtol=1e-14)
    assert np.all(Te[0, 3:] == 900.0) and np.all(Te[0, :3] == T[0])
    pe, _ = postproc.extend_top(p, T, 6, 1.0)        # own spacing goes beyond p_min: kept (top <= p_min)
    assert pe[0, -1] == pytest.approx(1e-3, rel=1e-13)
    pe, _ = postproc.extend_top(p, T, 2, 1.0)        # own spacing too fine: stretched to end exactly at p_min
    assert np.allclose(pe[0, 3:], [10 ** 1.5, 1.0], rtol=1e-13)
    pe, Te = postproc.extend_top(p, T, 0, 1.0)
    assert np.array_equal(pe, p) and np.array_equal(Te, T)


def test_extend_top_is_log_equally_spaced_and_reaches_p_min():
    from oracle import postproc
    rng = np.random.default_rng(5)
    p = np.sort(10 ** rng.uniform(0, 7, (8, 12)), axis=1)[:, ::-1].copy()
    T = rng.uniform(500, 2000, p.shape)
    pe, Te = postproc.extend_top(p, T, 7, 0.1)
    r = pe[:, 12:] / pe[:, 11:-1]
    assert np.allclose(r, r[:, :1], rtol=1e-12)
    assert np.all(pe[:, -1] <= 0.1 * (1 + 1e-12)) and np.all(np.diff(pe, axis=1) < 0)
    assert np.all(Te[:, 12:] == T[:, 11:12])


# ------------------------------------------------------------------------------------ 1-D mode, Eq. 20
def test_hydrostatic_rebalance_satisfies_the_discrete_balance_it_is_derived_from():
    """(P_i - P_{i-1}) / (z_i - z_{i-1}) = -g (rho_i + rho_{i-1}) / 2 with rho = P / (R_d T)  (L408, reading R25)."""
    from oracle import onedim
    rng = np.random.default_rng(3)
    z = np.cumsum(rng.uniform(2e4, 9e4, 30))
    T = rng.uniform(600, 2500, (4, 30))
    g, R = 47.0, 3553.0
    p, rho = onedim.hydrostatic_rebalance(z, T, 1e8, g, R)
    assert np.all(p[:, 0] == 1e8) and np.all(np.diff(p, axis=1) < 0)
    lhs = np.diff(p, axis=1) / np.diff(z)[None, :]
    rhs = -g * 0.5 * (rho[:, 1:] + rho[:, :-1])
    assert np.allclose(lhs, rhs, rtol=1e-12)
    assert np.allclose(rho, p / (R * T), rtol=1e-15)


def test_hydrostatic_rebalance_isothermal_limit_is_the_barometric_formula():
    from oracle import onedim
    g, R, T0 = 47.0, 3553.0, 1500.0
    H = R * T0 / g
    err = []
    for n in (200, 400):
        z = np.linspace(0.0, 5 * H, n)
        p, _ = onedim.hydrostatic_rebalance(z, np.full((1, n), T0), 1e7, g, R)
        err.append(np.max(np.abs(p[0] / (1e7 * np.exp(-z / H)) - 1)))
    assert err[1] < 1e-4 and 3.5 < err[0] / err[1] < 4.5      # second-order in dz


def test_one_d_run_with_a_relaxation_heating_has_the_geometric_closed_form():
    from oracle import onedim
    z = np.linspace(0, 2e6, 10)
    T0 = np.linspace(2000, 1000, 10)[None, :]
    Teq, tau, dt = 1400.0, 5000.0, 300.0
    p, T = onedim.run(lambda p, T: -(T - Teq) / tau, z, T0, 1e7, 47.0, 3553.0, dt, 25)
    assert np.allclose(T, Teq + (T0 - Teq) * (1 - dt / tau) ** 25, rtol=1e-13)
    p2, _ = onedim.hydrostatic_rebalance(z, T, 1e7, 47.0, 3553.0)
    assert np.array_equal(p, p2)
    assert np.array_equal(onedim.advance_temperature(T0, np.ones_like(T0), 2.0), T0 + 2.0)


# ------------------------------------------------------------------------------------ pair-wise iteration
def _column(rng, L):
    return 10 ** rng.uniform(-2, 0.7, L), rng.uniform(0, 0.95, L), rng.uniform(0, 0.8, L), rng.uniform(1, 3, L + 1)


def test_iteration_converges_to_the_dense_solution_of_the_system():
    """L258-270: N iterations propagate radiation across N layers; the limit is the solution of Eq.(12)."""
    import oracle
    rng = np.random.default_rng(17)
    L = 7
    dtau, w0, g0, B = _column(rng, L)
    mu, Fs, Fboa = 0.6, 5.0, 0.4
    A, Bm, C, D, fb = oracle.assemble_blocks(dtau, w0, g0, B[:-1], B[:-1], mu, Fs, Fboa)
    n = L + 1
    M = np.zeros((2 * n, 2 * n))
    for l in range(n):
        M[2 * l:2 * l + 2, 2 * l:2 * l + 2] = Bm[l]
        if l > 0:
            M[2 * l:2 * l + 2, 2 * l - 2:2 * l] = A[l]
        if l < n - 1:
            M[2 * l:2 * l + 2, 2 * l + 2:2 * l + 4] = C[l]
    X = np.linalg.solve(M, D.reshape(-1))
    prev = None
    for nit in (1, 3, 10, 400):
        fu, fd, fb2 = oracle.column_mono_iter(dtau, w0, g0, B[:-1], B[:-1], mu, Fs, Fboa, nit)
        err = max(np.abs(fu - X[0::2]).max(), np.abs(fd - X[1::2]).max())
        assert prev is None or err < prev
        prev = err
    assert prev < 1e-12 * np.abs(X).max()
    assert np.allclose(fb2, fb)


def test_one_iteration_is_exact_without_scattering():
    """omega0 = 0: the streams decouple (L258), so a single up + down pass gives the closed form
    F_dn[j] = T F_dn[j+1] + pi B (1 - T), F_up[0] = F_dn[0] + F_BOA + beam, F_up[j+1] = T F_up[j] + pi B (1 - T).
    With zero initial fluxes the upward pass of iteration 1 sees F_dn = 0 at the BOA, so 2 iterations are needed."""
    import oracle
    rng = np.random.default_rng(23)
    L = 8
    dtau = 10 ** rng.uniform(-2, 0.5, L)
    B = rng.uniform(1, 3, L)
    mu, Fs, Fboa = 0.45, 6.0, 0.7
    fu, fd, fb = oracle.column_mono_iter(dtau, np.zeros(L), np.zeros(L), B, B, mu, Fs, Fboa, 2)
    tr = np.exp(-2 * dtau)
    edn = np.zeros(L + 1)
    for j in range(L - 1, -1, -1):
        edn[j] = tr[j] * edn[j + 1] + np.pi * B[j] * (1 - tr[j])
    tau = np.concatenate([np.cumsum(dtau[::-1])[::-1], [0.0]])
    beam = mu * Fs * np.exp(-tau / mu)
    eup = np.zeros(L + 1)
    eup[0] = edn[0] + Fboa + beam[0]
    for j in range(L):
        eup[j + 1] = tr[j] * eup[j] + np.pi * B[j] * (1 - tr[j])
    assert np.allclose(fd, edn, rtol=1e-13) and np.allclose(fu, eup, rtol=1e-13) and np.allclose(fb, beam, rtol=1e-13)


def test_rt_step_with_iterations_approaches_the_thomas_step():
    import oracle
    from paper_2203_02293_b200 import workloads as W
    cfg, inp, meta = W.make(1, columns=slice(0, 4))
    ref = oracle.rt_step(cfg, inp, want=("F_net",))["F_net"]
    e = [np.abs(oracle.rt_step(dict(cfg, n_iterations=k), inp, want=("F_net",))["F_net"] - ref).max() for k in (2, 8, 60)]
    assert e[0] > e[1] > e[2] and e[2] < 1e-9 * np.abs(ref).max()


# ------------------------------------------------------------------------- 1-D mode run to a steady state (Sec. 3)
def _equilibrate(oracle_mod, cfg, inp, extra, n_steps):
    from oracle import onedim
    g = cfg["gravity"]
    step = lambda p, T: oracle_mod.rt_step(cfg, dict(inp, p=p, T=T), want=("dTdt",), real="f64")["dTdt"]
    p, T = onedim.run(step, extra["z"], inp["T"], extra["p_ref"], g, extra["R_d"], extra["dt"], n_steps)
    return p, T, oracle_mod.rt_step(cfg, dict(inp, p=p, T=T), want=("dTdt", "F_net", "F_up", "F_down"))


@pytest.mark.parametrize("zenith,cp,n_steps", [((0.0, 30.0, 60.0), 2000.0, 12000), ((89.0,), 500.0, 36000)])
def test_one_d_mode_reaches_radiative_equilibrium(oracle_mod, zenith, cp, n_steps):
    """PAPER.md Sec. 3 (L401-410): RT step + hydrostatic re-balance, stepped until nothing changes.  What makes this
    physics rather than plumbing: in a steady state every layer's heating rate vanishes, which by the heating-rate
    reading R14 means the net flux is the same at every interface, and by Eq.(10) (L237-239) that constant is the
    internal flux sum_b dlam_b pi B_b(T_int) fed in at the bottom -- whatever the zenith angle.  A sign error in the
    heating rate diverges instead of relaxing; a beam left out of F_down (L235) equilibrates to a net flux that is
    not F_BOA."""
    from paper_2203_02293_b200 import workloads as W
    cfg, inp, meta, extra = W.make_one_d(zenith, cp)
    p, T, r = _equilibrate(oracle_mod, cfg, inp, extra, n_steps)
    e = cfg["bin_edges"]
    SIGMA = 2 * np.pi**5 * 1.380649e-23**4 / (15 * 6.62607015e-34**3 * 299792458.0**2)
    T_int = (inp["f_internal"] / SIGMA) ** 0.25
    F_boa = sum((e[b + 1] - e[b]) * np.pi * oracle_mod.planck_bin_mean(T_int, e[b], e[b + 1]) for b in range(meta["n_bins"]))
    absorbed = inp["mu_star"] * meta["F_star_tot"]
    assert np.all(np.isfinite(T)) and T.min() > 100.0 and T.max() < 4000.0
    assert np.abs(T - inp["T"]).max() > 50.0                                   # it went somewhere
    # F_net constant with depth and equal to the internal flux, to 1e-9 of the stellar flux the column absorbs
    assert np.all(np.abs(r["F_net"] - F_boa) <= 1e-9 * absorbed[:, None])
    # ... although the fluxes themselves are of the order of the stellar flux
    assert np.all(r["F_down"][:, -1] > 0.5 * absorbed)
    # nothing changes any more: |dT/dt| dt below 1e-7 K per step everywhere
    assert np.abs(r["dTdt"]).max() * extra["dt"] < 1e-7
    # hotter under a higher sun
    if len(zenith) > 1:
        assert np.all(np.diff(T, axis=0) < 0)
