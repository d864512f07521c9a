"""Pins for the CPU oracle (oracle/helios_oracle.c): every part of it is checked against something
other than itself -- quadrature, closed forms, invariants, a library LU, an ODE integrator, the
iterative scheme the paper replaces, and a 40-digit worked example.  CPU only (-m "not gpu").

Citations are PAPER.md lines (/root/reference/PAPER.md at build time; not read at run time).
"""
from __future__ import annotations

from pathlib import Path

import mpmath as mp
import numpy as np
import pytest
from scipy.integrate import solve_ivp

H, CL, KB = 6.62607015e-34, 299792458.0, 1.380649e-23
SIGMA = 2 * np.pi**5 * KB**4 / (15 * H**3 * CL**2)
GOLD = Path(__file__).parent / "golden"


def _golden():
    d = {}
    for line in (GOLD / "worked_example.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        d[k] = np.array([float(x) for x in v])
    return d


# ------------------------------------------------------------------------------------------ Planck
@pytest.mark.parametrize("x", [1e-3, 0.05, 0.3, 0.999, 1.0, 1.7, 4.0, 12.0, 40.0, 150.0])
def test_planck_G_vs_quadrature(oracle_mod, x):
    """G(x) = int_x^inf t^3/(e^t-1) dt against adaptive quadrature (mpmath, 30 digits)."""
    mp.mp.dps = 30
    # scaled by e^x so that mpmath's absolute error control sees O(1) values; fine panels
    xm = mp.mpf(x)
    pts = [xm + k * mp.mpf("0.5") for k in range(161)] + [mp.inf]
    ref = mp.quad(lambda t: t**3 / mp.expm1(t) * mp.exp(xm), pts) * mp.exp(-xm)
    got = oracle_mod.planck_G(x)
    assert abs(got - float(ref)) <= 1e-13 * float(ref)


def test_planck_G_total(oracle_mod):
    assert abs(oracle_mod.planck_G(0.0) - np.pi**4 / 15) < 1e-15
    # continuity across the series switch at x = 1
    a, b = oracle_mod.planck_G(1.0 - 1e-12), oracle_mod.planck_G(1.0)
    assert abs(a - b) < 1e-11


@pytest.mark.parametrize("T,frac", [(100.0, 0.98555), (400.0, 0.99972), (1000.0, 0.99998),
                                    (3000.0, 0.99991), (4798.0, 0.99042)])
def test_planck_band_sum_fraction_of_sigmaT4(oracle_mod, T, frac):
    """sum_b dlam_b pi B_b(T) over 0.3-200 um = sigma T^4 x the blackbody fraction in that band
    (fractions as tabulated in SURVEY.md 8(c); re-derived here by quadrature of the pointwise
    Planck function as well)."""
    from paper_2203_02293_b200.workloads import bin_edges_equal_wavenumber
    edges = bin_edges_equal_wavenumber(30)
    tot = sum((edges[b + 1] - edges[b]) * np.pi * oracle_mod.planck_bin_mean(T, edges[b], edges[b + 1])
              for b in range(30))
    assert abs(tot / (SIGMA * T**4) - frac) < 1.5e-5
    mp.mp.dps = 25
    planck = lambda lam: 2 * H * CL**2 / lam**5 / mp.expm1(H * CL / (lam * KB * T))
    peak = 2.898e-3 / T
    pts = sorted({0.3e-6, 200e-6, *[x for x in (peak / 3, peak, 3 * peak, 10 * peak) if 0.3e-6 < x < 200e-6]})
    ref = mp.pi * mp.quad(planck, pts)
    assert abs(tot - float(ref)) < 1e-11 * float(ref)


def test_planck_all_wavelengths_is_sigmaT4(oracle_mod):
    T = 1500.0
    edges = np.concatenate([[1e-9], np.logspace(-7, -2, 60), [10.0]])
    tot = sum((edges[b + 1] - edges[b]) * np.pi * oracle_mod.planck_bin_mean(T, edges[b], edges[b + 1])
              for b in range(len(edges) - 1))
    assert abs(tot - SIGMA * T**4) < 1e-9 * SIGMA * T**4


def test_planck_narrow_bin_is_pointwise_planck(oracle_mod):
    """A narrow bin's mean equals the textbook B_lambda(T) at its centre (to O(width^2))."""
    for T, lam in [(300.0, 10e-6), (1500.0, 2e-6), (2500.0, 0.5e-6), (150.0, 100e-6)]:
        lo, hi = lam * (1 - 1e-4), lam * (1 + 1e-4)
        ref = 2 * H * CL**2 / lam**5 / np.expm1(H * CL / (lam * KB * T))
        got = oracle_mod.planck_bin_mean(T, lo, hi)
        assert abs(got - ref) < 2e-6 * ref


def test_planck_f64_build_agrees(oracle_mod):
    for T in (120.0, 900.0, 2900.0):
        for lo, hi in [(0.3e-6, 0.31e-6), (1e-6, 1.5e-6), (20e-6, 200e-6)]:
            a, b = oracle_mod.planck_bin_mean(T, lo, hi), oracle_mod.planck_bin_mean(T, lo, hi, real="f64")
            assert abs(a - b) <= 1e-12 * abs(a) + 1e-300


# ----------------------------------------------------------------------------------- interpolation
def _toy_table(rng, nP=5, nT=4, nb=3, ng=2):
    ktab_p = np.sort(10 ** rng.uniform(0, 6, nP))
    ktab_t = np.sort(rng.uniform(200, 2500, nT))
    ktab = np.exp(rng.normal(-9, 2, (nP, nT, nb, ng)))
    return ktab_p, ktab_t, ktab


def test_interp_nodes_and_clamp(oracle_mod):
    rng = np.random.default_rng(1)
    kp, kt, k = _toy_table(rng)
    for ip in range(len(kp)):
        for it in range(len(kt)):
            got = oracle_mod.kappa(kp, kt, k, kp[ip], kt[it], 2, 1)
            assert abs(got - k[ip, it, 2, 1]) <= 1e-14 * k[ip, it, 2, 1]
    # clamped outside the table: equals the edge value
    assert oracle_mod.kappa(kp, kt, k, kp[0] / 50, kt[1], 0, 0) == pytest.approx(k[0, 1, 0, 0], rel=1e-14)
    assert oracle_mod.kappa(kp, kt, k, kp[-1] * 7, kt[-1] + 900, 1, 1) == pytest.approx(k[-1, -1, 1, 1], rel=1e-14)
    assert oracle_mod.kappa(kp, kt, k, kp[2], kt[0] - 100, 1, 0) == pytest.approx(k[2, 0, 1, 0], rel=1e-14)


def test_interp_reproduces_bilinear_lnk(oracle_mod):
    """ln kappa = a + b log10(P) + c T + d log10(P) T is reproduced exactly on a non-uniform grid."""
    rng = np.random.default_rng(2)
    kp, kt, _ = _toy_table(rng)
    a, b, c, d = -8.0, 0.7, 1.1e-3, -2.5e-4
    f = lambda P, T: a + b * np.log10(P) + c * T + d * np.log10(P) * T
    k = np.exp(f(kp[:, None], kt[None, :]))[:, :, None, None] * np.ones((1, 1, 2, 2))
    for _ in range(50):
        P = 10 ** rng.uniform(np.log10(kp[0]), np.log10(kp[-1]))
        T = rng.uniform(kt[0], kt[-1])
        got = oracle_mod.kappa(kp, kt, k, P, T, 1, 0)
        assert abs(np.log(got) - f(P, T)) < 2e-14 * abs(f(P, T))


def test_levels_reading_R9(oracle_mod):
    """Interfaces: midpoints in ln p / mean T inside, half-step extrapolation in ln p and constant T
    at the ends (reading R9)."""
    p = np.array([1e6, 2e5, 5e4, 1e3])
    T = np.array([2000.0, 1500.0, 1200.0, 900.0])
    pi, ti = oracle_mod.levels(p, T)
    assert np.allclose(pi[1:-1], np.sqrt(p[:-1] * p[1:]), rtol=1e-15)
    assert np.allclose(ti[1:-1], 0.5 * (T[:-1] + T[1:]), rtol=1e-15)
    assert pi[0] == pytest.approx(p[0] * np.sqrt(p[0] / p[1]), rel=1e-14)
    assert pi[-1] == pytest.approx(p[-1] / np.sqrt(p[-2] / p[-1]), rel=1e-14)
    assert ti[0] == T[0] and ti[-1] == T[-1]


# --------------------------------------------------------------------------- layer relations vs ODE
def _ode_layer(w0, g0, E, eps2, mu, Fstar, tau_b, dtau, B_b, B_a, Fup_a, Fdn_b):
    """Integrate the two-stream equations (Heng et al. 2018 / Toon et al. 1989 form) across one layer
    from tau_b (top) to tau_a = tau_b + dtau (bottom) and solve the two-point problem by linear
    shooting.  Returns (F_up at top, F_dn at bottom)."""
    ga = 2 * E - w0 * (1 + E * g0)
    gs = w0 * (1 - E * g0)
    g3 = 0.5 * (1 - g0 * mu / eps2) if mu > 0 else 0.0
    g4 = 1 - g3
    Bp = (B_a - B_b) / dtau

    def rhs(tau, y):
        B = B_b + Bp * (tau - tau_b)
        beam = Fstar * np.exp(-tau / mu) if mu > 0 else 0.0
        return [ga * y[0] - gs * y[1] - 2 * np.pi * (1 - w0) * B - g3 * w0 * beam,
                -ga * y[1] + gs * y[0] + 2 * np.pi * (1 - w0) * B + g4 * w0 * beam]

    def shoot(fup_top):
        s = solve_ivp(rhs, [tau_b, tau_b + dtau], [fup_top, Fdn_b], method="DOP853", rtol=1e-13, atol=1e-14)
        return s.y[0, -1], s.y[1, -1]

    u0, d0 = shoot(0.0)
    u1, d1 = shoot(1.0)
    x = (Fup_a - u0) / (u1 - u0)
    return x, d0 + x * (d1 - d0)


@pytest.mark.parametrize("seed", range(12))
@pytest.mark.parametrize("linear_source", [False, True])
def test_layer_relations_match_two_stream_ode(oracle_mod, seed, linear_source):
    """Eqs.(2),(3) [isothermal] and (4),(6) [linear-in-tau source] with (B1),(B2),(B5),(B8) and
    mu_star = -mu reproduce the numerically integrated two-stream ODE (pins signs, Theta, G+-)."""
    rng = np.random.default_rng(100 + seed)
    improved = bool(seed % 2)
    w0 = rng.uniform(0.15, 0.95)
    g0 = rng.uniform(0.0, 0.85)
    eps2 = [2 / 3, 0.5, 1 / np.sqrt(3)][seed % 3]
    mu = rng.uniform(0.15, 1.0) if seed % 4 else -0.3
    dtau_top, dtau = rng.uniform(0.05, 1.0), rng.uniform(0.2, 2.5)
    Fstar, Fup_a, Fdn_b = 7.0, rng.uniform(0, 5), rng.uniform(0, 5)
    B_b, B_a = rng.uniform(0.5, 3), rng.uniform(0.5, 3)
    if not linear_source:
        B_a = B_b
    # two layers; the one under test is the lower one (so that tau at its top is not 0)
    dt = [dtau, dtau_top]
    A, Bm, C, D, fb = oracle_mod.assemble_blocks(dt, [w0, 0.3], [g0, 0.1], [B_a, 1.0], [B_b, 1.0], mu, Fstar,
                                                0.0, improved=improved, linear_source=linear_source, eps2=eps2)
    co = oracle_mod.layer_coeffs(w0, g0, dtau, mu, improved=improved, eps2=eps2)
    chi, xi, psi = Bm[1, 0, 0], Bm[1, 0, 1], -A[1, 0, 0]
    assert (chi, xi, psi) == pytest.approx((co["chi"], co["xi"], co["psi"]), rel=1e-15)
    fup_top = (D[1, 0] + psi * Fup_a - xi * Fdn_b) / chi           # Eq.(2)/(4)
    fdn_bot = (D[0, 1] - Bm[0, 1, 0] * Fup_a + psi * Fdn_b) / Bm[0, 1, 1]   # Eq.(3)/(6)
    ref_up, ref_dn = _ode_layer(w0, g0, co["E"], eps2, mu, Fstar, dtau_top, dtau, B_b, B_a, Fup_a, Fdn_b)
    assert fup_top == pytest.approx(ref_up, rel=2e-10, abs=1e-11)
    assert fdn_bot == pytest.approx(ref_dn, rel=2e-10, abs=1e-11)
    if mu > 0:
        assert fb[1] == pytest.approx(mu * Fstar * np.exp(-dtau_top / mu), rel=1e-14)


# ------------------------------------------------------------------------------- Thomas vs dense LU
def _random_column(rng, L, thick=False):
    dtau = 10 ** rng.uniform(-3, 1.2 if thick else 0.5, L)
    w0 = rng.uniform(0.0, 0.98, L)
    g0 = rng.uniform(0.0, 0.9, L)
    B = rng.uniform(0.2, 4.0, L + 1)
    return dtau, w0, g0, B


def _dense_from_blocks(A, Bm, C, D):
    n = A.shape[0]
    M = np.zeros((2 * n, 2 * n))
    for i in range(n):
        M[2 * i:2 * i + 2, 2 * i:2 * i + 2] = Bm[i]
        if i > 0:
            M[2 * i:2 * i + 2, 2 * i - 2:2 * i] = A[i]
        if i < n - 1:
            M[2 * i:2 * i + 2, 2 * i + 2:2 * i + 4] = C[i]
    return M, D.reshape(-1)


@pytest.mark.parametrize("seed", range(8))
def test_thomas_matches_dense_lu(oracle_mod, seed):
    """Eqs.(13)-(15) on 2x2 blocks == LAPACK LU (partial pivoting) of the assembled matrix."""
    rng = np.random.default_rng(200 + seed)
    L = [3, 6, 10, 17][seed % 4]
    dtau, w0, g0, B = _random_column(rng, L)
    lin = bool(seed % 2)
    mu = 0.7 if seed % 3 else -0.2
    kw = dict(improved=True, linear_source=lin, f_toa=0.3 if seed == 5 else 0.0)
    blo, bhi = (B[:-1], B[1:]) if lin else (B[:-1], B[:-1])
    A, Bm, C, D, fb = oracle_mod.assemble_blocks(dtau, w0, g0, blo, bhi, mu, 5.0, 0.4, **kw)
    M, rhs = _dense_from_blocks(A, Bm, C, D)
    x = np.linalg.solve(M, rhs)
    fu, fd, fb2 = oracle_mod.column_mono(dtau, w0, g0, blo, bhi, mu, 5.0, 0.4, **kw)
    scale = np.abs(x).max()
    assert np.allclose(fu, x[0::2], rtol=0, atol=1e-12 * scale * np.linalg.cond(M) ** 0.5 + 1e-13)
    assert np.allclose(fd, x[1::2], rtol=0, atol=1e-12 * scale * np.linalg.cond(M) ** 0.5 + 1e-13)
    # residual of the oracle's solution in the assembled system (independent of the LU)
    X = np.stack([fu, fd], 1).reshape(-1)
    assert np.abs(M @ X - rhs).max() < 1e-13 * max(1.0, np.abs(rhs).max()) * 10


def test_thomas_structure_of_blocks(oracle_mod):
    """A and C have exactly one non-zero each (-psi), B_0 and B_top carry the boundary rows
    (Eq.10; F_dn,top = F_TOA, L213)."""
    rng = np.random.default_rng(7)
    dtau, w0, g0, B = _random_column(rng, 5)
    A, Bm, C, D, fb = oracle_mod.assemble_blocks(dtau, w0, g0, B[:-1], B[:-1], 0.5, 3.0, 0.7, f_toa=0.11)
    assert np.all(A[:, 0, 1] == 0) and np.all(A[:, 1, :] == 0) and A[0, 0, 0] == 0
    assert np.all(C[:, 0, :] == 0) and np.all(C[:, 1, 0] == 0) and C[-1, 1, 1] == 0
    assert np.array_equal(Bm[0, 0], [1.0, -1.0]) and D[0, 0] == pytest.approx(0.7 + fb[0], rel=1e-15)
    assert np.array_equal(Bm[-1, 1], [0.0, 1.0]) and D[-1, 1] == 0.11
    for s in range(5):
        co = oracle_mod.layer_coeffs(w0[s], g0[s], dtau[s], 0.5)
        assert A[s + 1, 0, 0] == pytest.approx(-co["psi"], rel=1e-15)
        assert C[s, 1, 1] == pytest.approx(-co["psi"], rel=1e-15)
        assert Bm[s + 1, 0] == pytest.approx([co["chi"], co["xi"]], rel=1e-15)
        assert Bm[s, 1] == pytest.approx([co["xi"], co["chi"]], rel=1e-15)


# ----------------------------------------------------- Thomas vs the pair-wise iteration it replaces
def test_thomas_equals_converged_pairwise_iteration(oracle_mod):
    """iterating the two-stream solutions pair-wise over the atmosphere
    (upward sweep with the current F_dn, downward sweep with the current F_up) converges to the
    direct solution."""
    rng = np.random.default_rng(11)
    L = 6
    dtau, w0, g0, B = _random_column(rng, L)
    w0 = np.minimum(w0, 0.9)
    mu, Fstar, Fboa = 0.55, 4.0, 0.3
    A, Bm, C, D, fb = oracle_mod.assemble_blocks(dtau, w0, g0, B[:-1], B[:-1], mu, Fstar, Fboa)
    chi, xi = Bm[1:, 0, 0], Bm[1:, 0, 1]
    psi = -A[1:, 0, 0]
    rhs_up, rhs_dn = D[1:, 0], D[:-1, 1]
    fu, fd = np.zeros(L + 1), np.zeros(L + 1)
    hist = []
    for it in range(400):
        old = np.concatenate([fu, fd])
        fu[0] = fd[0] + Fboa + fb[0]                                  # Eq.(10)
        for s in range(L):                                            # Eq.(2), upward
            fu[s + 1] = (psi[s] * fu[s] - xi[s] * fd[s + 1] + rhs_up[s]) / chi[s]
        fd[L] = 0.0
        for s in range(L - 1, -1, -1):                                # Eq.(3), downward
            fd[s] = (psi[s] * fd[s + 1] - xi[s] * fu[s] + rhs_dn[s]) / chi[s]
        hist.append(np.abs(np.concatenate([fu, fd]) - old).max())
        if hist[-1] < 1e-14 * np.abs(fu).max():
            break
    tu, td, _ = oracle_mod.column_mono(dtau, w0, g0, B[:-1], B[:-1], mu, Fstar, Fboa)
    assert len(hist) > 3            # genuinely iterative: one sweep is not enough
    assert np.allclose(fu, tu, rtol=1e-10, atol=1e-12) and np.allclose(fd, td, rtol=1e-10, atol=1e-12)


# --------------------------------------------------------------------------------- physics limits
def test_pure_absorption_closed_form(oracle_mod):
    """omega0 = 0 (E = 1): zeta+ = 1, zeta- = 0, chi = -1, xi = 0, psi = -T, T = exp(-2 dtau), G = 0;
    beam = mu F* exp(-tau/mu) (Beer's law, L235); diffuse streams decouple (L258)."""
    rng = np.random.default_rng(21)
    L = 9
    dtau = 10 ** rng.uniform(-3, 1, L)
    B = rng.uniform(0.5, 3, L)
    mu, Fstar, Fboa = 0.37, 12.0, 0.8
    for s in range(L):
        co = oracle_mod.layer_coeffs(0.0, 0.0, dtau[s], mu)
        assert co["zeta_p"] == 1 and co["zeta_m"] == 0 and co["chi"] == -1 and co["xi"] == 0
        assert co["psi"] == pytest.approx(-np.exp(-2 * dtau[s]), rel=1e-15)
        assert co["G_p"] == 0 and co["G_m"] == 0 and co["Pi"] == pytest.approx(np.pi, rel=1e-16)
    fu, fd, fb = oracle_mod.column_mono(dtau, np.zeros(L), np.zeros(L), B, B, mu, Fstar, Fboa)
    tau = np.concatenate([np.cumsum(dtau[::-1])[::-1], [0.0]])
    assert np.allclose(fb, mu * Fstar * np.exp(-tau / mu), rtol=1e-13, atol=0)
    tr = np.exp(-2 * dtau)
    ed = np.zeros(L + 1)
    for s in range(L - 1, -1, -1):
        ed[s] = tr[s] * ed[s + 1] + np.pi * B[s] * (1 - tr[s])
    eu = np.zeros(L + 1)
    eu[0] = ed[0] + Fboa + fb[0]
    for s in range(L):
        eu[s + 1] = tr[s] * eu[s] + np.pi * B[s] * (1 - tr[s])
    assert np.allclose(fd, ed, rtol=1e-13, atol=1e-15) and np.allclose(fu, eu, rtol=1e-13, atol=1e-15)


def test_conservative_scattering_conserves_net_flux(oracle_mod):
    """REGULAR closure (E = 1), omega0 = 1 - delta, no thermal source, F_BOA = 0: the total net flux
    (diffuse + beam) is constant with depth and equals F_BOA = 0, up to O(delta tau F*)."""
    delta, Fstar, mu = 1e-8, 5.0, 0.6
    rng = np.random.default_rng(31)
    L = 8
    dtau = rng.uniform(0.05, 1.2, L)
    g0 = rng.uniform(0, 0.8, L)
    fu, fd, fb = oracle_mod.column_mono(dtau, np.full(L, 1 - delta), g0, np.zeros(L), np.zeros(L), mu, Fstar,
                                        0.0, improved=False)
    net = fu - fd - fb
    assert np.abs(net).max() < 100 * delta * Fstar
    assert fu[-1] == pytest.approx(mu * Fstar, rel=1e-5)      # everything that enters leaves at the TOA
    # the improved closure with E > 1 does NOT conserve at omega0 -> 1: the check has teeth
    fu2, fd2, fb2 = oracle_mod.column_mono(dtau, np.full(L, 1 - delta), g0, np.zeros(L), np.zeros(L), mu,
                                           Fstar, 0.0, improved=True)
    assert np.abs(fu2 - fd2 - fb2).max() > 1e-3


def test_opaque_isothermal_limit(oracle_mod):
    """L372-377: an opaque, weakly scattering (omega0 <= 0.1 -> E = 1, Pi = pi) isothermal atmosphere
    without irradiation emits pi B in both directions; net flux 0 two layers below the TOA."""
    L = 8
    B = np.full(L, 2.5)
    fu, fd, fb = oracle_mod.column_mono(np.full(L, 60.0), np.full(L, 0.08), np.full(L, 0.3), B, B, -0.5, 9.0, 0.0)
    assert np.all(fb == 0)
    assert np.allclose(fu[: L - 1], np.pi * 2.5, rtol=1e-12) and np.allclose(fd[: L - 1], np.pi * 2.5, rtol=1e-12)
    assert np.abs((fu - fd)[: L - 1]).max() < 1e-12 * np.pi * 2.5


@pytest.mark.parametrize("mu", [0.45, -1.0])
def test_layer_splitting_is_exact(oracle_mod, mu):
    """The layer relations are exact solutions for a homogeneous isothermal layer: splitting every
    layer in two halves with identical properties leaves the interface fluxes unchanged."""
    rng = np.random.default_rng(41)
    L = 7
    dtau, w0, g0, B = _random_column(rng, L, thick=True)
    fu, fd, fb = oracle_mod.column_mono(dtau, w0, g0, B[:-1], B[:-1], mu, 6.0, 0.2)
    r2 = lambda a: np.repeat(a, 2)
    fu2, fd2, fb2 = oracle_mod.column_mono(r2(dtau) / 2, r2(w0), r2(g0), r2(B[:-1]), r2(B[:-1]), mu, 6.0, 0.2)
    assert np.allclose(fu2[::2], fu, rtol=1e-12, atol=1e-14)
    assert np.allclose(fd2[::2], fd, rtol=1e-12, atol=1e-14)
    assert np.allclose(fb2[::2], fb, rtol=1e-13, atol=0)


def test_linear_source_splitting_is_exact(oracle_mod):
    """Same for the linear-in-tau source (Eqs. 4-9): splitting a sub-layer at its tau-midpoint with the
    Planck value interpolated linearly in tau leaves the solution unchanged."""
    rng = np.random.default_rng(43)
    L = 6
    dtau, w0, g0, B = _random_column(rng, L)
    dtau = np.maximum(dtau, 1e-2)       # keep every half above e_tau
    fu, fd, fb = oracle_mod.column_mono(dtau, w0, g0, B[:-1], B[1:], 0.8, 6.0, 0.2, linear_source=True)
    r2 = lambda a: np.repeat(a, 2)
    mid = 0.5 * (B[:-1] + B[1:])
    blo = np.stack([B[:-1], mid], 1).reshape(-1)
    bhi = np.stack([mid, B[1:]], 1).reshape(-1)
    fu2, fd2, fb2 = oracle_mod.column_mono(r2(dtau) / 2, r2(w0), r2(g0), blo, bhi, 0.8, 6.0, 0.2, linear_source=True)
    assert np.allclose(fu2[::2], fu, rtol=1e-12, atol=1e-14) and np.allclose(fd2[::2], fd, rtol=1e-12, atol=1e-14)


def test_boa_condition(oracle_mod):
    """Eq.(10): F_up0 - F_dn0 = F_BOA + F_beam0, for a column thin enough that the beam reaches
    the bottom."""
    rng = np.random.default_rng(51)
    dtau, w0, g0, B = _random_column(rng, 5)
    dtau *= 0.05
    fu, fd, fb = oracle_mod.column_mono(dtau, w0, g0, B[:-1], B[:-1], 0.9, 10.0, 1.25)
    assert fb[0] > 1.0
    assert fu[0] - fd[0] == pytest.approx(1.25 + fb[0], rel=1e-13)
    assert fd[-1] == 0.0


def test_f_toa_option(oracle_mod):
    """Fig. 5 caption (L213): the diffuse TOA flux option is the downward flux at the top level."""
    rng = np.random.default_rng(52)
    dtau, w0, g0, B = _random_column(rng, 4)
    fu, fd, fb = oracle_mod.column_mono(dtau, w0, g0, B[:-1], B[:-1], -1.0, 0.0, 0.0, f_toa=0.77)
    assert fd[-1] == pytest.approx(0.77, rel=1e-15)


# ------------------------------------------------------------------------------------------ guards
def test_E_branches(oracle_mod):
    """Eq.(19): strict omega0 > 0.1 for the fit (R6); regular mode E = 1; E <- max(1, fit) (R5)."""
    fit = lambda w, g: 1.225 - 0.1582 * g - 0.1777 * w - 0.07465 * g * g + 0.2351 * w * g - 0.05582 * w * w
    assert oracle_mod.layer_coeffs(0.1, 0.5, 1.0, -1)["E"] == 1.0
    assert oracle_mod.layer_coeffs(0.1000001, 0.5, 1.0, -1)["E"] == pytest.approx(fit(0.1000001, 0.5), rel=1e-15)
    assert oracle_mod.layer_coeffs(0.6, 0.5, 1.0, -1)["E"] == pytest.approx(1.0710523, rel=1e-12)
    assert oracle_mod.layer_coeffs(0.6, 0.5, 1.0, -1, improved=False)["E"] == 1.0
    assert fit(0.999, 0.0) < 0.999                     # the raw fit would make E - omega0 negative
    co = oracle_mod.layer_coeffs(0.999, 0.0, 1.0, -1)
    assert co["E"] == 1.0 and np.isfinite(co["chi"]) and co["Pi"] == pytest.approx(np.pi, rel=1e-12)


def test_mu_crit_guard(oracle_mod):
    """Eq.(11), L247-254 (reading R4): |4 E mu^2 (E-w0)(1-w0 g0) - 1| < 1e-5 -> the term becomes
    2 mu_star = -2 mu; G+- stay finite and equal (B8) evaluated with that replacement."""
    w0, g0, eps2 = 0.5, 0.3, 2 / 3
    E = oracle_mod.layer_coeffs(w0, g0, 1.0, -1)["E"]
    mu_crit = 1 / (2 * np.sqrt(E * (E - w0) * (1 - w0 * g0)))
    assert 0 < mu_crit < 1
    co = oracle_mod.layer_coeffs(w0, g0, 1.0, mu_crit)
    P = 2 * E * (1 - w0 * g0)
    mustar = -mu_crit
    lead = w0 * (P + g0 / eps2) / (2 * mustar)
    assert co["G_p"] == pytest.approx(0.5 * (lead * (mustar + 1 / P) + w0 * g0 / (eps2 * P)), rel=1e-12)
    assert co["G_m"] == pytest.approx(0.5 * (lead * (mustar - 1 / P) - w0 * g0 / (eps2 * P)), rel=1e-12)
    # just outside the guard the full term is used (large but finite, different value)
    co2 = oracle_mod.layer_coeffs(w0, g0, 1.0, mu_crit * (1 + 1e-4))
    assert abs(co2["G_p"]) > 100 * abs(co["G_p"])
    # a small tolerance switches the guard off
    co3 = oracle_mod.layer_coeffs(w0, g0, 1.0, mu_crit * (1 + 1e-7), gcrit_tol=1e-12)
    assert abs(co3["G_p"]) > 1e4


def test_nightside_has_no_beam(oracle_mod):
    for mu in (0.0, -0.4):
        co = oracle_mod.layer_coeffs(0.7, 0.4, 0.5, mu)
        assert co["G_p"] == 0 and co["G_m"] == 0
        fu, fd, fb = oracle_mod.column_mono([0.5, 0.2], [0.7, 0.2], [0.4, 0.0], [1.0, 2.0], [1.0, 2.0], mu, 50.0, 0.0)
        assert np.all(fb == 0)


def test_e_tau_rule(oracle_mod):
    """L209/L223 (reading R15): a sub-layer thinner than e_tau drops the gradient term and uses the mean
    Planck value; the switch is strict '<'."""
    kw = dict(improved=True, linear_source=True)
    args = lambda dt: ([dt, 0.3], [0.4, 0.2], [0.2, 0.1], [2.0, 1.5], [1.0, 1.2], -1.0, 0.0, 0.0)
    thin = oracle_mod.column_mono(*args(0.99e-4), **kw)
    iso_mean = oracle_mod.column_mono([0.99e-4, 0.3], [0.4, 0.2], [0.2, 0.1], [1.5, 1.5], [1.5, 1.2], -1.0, 0.0, 0.0, **kw)
    assert np.allclose(thin[0], iso_mean[0], rtol=1e-14) and np.allclose(thin[1], iso_mean[1], rtol=1e-14)
    # with the rule switched off (e_tau = 0) the same thin layer gives a (slightly) different answer
    off = oracle_mod.column_mono(*args(0.99e-4), e_tau=0.0, **kw)
    assert not np.allclose(thin[1], off[1], rtol=1e-9, atol=0)


# --------------------------------------------------------------------------------- worked example
def test_worked_example_golden(oracle_mod):
    g = _golden()
    for i in range(3):
        co = oracle_mod.layer_coeffs(g["w0"][i], g["g0"][i], g["dtau"][i], 0.6)
        for k, name in (("imp_E", "E"), ("imp_chi", "chi"), ("imp_xi", "xi"), ("imp_psi", "psi"), ("imp_Pi", "Pi"),
                        ("imp_Gp", "G_p"), ("imp_Gm", "G_m")):
            assert co[name] == pytest.approx(g[k][i], rel=2e-12), (k, i)
    fu, fd, fb = oracle_mod.column_mono(g["dtau"], g["w0"], g["g0"], g["B_iso"], g["B_iso"], 0.6, 10.0, 0.25)
    assert np.allclose(fb, g["F_beam"], rtol=1e-12) and np.allclose(fu, g["imp_F_up"], rtol=1e-12)
    assert np.allclose(fd, g["imp_F_dn"], rtol=1e-12, atol=1e-15)
    assert np.allclose(fu - fd - fb, g["imp_F_net"], rtol=1e-11)
    fu, fd, fb = oracle_mod.column_mono(g["dtau"], g["w0"], g["g0"], g["B_iso"], g["B_iso"], 0.6, 10.0, 0.25,
                                        improved=False)
    assert np.allclose(fu, g["reg_F_up"], rtol=1e-12) and np.allclose(fd, g["reg_F_dn"], rtol=1e-12, atol=1e-15)
    r2 = lambda a: np.repeat(a, 2)
    fu, fd, fb = oracle_mod.column_mono(r2(g["dtau"]) / 2, r2(g["w0"]), r2(g["g0"]), g["B_levels"][:-1],
                                        g["B_levels"][1:], 0.6, 10.0, 0.25, linear_source=True)
    assert np.allclose(fu[::2], g["ni_F_up_int"], rtol=1e-12) and np.allclose(fd[::2], g["ni_F_dn_int"], rtol=1e-12, atol=1e-15)
    assert np.allclose(fu[1::2], g["ni_F_up_cen"], rtol=1e-12) and np.allclose(fd[1::2], g["ni_F_dn_cen"], rtol=1e-12)


def test_worked_example_mpmath():
    """Re-derive the golden isothermal values at 40 digits from Eqs.(2),(3),(10),(19),(B1),(B2),(B5),
    (B6),(B8) with a dense scalar LU -- neither the oracle nor the CUDA path is involved."""
    mp.mp.dps = 40
    g = _golden()
    mu, Fs, Fboa, eps2 = mp.mpf("0.6"), mp.mpf(10), mp.mpf("0.25"), mp.mpf(2) / 3
    dt = [mp.mpf("2.0"), mp.mpf("0.5"), mp.mpf("0.05")]
    w = [mp.mpf("0.05"), mp.mpf("0.6"), mp.mpf("0.9")]
    gg = [mp.mpf(0), mp.mpf("0.5"), mp.mpf("0.8")]
    B = [mp.mpf(3), mp.mpf(2), mp.mpf(1)]
    L = 3
    tau = [sum(dt[s:]) for s in range(L)] + [mp.mpf(0)]
    fb = [mu * Fs * mp.e ** (-t / mu) for t in tau]
    M = mp.zeros(2 * (L + 1))
    r = mp.zeros(2 * (L + 1), 1)
    up = lambda i: 2 * i
    dn = lambda i: 2 * i + 1
    M[0, up(0)], M[0, dn(0)], r[0] = 1, -1, Fboa + fb[0]
    M[1, dn(L)], r[1] = 1, 0
    row = 2
    for s in range(L):
        E = mp.mpf(1)
        if w[s] > mp.mpf("0.1"):
            E = (mp.mpf("1.225") - mp.mpf("0.1582") * gg[s] - mp.mpf("0.1777") * w[s] - mp.mpf("0.07465") * gg[s] ** 2
                 + mp.mpf("0.2351") * w[s] * gg[s] - mp.mpf("0.05582") * w[s] ** 2)
            E = max(E, mp.mpf(1))
        root = mp.sqrt((E - w[s]) / (E * (1 - w[s] * gg[s])))
        zp, zm = (1 + root) / 2, (1 - root) / 2
        T = mp.e ** (-2 * mp.sqrt(E * (E - w[s]) * (1 - w[s] * gg[s])) * dt[s])
        chi, xi, psi = zm**2 * T**2 - zp**2, zp * zm * (1 - T**2), (zm**2 - zp**2) * T
        Pi = mp.pi * (1 - w[s]) / (E - w[s])
        P = 2 * E * (1 - w[s] * gg[s])
        ms = -mu
        Dn = 4 * E * ms**2 * (E - w[s]) * (1 - w[s] * gg[s]) - 1
        lead = w[s] * (P + gg[s] / eps2) / Dn
        Gp = (lead * (ms + 1 / P) + w[s] * gg[s] / (eps2 * P)) / 2
        Gm = (lead * (ms - 1 / P) - w[s] * gg[s] / (eps2 * P)) / 2
        # Eq.(2): chi Fup[s+1] - psi Fup[s] + xi Fdn[s+1] = ...
        M[row, up(s + 1)], M[row, up(s)], M[row, dn(s + 1)] = chi, -psi, xi
        r[row] = Pi * B[s] * (chi + xi - psi) + psi * Gp * fb[s] - (xi * Gm + chi * Gp) * fb[s + 1]
        row += 1
        # Eq.(3): chi Fdn[s] - psi Fdn[s+1] + xi Fup[s] = ...
        M[row, dn(s)], M[row, dn(s + 1)], M[row, up(s)] = chi, -psi, xi
        r[row] = Pi * B[s] * (chi + xi - psi) + psi * Gm * fb[s + 1] - (xi * Gp + chi * Gm) * fb[s]
        row += 1
    x = mp.lu_solve(M, r)
    for i in range(L + 1):
        assert abs(float(x[up(i)]) - g["imp_F_up"][i]) < 1e-13 * 10
        assert abs(float(x[dn(i)]) - g["imp_F_dn"][i]) < 1e-13 * 10
        assert abs(float(fb[i]) - g["F_beam"][i]) < 1e-14 * 10


# -------------------------------------------------------------------------- full step plumbing (O1-O9)
def test_full_step_equals_manual_composition(oracle_mod):
    """oracle.rt_step == levels -> kappa -> optics -> Planck -> column_mono -> weighted sums composed
    by hand in numpy for one column (pins indexing, weights, the beam bookkeeping of L235 and the
    heating-rate reading R14)."""
    from paper_2203_02293_b200 import workloads as W
    for config, col in ((1, 5), (1, 0)):
        cfg, inp, meta = W.make(config)
        for flags in (W.IMPROVED, W.IMPROVED | W.NONISOTHERMAL):
            cfg = dict(cfg, flags=flags, cloud_ext=np.full(meta["n_bins"], 3e-4), cloud_w0=np.linspace(0.2, 0.9, meta["n_bins"]),
                       cloud_g0=np.linspace(0.1, 0.7, meta["n_bins"]), cloud_p_top=1e2, cloud_p_bot=1e5)
            one = dict(inp, p=inp["p"][col:col + 1], T=inp["T"][col:col + 1], mu_star=np.abs(inp["mu_star"][col:col + 1]))
            res = oracle_mod.rt_step(cfg, one, dbg_column=0)
            N, nb, ng = meta["n_layers"], meta["n_bins"], meta["n_gauss"]
            p, T, mu = one["p"][0], one["T"][0], one["mu_star"][0]
            p_int, T_int = oracle_mod.levels(p, T)
            noniso = bool(flags & W.NONISOTHERMAL)
            if noniso:
                pl = np.empty(2 * N + 1); tl = np.empty(2 * N + 1)
                pl[0::2], pl[1::2], tl[0::2], tl[1::2] = p_int, p, T_int, T
            else:
                pl, tl = p, T
            T_internal = (one["f_internal"] / SIGMA) ** 0.25
            up = np.zeros(N + 1); dn = np.zeros(N + 1); bm = np.zeros(N + 1); toa = np.zeros(nb)
            for b in range(nb):
                lo, hi = cfg["bin_edges"][b], cfg["bin_edges"][b + 1]
                Bl = np.array([oracle_mod.planck_bin_mean(t, lo, hi) for t in tl])
                Fboa = np.pi * oracle_mod.planck_bin_mean(T_internal, lo, hi)
                for g in range(ng):
                    ka = np.array([oracle_mod.kappa(cfg["ktab_p"], cfg["ktab_t"], cfg["ktab"], pp, tt, b, g) for pp, tt in zip(pl, tl)])
                    cl = (pl >= cfg["cloud_p_top"]) & (pl <= cfg["cloud_p_bot"])
                    kc = np.where(cl, cfg["cloud_ext"][b], 0.0)
                    sc = kc * cfg["cloud_w0"][b]
                    sg = cfg["scat_gas"][b]
                    kx = ka + sg + kc
                    w0 = (sg + sc) / kx
                    g0 = sc * cfg["cloud_g0"][b] / (sg + sc)
                    if noniso:
                        dm = (pl[:-1] - pl[1:]) / cfg["gravity"]
                        dtau = 0.5 * (kx[:-1] + kx[1:]) * dm
                        fu, fd, fb = oracle_mod.column_mono(dtau, 0.5 * (w0[:-1] + w0[1:]), 0.5 * (g0[:-1] + g0[1:]),
                                                            Bl[:-1], Bl[1:], mu, one["stellar_flux"][b], Fboa,
                                                            linear_source=True)
                        fu, fd, fb = fu[::2], fd[::2], fb[::2]
                    else:
                        dm = (p_int[:-1] - p_int[1:]) / cfg["gravity"]
                        fu, fd, fb = oracle_mod.column_mono(kx * dm, w0, g0, Bl, Bl, mu, one["stellar_flux"][b], Fboa)
                    wgt = (hi - lo) * cfg["gauss_w"][g]
                    up += wgt * fu; dn += wgt * (fd + fb); bm += wgt * fb
                    toa[b] += cfg["gauss_w"][g] * fu[-1]
                    assert np.allclose(res["dbg_F_up_pt"][:, b * ng + g], fu, rtol=1e-12)
            assert np.allclose(res["F_up"][0], up, rtol=1e-12) and np.allclose(res["F_down"][0], dn, rtol=1e-12)
            assert np.allclose(res["F_beam"][0], bm, rtol=1e-12, atol=1e-300) and np.allclose(res["F_up_toa_bin"][0], toa, rtol=1e-12)
            assert np.allclose(res["F_net"][0], up - dn, rtol=1e-9, atol=1e-9 * np.abs(up).max())
            dmf = (p_int[:-1] - p_int[1:]) / cfg["gravity"]
            assert np.allclose(res["dTdt"][0], -np.diff(res["F_net"][0]) / (cfg["cp"] * dmf), rtol=1e-6, atol=1e-12)


def test_full_step_opaque_isothermal_atmosphere(oracle_mod):
    """north_star pin: isothermal, optically thick atmosphere, no irradiation: F_up = F_down =
    sum_b dlam_b pi B_b(T) and the heating rate vanishes (deep layers)."""
    from paper_2203_02293_b200 import workloads as W
    cfg, inp, meta = W.make(1)
    cfg = dict(cfg, ktab=cfg["ktab"] * 1e6, scat_gas=cfg["scat_gas"] * 1e3)      # tau >> 1 per layer, w0 <= 0.1
    T0 = 1234.0
    one = dict(inp, p=inp["p"][:2], T=np.full((2, meta["n_layers"]), T0), mu_star=np.array([-1.0, 0.0]), f_internal=0.0)
    for flags in (W.IMPROVED, W.IMPROVED | W.NONISOTHERMAL):
        res = oracle_mod.rt_step(dict(cfg, flags=flags), one)
        e = cfg["bin_edges"]
        ref = sum((e[b + 1] - e[b]) * np.pi * oracle_mod.planck_bin_mean(T0, e[b], e[b + 1]) for b in range(meta["n_bins"]))
        # the top three layers of this column are not opaque (dtau falls with pressure): check below them
        assert np.allclose(res["F_up"][:, :-3], ref, rtol=1e-12) and np.allclose(res["F_down"][:, :-3], ref, rtol=1e-12)
        dm = np.abs(np.diff(oracle_mod.levels(one["p"][0], one["T"][0])[0])) / cfg["gravity"]
        assert np.all(np.abs(res["dTdt"][:, :-4]) <= 1e-12 * ref / (cfg["cp"] * dm[:-4]))


# ---------------------------------------------------------------- round 2: pins that are not restatements
# level_optics (Eqs. 17-18), the sub-layer means (L171, reading R10) and the heating rate
# (L393 / L1032, reading R14) were only checked against numpy re-typings of the same expressions.  The tests
# below start from what the paper prints (number densities and cross sections; the sentence of L171; energy
# conservation and Beer's law) and each names the planted mistake it fails on.

AMU = 1.66053906660e-27


def _optics_cfg(kappa, scat_gas, cloud_ext, cloud_w0, cloud_g0, p_top=1e2, p_bot=1e5, nb=1, ng=1):
    """A k-table that is constant in (P, T): kappa_abs = `kappa` at every level."""
    return dict(ktab_p=np.array([1.0, 1e7]), ktab_t=np.array([100.0, 3000.0]),
                ktab=np.broadcast_to(np.asarray(kappa, dtype=float).reshape(1, 1, nb, ng), (2, 2, nb, ng)).copy(),
                bin_edges=np.linspace(1e-6, 2e-6, nb + 1), gauss_w=np.full(ng, 1.0 / ng),
                scat_gas=np.full(nb, scat_gas), cloud_ext=np.full(nb, cloud_ext), cloud_w0=np.full(nb, cloud_w0),
                cloud_g0=np.full(nb, cloud_g0), cloud_p_top=p_top, cloud_p_bot=p_bot, gravity=10.0, cp=1e4, flags=1)


def test_eq17_eq18_from_number_density_form(oracle_mod):
    """Eqs.(17),(18) as printed: cross sections per particle weighted by number densities,
        w0 = (sig_scat,gas + f sig_scat,cloud) / (sig_scat,gas + kappa mbar + f (sig_abs,cloud + sig_scat,cloud)),
        g0 = f sig_scat,cloud / (sig_scat,gas + f sig_scat,cloud) * g0,cloud,
    evaluated at 40 digits from hand numbers; the library inputs are those numbers divided by mbar
    (include/helios_rt.h: scat_gas = sig_scat,gas / mbar, cloud_ext = f (sig_abs + sig_scat)_cloud / mbar,
    cloud_w0 = sig_scat / (sig_abs + sig_scat)).  Planted mistakes that fail here: s_c <-> k_c (cloud extinction
    instead of cloud scattering in either numerator), kappa_abs missing from / doubled in the denominator,
    g0 weighted by the extinction instead of the scattering fraction."""
    mp.mp.dps = 40
    mbar = mp.mpf("2.34") * mp.mpf(AMU)                      # L348: 2.34 amu
    sig_gas = mp.mpf("2.0e-31")                              # m^2 per gas particle
    kap = mp.mpf("5.0e-5")                                   # m^2 / kg
    f = mp.mpf("1e-17")                                      # L364
    sig_abs, sig_sca, g_cl = mp.mpf("1.0e-12"), mp.mpf("3.0e-12"), mp.mpf("0.6")
    w0_ref = (sig_gas + f * sig_sca) / (sig_gas + kap * mbar + f * (sig_abs + sig_sca))
    g0_ref = f * sig_sca / (sig_gas + f * sig_sca) * g_cl
    kext_ref = (sig_gas + kap * mbar + f * (sig_abs + sig_sca)) / mbar
    cfg = _optics_cfg(float(kap), float(sig_gas / mbar), float(f * (sig_abs + sig_sca) / mbar),
                      float(sig_sca / (sig_abs + sig_sca)), float(g_cl))
    kx, w0, g0 = oracle_mod.level_optics(cfg, 1e4, 1000.0, 0, 0)            # inside the cloud deck
    assert abs(w0 - float(w0_ref)) <= 1e-14 * float(w0_ref)
    assert abs(g0 - float(g0_ref)) <= 1e-14 * float(g0_ref)
    assert abs(kx - float(kext_ref)) <= 1e-14 * float(kext_ref)
    # the hand numbers make the planted mistakes visible: scattering vs extinction differ by 4/3
    assert abs(float((sig_gas + f * (sig_abs + sig_sca)) / (sig_gas + kap * mbar + f * (sig_abs + sig_sca))) - w0) > 0.05
    # outside the deck (p < cloud_p_top or p > cloud_p_bot) the cloud terms drop out: f = 0 in Eqs.(17),(18)
    for p_out in (50.0, 2e5):
        kx, w0, g0 = oracle_mod.level_optics(cfg, p_out, 1000.0, 0, 0)
        assert g0 == 0.0
        assert abs(w0 - float(sig_gas / (sig_gas + kap * mbar))) <= 1e-14 * w0
        assert abs(kx - float((sig_gas + kap * mbar) / mbar)) <= 1e-14 * kx
    # deck edges are inclusive (include/helios_rt.h: cloud_p_top <= p <= cloud_p_bot)
    assert oracle_mod.level_optics(cfg, 1e2, 1000.0, 0, 0)[2] > 0 and oracle_mod.level_optics(cfg, 1e5, 1000.0, 0, 0)[2] > 0


def test_eq17_eq18_limits(oracle_mod):
    """Limits of Eqs.(17),(18): no gas scattering => g0 = g0,cloud exactly and w0 = cloud_w0 k_c / (kappa + k_c);
    no cloud (cloud_ext = 0) => g0 = 0 and w0 = s / (kappa + s); purely scattering cloud without gas absorption
    would give w0 -> 1.  A g0 weighted with the extinction instead of the scattering fraction fails the first."""
    cfg = _optics_cfg(2e-3, 0.0, 6e-3, 0.25, 0.7)
    kx, w0, g0 = oracle_mod.level_optics(cfg, 1e4, 500.0, 0, 0)
    assert g0 == 0.7
    assert abs(w0 - 0.25 * 6e-3 / 8e-3) < 1e-15 and abs(kx - 8e-3) < 1e-17
    cfg = _optics_cfg(2e-3, 5e-4, 0.0, 0.9, 0.7)
    kx, w0, g0 = oracle_mod.level_optics(cfg, 1e4, 500.0, 0, 0)
    assert g0 == 0.0 and abs(w0 - 0.2) < 1e-15 and abs(kx - 2.5e-3) < 1e-17
    # gas and cloud scattering equal => g0 is exactly half the cloud's (number-density weighting of Eq. 18)
    cfg = _optics_cfg(1e-3, 3e-3, 6e-3, 0.5, 0.8)
    assert abs(oracle_mod.level_optics(cfg, 1e4, 500.0, 0, 0)[2] - 0.4) < 1e-15


def test_sublayer_means_are_means_of_final_quantities(oracle_mod):
    """Reading R10 of L171 ("their values in the upper and lower sub-layers are taken to be the arithmetic mean of
    their central and interface values", said of the opacities AND the single-scattering albedos): a two-layer
    hand example in which the mean of w0 differs from the w0 of the mean ingredients.  Level values (typed by hand):
        kappa_abs = 1, 3, 9, 27, 81 e-3 at the five levels (bottom interface, centre 0, interface 1, centre 1, top),
        gas scattering 1e-3, no cloud  =>  kappa_ext = 2, 4, 10, 28, 82 e-3;  w0 = 1/2, 1/4, 1/10, 1/28, 1/82
        sub-layer means   kappa_ext: 3, 7, 19, 55 e-3     w0: 3/8, 7/40, 19/280, 55/2296
        (ingredient averaging would give w0 = 1/3, 1/7, 1/19, 1/55 instead.)
    The full step must equal column_mono (pinned by the ODE / LU / worked-example tests) fed with the hand values;
    it must NOT equal column_mono fed with the ingredient-averaged albedos."""
    sq = np.sqrt(10.0)
    p = np.array([[1e5, 1e4]])
    p_lev = np.array([1e5 * sq, 1e5, np.sqrt(1e9), 1e4, 1e4 / sq])          # reading R9, pinned by test_levels_*
    kap = np.array([1.0, 3.0, 9.0, 27.0, 81.0]) * 1e-3
    order = np.argsort(p_lev)
    cfg = dict(ktab_p=p_lev[order], ktab_t=np.array([100.0, 3000.0]),
               ktab=np.repeat(kap[order].reshape(5, 1, 1, 1), 2, axis=1).copy(),
               bin_edges=np.array([1e-6, 2e-6]), gauss_w=np.array([1.0]), scat_gas=np.array([1e-3]),
               cloud_ext=np.array([0.0]), cloud_w0=np.array([0.0]), cloud_g0=np.array([0.0]), cloud_p_top=1.0,
               cloud_p_bot=2.0, gravity=10.0, cp=1e4, flags=1 | 2)
    T = np.array([[1500.0, 900.0]])
    inp = dict(p=p, T=T, mu_star=np.array([0.7]), stellar_flux=np.array([3e9]), f_internal=0.0)
    res = oracle_mod.rt_step(cfg, inp, want=("F_up", "F_down", "F_beam"))
    dm = (p_lev[:-1] - p_lev[1:]) / 10.0
    kx_mean = np.array([3.0, 7.0, 19.0, 55.0]) * 1e-3
    w_mean = np.array([3 / 8, 7 / 40, 19 / 280, 55 / 2296])
    w_ingr = np.array([1 / 3, 1 / 7, 1 / 19, 1 / 55])
    T_lev = np.array([1500.0, 1500.0, 1200.0, 900.0, 900.0])                # reading R9: ends held, interior mean
    B = np.array([oracle_mod.planck_bin_mean(t, 1e-6, 2e-6) for t in T_lev])
    dlam = 1e-6

    def mono(w):
        fu, fd, fb = oracle_mod.column_mono(kx_mean * dm, w, np.zeros(4), B[:-1], B[1:], 0.7, 3e9, 0.0, linear_source=True)
        return dlam * fu[::2], dlam * (fd + fb)[::2]

    up, dn = mono(w_mean)
    assert np.allclose(res["F_up"][0], up, rtol=1e-12) and np.allclose(res["F_down"][0], dn, rtol=1e-12)
    up_bad, dn_bad = mono(w_ingr)
    assert np.max(np.abs(res["F_up"][0] - up_bad) / np.abs(up)) > 1e-3        # the other reading is far away
    # the same for the opacity: kappa_ext of a sub-layer is the mean of the two level values (not e.g. the
    # geometric mean or the lower level's value): tau at the bottom from the beam, Eq.(B6)
    tau0 = -0.7 * np.log(res["F_beam"][0, 0] / (dlam * 0.7 * 3e9))
    assert abs(tau0 - float(np.sum(kx_mean * dm))) <= 1e-11 * tau0


def _beam_only_case(nb=2, ng=2):
    """Cold, purely absorbing column under the stellar beam only, opaque at the bottom."""
    N = 12
    p = np.logspace(5, 0.5, N)[None, :]
    kap = np.array([[2e-3, 8e-3], [5e-4, 3e-2]])[:nb, :ng]
    cfg = _optics_cfg(kap, 0.0, 0.0, 0.0, 0.0, nb=nb, ng=ng)
    cfg["bin_edges"] = np.array([0.4e-6, 0.9e-6, 2.5e-6])[:nb + 1]       # x = hc/(lam k T) > 100 at T = 50 K: B = 0
    cfg["gauss_w"] = np.array([0.35, 0.65])[:ng] if ng == 2 else np.array([1.0])
    inp = dict(p=p, T=np.full((1, N), 50.0), mu_star=np.array([0.05]), stellar_flux=np.array([4e11, 1.5e11])[:nb],
               f_internal=0.0)
    return cfg, inp, N, kap


def test_heating_rate_energy_closure(oracle_mod):
    """Reading R14 (L393, L1032: the heating term 'depends on the spatial gradient of the net flux'): whatever the
    column, the energy deposited per unit area and time, sum_j c_P dm_j dT/dt_j, must equal what enters through the
    boundaries, F_net[0] - F_net[N] (F_net positive upward): energy conservation, not a re-typing of the difference
    formula.  dm_j comes from the separately pinned interface pressures.  Fails on: sign flip of dT/dt, dm of the
    wrong layer (j+1 or the sub-layer), a missing 1/c_P or 1/g, F_net differenced across two layers."""
    from paper_2203_02293_b200 import workloads as W
    cfg, inp, meta = W.make(1)
    for flags in (W.IMPROVED, W.IMPROVED | W.NONISOTHERMAL):
        c = dict(cfg, flags=flags)
        sub = dict(inp, p=inp["p"][:6], T=inp["T"][:6], mu_star=inp["mu_star"][:6])
        res = oracle_mod.rt_step(c, sub, want=("F_net", "dTdt"))
        for k in range(6):
            p_int, _ = oracle_mod.levels(sub["p"][k], sub["T"][k])
            dm = (p_int[:-1] - p_int[1:]) / c["gravity"]
            dep = np.sum(c["cp"] * dm * res["dTdt"][k])
            scale = np.sum(np.abs(c["cp"] * dm * res["dTdt"][k]))
            assert abs(dep - (res["F_net"][k, 0] - res["F_net"][k, -1])) <= 1e-12 * scale
            # and layer by layer the deposited power is the flux convergence (sign: net upward flux leaving > entering cools)
            assert np.allclose(c["cp"] * dm * res["dTdt"][k], res["F_net"][k, :-1] - res["F_net"][k, 1:], rtol=1e-10,
                               atol=1e-13 * scale)


def test_heating_rate_beam_only_closed_form(oracle_mod):
    """Sign AND scale of dT/dt from a closed form: cold (B = 0), purely absorbing (w0 = 0), no internal flux, opaque at
    the bottom (so the BOA reflection of Eq. 10 returns nothing): the only flux is the direct beam of Eq.(B6) /
    Beer's law (L235), F_net = -sum_b dlam_b sum_g w_g mu F*_b exp(-tau/mu), so every layer is HEATED by
        dT/dt_j = sum_b dlam_b sum_g w_g mu F*_b (exp(-tau_{j+1}/mu) - exp(-tau_j/mu)) / (c_P dm_j)  > 0,
    tau_j = kappa (p_int,j - p_int,N) / g.  Evaluated at 30 digits.  Fails on: sign flip, dm of a neighbouring
    layer, missing c_P, dlam or w_g weights dropped, beam not counted in F_down (L235)."""
    mp.mp.dps = 30
    cfg, inp, N, kap = _beam_only_case()
    for flags in (1, 1 | 2):
        res = oracle_mod.rt_step(dict(cfg, flags=flags), inp, want=("F_up", "F_net", "dTdt"))
        p_int, _ = oracle_mod.levels(inp["p"][0], inp["T"][0])
        mu, g, cp = mp.mpf(inp["mu_star"][0]), mp.mpf(10), mp.mpf(1e4)
        pi = [mp.mpf(float(x)) for x in p_int]
        ref = []
        for j in range(N):
            acc = mp.mpf(0)
            for b in range(2):
                dlam = mp.mpf(float(cfg["bin_edges"][b + 1])) - mp.mpf(float(cfg["bin_edges"][b]))
                for gq in range(2):
                    k = mp.mpf(float(kap[b, gq]))
                    t_hi, t_lo = k * (pi[j + 1] - pi[N]) / g, k * (pi[j] - pi[N]) / g
                    acc += dlam * mp.mpf(float(cfg["gauss_w"][gq])) * mu * mp.mpf(float(inp["stellar_flux"][b])) * \
                        (mp.e ** (-t_hi / mu) - mp.e ** (-t_lo / mu))
            ref.append(acc / (cp * (pi[j] - pi[j + 1]) / g))
        ref = np.array([float(r) for r in ref])
        assert np.all(ref > 0) and ref.max() > 1e-3                         # a real heating profile
        assert np.all(res["dTdt"][0] > 0)
        # (kappa is constant with depth, so the non-isothermal sub-layer treatment must give the same profile)
        assert np.allclose(res["dTdt"][0], ref, rtol=1e-11, atol=1e-14 * ref.max())
        assert np.all(np.abs(res["F_up"][0]) <= 1e-40)                        # nothing comes back up (B(50 K) ~ 1e-46)


def test_opcount_build_matches_the_oracle_and_counts(oracle_mod):
    """oracle/opcount.py compiles helios_oracle.c unchanged with an op-counting scalar (BASELINE.md section 3's audit):
    its results equal the long-double build's, and the counts per layer.point are what BASELINE.md quotes (every
    dayside layer.point takes 3 exponentials in the method -- kappa is tabulated, so the oracle's 4th is Planck's share --
    and at least 2 square roots and 16 divisions in the literal form)."""
    import ctypes as C
    from oracle import opcount
    from paper_2203_02293_b200 import workloads as W
    per = opcount.count(2, True, n_cols=2)
    assert 3.0 <= per["exp"] <= 4.5 and per["sqrt"] == 2.0 and per["div"] >= 16 and per["log"] == 8.0
    night = opcount.count(2, False, n_cols=2)
    assert night["exp"] < per["exp"] and night["div"] < per["div"]          # no direct beam: fewer of both
    cfg, inp, meta = W.make(1)
    a = oracle_mod.rt_step(cfg, inp, real="opcount", want=("F_net", "dTdt"))
    b = oracle_mod.rt_step(cfg, inp, real="ld", want=("F_net", "dTdt"))
    for k in a:
        assert np.array_equal(a[k], b[k]), k


# ---------------------------------------------------------------- round 3: the last two unpinned parts
# (a) the per-bin TOA spectrum F_up_toa_bin[b] = sum_g w_g F_up[N](b, g) -- the
#     only output of config 5 and of the post-processing step -- was checked by a numpy re-typing of its own line only;
# (b) the interfaces of a single-layer column (reading R27) by nothing.
# Planted mistakes these fail on: "toa_bin += dlam * w_g * Fu", "toa_bin += Fu" (w_g dropped), "Fu[N]" for
# "Fu[N * stride]" on non-isothermal columns, sqrt(10) -> any other factor in levels().

@pytest.mark.parametrize("config", [1, 5])
@pytest.mark.parametrize("noniso", [False, True])
def test_toa_spectrum_integrates_to_the_toa_flux(oracle_mod, config, noniso):
    """sum_b dlam_b F_up_toa_bin[c, b] = F_up[c, N]: the left side goes through the per-bin accumulation, the right
    through the interface accumulation that the closed-form pins above cover (pure absorption, opaque limit, energy
    closure).  Non-isothermal columns have 2N + 1 levels per point: the TOA is level 2N, not N."""
    from paper_2203_02293_b200 import workloads as W
    cfg, inp, meta = W.make(config, columns=slice(0, 6)) if config == 1 else W.make(config, columns=slice(5, None, 640))
    flags = (cfg["flags"] & ~W.TOA_SPECTRUM & ~W.NONISOTHERMAL) | (W.NONISOTHERMAL if noniso else 0)
    res = oracle_mod.rt_step(dict(cfg, flags=flags), inp, want=("F_up", "F_up_toa_bin"))
    dlam = np.diff(np.asarray(cfg["bin_edges"]))
    assert np.all(dlam > 0) and np.ptp(dlam) > 0.5 * dlam.min()          # unequal bins: a missing / doubled dlam shows
    integral = res["F_up_toa_bin"] @ dlam
    assert np.all(integral > 0)
    assert np.allclose(integral, res["F_up"][:, -1], rtol=1e-13, atol=0)
    # ... and the spectrum is not the flux at some other level: in these columns F_up changes with height
    assert np.all(np.abs(res["F_up"][:, meta["n_layers"] // 2] / res["F_up"][:, -1] - 1) > 1e-3)


def test_toa_spectrum_pure_absorption_closed_form(oracle_mod):
    """One isothermal, purely absorbing, night-side column with a (P, T)-independent opacity: per spectral point
    F_up[N] = pi B (1 - e^{-2 tau}) + e^{-2 tau} (pi B (1 - e^{-2 tau}) + pi B(T_int)), tau = kappa_g (p_0 - p_N) / g
    (the closed form of test_pure_absorption_closed_form with one source value).  Two bins of different width, three
    Gauss points with UNEQUAL weights and opacities a decade apart: F_up_toa_bin[b] must be their w_g-weighted sum, per
    unit wavelength (no dlam), with no cross-talk between bins."""
    nb, ng = 2, 3
    kap = np.array([[3e-4, 3e-3, 3e-2], [1e-3, 2e-4, 5e-2]])
    gw = np.array([0.2, 0.5, 0.3])
    cfg = _optics_cfg(kap, 0.0, 0.0, 0.0, 0.0, nb=nb, ng=ng)
    cfg["bin_edges"] = np.array([2e-6, 3e-6, 5e-6])
    cfg["gauss_w"] = gw
    N, T0, f_int = 6, 1500.0, 4000.0
    p = np.logspace(5, 2, N)[None, :]
    inp = dict(p=p, T=np.full((1, N), T0), mu_star=np.array([-1.0]), stellar_flux=np.array([7.0, 9.0]), f_internal=f_int)
    for flags in (1, 3):
        res = oracle_mod.rt_step(dict(cfg, flags=flags), inp, want=("F_up_toa_bin", "F_up"))
        p_int, _ = oracle_mod.levels(p[0], inp["T"][0])
        col = (p_int[0] - p_int[-1]) / cfg["gravity"]
        T_int = (f_int / 5.670374419e-8) ** 0.25
        expect = np.zeros(nb)
        for b in range(nb):
            lo, hi = cfg["bin_edges"][b], cfg["bin_edges"][b + 1]
            piB, piB_int = np.pi * oracle_mod.planck_bin_mean(T0, lo, hi), np.pi * oracle_mod.planck_bin_mean(T_int, lo, hi)
            for g in range(ng):
                tr = np.exp(-2.0 * kap[b, g] * col)
                expect[b] += gw[g] * (piB * (1 - tr) + tr * (piB * (1 - tr) + piB_int))
        assert np.allclose(res["F_up_toa_bin"][0], expect, rtol=1e-12, atol=0), flags
        assert abs(expect[0] / expect[1] - 1) > 0.1                 # the two bins differ: swapping them would show


def test_levels_single_layer_reading_R27(oracle_mod):
    """N = 1 (reading R27): with no neighbour to take a half step from, the one layer spans one decade of pressure
    centred (in ln p) on its own pressure.  Hand values: p = 2e4 Pa -> interfaces 2e4 * 10^(+-1/2)."""
    pi, ti = oracle_mod.levels(np.array([2.0e4]), np.array([1234.5]))
    assert pi.shape == (2,) and ti.shape == (2,)
    assert pi[0] == pytest.approx(63245.553203367587, rel=1e-15)     # 2e4 * 3.1622776601683793...
    assert pi[1] == pytest.approx(6324.5553203367587, rel=1e-15)     # 2e4 / 3.1622776601683793...
    assert pi[0] / pi[1] == pytest.approx(10.0, rel=1e-15) and pi[0] * pi[1] == pytest.approx(4.0e8, rel=1e-15)
    assert ti[0] == 1234.5 and ti[1] == 1234.5
    # the same rule is what R9 gives a two-layer column whose layers are one decade apart: the limits agree
    pi2, _ = oracle_mod.levels(np.array([2.0e4, 2.0e3]), np.array([1000.0, 900.0]))
    assert pi2[0] == pytest.approx(pi[0], rel=1e-14) and pi2[1] == pytest.approx(pi[1], rel=1e-14)
