"""Seeded synthetic workloads shaped like the paper's WASP-43b runs.

This module holds NONE of the method's arithmetic: it only draws / tabulates inputs (numpy) and is
the one place both the CPU oracle and the CUDA path get their inputs from, so they see bit-identical
arrays.  It imports neither of them.

The paper's real inputs (HELIOS-K k-tables, FastChem abundances, LX-MIE cloud, PHOENIX template,
THOR-evolved P,T) are not available; the generators below take their
shapes, sizes and value ranges from the paper and BASELINE.json and stand in for them.

Configs (BASELINE.json `configs`):
  1  tiny        64 x 10 x (4 x 4)      isothermal, improved, no cloud
  2  wasp43b     2562 x 40 x (30 x 20)  isothermal, improved, cloud 1e-3..1 bar        (headline)
  3  wasp43b-ni  as 2, non-isothermal, T_int = 400 K
  4  hires       10242 x 40 x (30 x 20) non-isothermal
  5  spectrum    2562 x 40 x (300 x 20) isothermal, TOA spectrum only
  6  postproc the post-processing step of PAPER.md L385: 2562 columns x 40 layers from
                 1e3 to 1e-3 bar, extended by 20 isothermal layers to 1 ubar (-> 60 layers), opacity sampling at
                 R = 500 (3255 wavelength points x 1 "Gauss point", Fig. 7), TOA spectrum only; with the grid's
                 lon / lat / control-volume areas and 64 orbital phases for the phase curve (Eqs. 23-26)
"""
from __future__ import annotations

import numpy as np

IMPROVED = 1
NONISOTHERMAL = 2
TOA_SPECTRUM = 4

SIGMA_SB = 5.670374419e-8  # W m^-2 K^-4 (CODATA 2019)
BAR = 1.0e5                # Pa
# Table 3 of the paper
GRAVITY = 47.0
CP = 12436.0
EPS2 = 2.0 / 3.0
R_STAR = 4.64e8
SEMI_MAJOR = 2.28e9
T_STAR = 4798.0

_SEED_BASE = 220302293 * 10


def gauss_legendre_01(n: int):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (x + 1.0), 0.5 * w


def bin_edges_equal_wavenumber(n_bins: int, lam_min=0.3e-6, lam_max=200e-6) -> np.ndarray:
    """n_bins bins of equal width in wavenumber between lam_min and lam_max;
    returned as ascending wavelength edges in metres."""
    nu = np.linspace(1.0 / lam_max, 1.0 / lam_min, n_bins + 1)
    return (1.0 / nu)[::-1].copy()


def _blackbody_bin_mean_quadrature(T: float, edges: np.ndarray, n: int = 4001) -> np.ndarray:
    """Bin-mean blackbody radiance per unit wavelength by composite Simpson quadrature in
    ln(lambda).  Only shapes the synthetic stellar spectrum (stand-in for the PHOENIX template,
    PAPER.md Fig. 4); it is an INPUT, not part of the method."""
    h, c, k = 6.62607015e-34, 299792458.0, 1.380649e-23
    out = np.empty(len(edges) - 1)
    for b in range(len(edges) - 1):
        u = np.linspace(np.log(edges[b]), np.log(edges[b + 1]), n)
        lam = np.exp(u)
        x = h * c / (lam * k * T)
        f = 2 * h * c * c / lam**5 / np.expm1(np.minimum(x, 700.0)) * lam  # B_lambda dlam = B_lambda lam du
        du = u[1] - u[0]
        s = f[0] + f[-1] + 4 * f[1:-1:2].sum() + 2 * f[2:-1:2].sum()
        out[b] = s * du / 3.0 / (edges[b + 1] - edges[b])
    return out


def icosahedral_grid(g_level: int) -> np.ndarray:
    """Vertices (unit vectors, [10*4^g+2, 3]) of a recursively subdivided icosahedron projected to the
    sphere (plain subdivision, no spring dynamics)."""
    t = (1.0 + 5.0**0.5) / 2.0
    v = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t), (0, -1, -t), (0, 1, -t),
         (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    verts = [np.array(x, dtype=np.float64) / np.linalg.norm(x) for x in v]
    faces = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2),
             (10, 7, 6), (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5),
             (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    for _ in range(g_level):
        cache: dict[tuple[int, int], int] = {}

        def mid(a: int, b: int) -> int:
            key = (a, b) if a < b else (b, a)
            if key not in cache:
                m = verts[a] + verts[b]
                verts.append(m / np.linalg.norm(m))
                cache[key] = len(verts) - 1
            return cache[key]

        nf = []
        for a, b, c in faces:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            nf += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        faces = nf
    return np.array(verts)


def grid_geometry(g_level: int):
    """Longitude, latitude (radians) and control-volume solid angle A_i / R_p^2 of every vertex of the
    icosahedral grid (Eq. 25): the control volumes are the spherical Voronoi cells of the
    vertices.  Inputs of the phase-curve reduction; no method arithmetic."""
    from scipy.spatial import SphericalVoronoi
    xyz = icosahedral_grid(g_level)
    lon = np.mod(np.arctan2(xyz[:, 1], xyz[:, 0]), 2.0 * np.pi)      # 0 <= phi < 2 pi (L533)
    lat = np.arcsin(np.clip(xyz[:, 2], -1.0, 1.0))
    area = SphericalVoronoi(xyz, radius=1.0).calculate_areas()
    return lon, lat, np.ascontiguousarray(area)


def _ktable(rng, ktab_p, ktab_t, n_bins, n_gauss):
    """ln kappa = ln(1e-4) + 2 z_sorted[b,g] + a_b/2 ln(P/bar) + c_b (T-1500)/1500 + 0.3 eta[iP,iT,b];
    log-normal (median 1e-3 cm^2/g = 1e-4 m^2/kg, sigma_ln = 2), ascending in g within each bin as
    k-distributions are."""
    z = np.sort(rng.standard_normal((n_bins, n_gauss)), axis=1)
    a_b = rng.uniform(0.0, 0.5, n_bins)
    c_b = rng.uniform(-1.0, 1.0, n_bins)
    eta = rng.standard_normal((len(ktab_p), len(ktab_t), n_bins))
    lnk = (np.log(1e-4) + 2.0 * z[None, None, :, :]
           + (a_b * 0.5)[None, None, :, None] * np.log(ktab_p / BAR)[:, None, None, None]
           + c_b[None, None, :, None] * ((ktab_t - 1500.0) / 1500.0)[None, :, None, None]
           + 0.3 * eta[:, :, :, None])
    return np.ascontiguousarray(np.exp(lnk)), z


def _guillot_like(p, mu, T_int):
    """Closed form fixed by the generator (shape of Guillot 2010 Eq. 27):
    T^4 = 3/4 T_int^4 (2/3 + tau) + 3/4 T_irr^4 f(mu) (5/3 - 2/3 e^-tau), tau = p / 1 bar."""
    T_irr = 2440.0
    tau = (p / BAR)[None, :]
    f = (0.1 + 0.9 * np.maximum(mu, 0.0))[:, None]
    T4 = 0.75 * T_int**4 * (2.0 / 3.0 + tau) + 0.75 * T_irr**4 * f * (5.0 / 3.0 - 2.0 / 3.0 * np.exp(-tau))
    return np.clip(T4**0.25, 100.0, 3000.0)


def make(config: int, columns=None) -> tuple[dict, dict, dict]:
    """Build BASELINE.json config 1..5.  Returns (cfg, inp, meta) of host numpy arrays.

    `columns`: optional index array / slice selecting a subset of the columns AFTER generation (the
    random draws are always those of the full config, so a subset is a true sub-sample)."""
    if config == 6:
        return _make_postproc(columns)
    if config not in (1, 2, 3, 4, 5):
        raise ValueError("config must be 1..6")
    rng = np.random.default_rng(_SEED_BASE + config)
    if config == 1:
        n_col, N, nb, ng = 64, 10, 4, 4
        ktab_p = np.logspace(-5, 2, 6) * BAR
        ktab_t = np.linspace(500.0, 2000.0, 6)
        p1 = np.logspace(1, -4, N) * BAR
    else:
        N, nb, ng = 40, (300 if config == 5 else 30), 20
        n_col = 10242 if config == 4 else 2562
        ktab_p = np.logspace(-6, 3, 20) * BAR
        ktab_t = np.linspace(100.0, 3000.0, 30)
        p1 = np.logspace(3, -6, N) * BAR
    edges = bin_edges_equal_wavenumber(nb)
    _, gw = gauss_legendre_01(ng)
    ktab, z = _ktable(rng, ktab_p, ktab_t, nb, ng)
    lam_c = 0.5 * (edges[:-1] + edges[1:])
    stellar = np.pi * _blackbody_bin_mean_quadrature(T_STAR, edges) * (R_STAR / SEMI_MAJOR) ** 2

    flags = IMPROVED
    if config == 1:
        T = 800.0 + 800.0 / (1.0 + np.exp(-(np.log10(p1 / BAR) + 1.0) / 0.5))
        T = T[None, :] + rng.normal(0.0, 30.0, (n_col, N))
        mu = rng.uniform(-1.0, 1.0, n_col)
        scat_gas = (3.0 / 7.0) * ktab.min(axis=(0, 1, 3))
        cloud_ext = np.zeros(nb)
        cloud_w0 = np.zeros(nb)
        cloud_g0 = np.zeros(nb)
        cloud_p_top, cloud_p_bot = 1.0, 0.0  # empty range: no cloud anywhere
        f_internal = SIGMA_SB * 100.0**4
    else:
        xyz = icosahedral_grid(5 if config == 4 else 4)
        assert xyz.shape[0] == n_col
        mu = xyz[:, 0].copy()  # substellar point at lat = lon = 0: mu = cos(lat) cos(lon)
        T_int = 400.0 if config in (3, 4) else 100.0
        T = _guillot_like(p1, mu, T_int)
        f_internal = SIGMA_SB * T_int**4
        if config in (3, 4):
            flags |= NONISOTHERMAL
        scat_gas = 1e-6 * (lam_c / 1e-6) ** -4.0
        cloud_ext = 10.0 * np.exp(np.log(1e-4) + 2.0 * np.median(z, axis=1))
        if config == 5:
            phi = rng.uniform(0.0, 2.0 * np.pi, 2)
            b = np.arange(nb)
            cloud_w0 = 0.5 + 0.499 * np.sin(3.0 * np.pi * b / nb + phi[0])
            cloud_g0 = 0.45 + 0.45 * np.cos(2.0 * np.pi * b / nb + phi[1])
            flags |= TOA_SPECTRUM
        else:
            cloud_w0 = rng.uniform(0.0, 0.999, nb)
            cloud_g0 = rng.uniform(0.0, 0.9, nb)
        cloud_p_top, cloud_p_bot = 1e-3 * BAR, 1.0 * BAR
    p = np.broadcast_to(p1, (n_col, N)).copy()

    if columns is not None:
        idx = np.arange(n_col)[columns]
        p, T, mu = p[idx].copy(), T[idx].copy(), mu[idx].copy()

    cfg = dict(n_layers=N, ktab_p=ktab_p, ktab_t=ktab_t, ktab=ktab, bin_edges=edges, gauss_w=gw, scat_gas=scat_gas,
               cloud_ext=cloud_ext, cloud_w0=cloud_w0, cloud_g0=cloud_g0, cloud_p_top=cloud_p_top,
               cloud_p_bot=cloud_p_bot, gravity=GRAVITY, cp=CP, eps2=EPS2, e_tau=1e-4, gcrit_tol=1e-5,
               w0_transition=0.1, f_toa=0.0, flags=flags)
    inp = dict(p=np.ascontiguousarray(p), T=np.ascontiguousarray(T), mu_star=mu, stellar_flux=stellar,
               f_internal=f_internal)
    meta = dict(config=config, n_columns=p.shape[0], n_layers=N, n_bins=nb, n_gauss=ng,
                F_star_tot=float(np.sum(np.diff(edges) * stellar)),
                name={1: "tiny", 2: "wasp43b-iso", 3: "wasp43b-noniso", 4: "hires-noniso", 5: "spectrum-toa"}[config])
    return cfg, inp, meta


def _make_postproc(columns=None, n_col_level: int = 4, nb: int = 3255, N: int = 40, n_extra: int = 20):
    """Config 6: see the module docstring.  cfg["n_layers"] is the EXTENDED layer count (what the RT handle is
    created with); inp["p"], inp["T"] are the model's own 40 layers; meta carries n_extra, p_min and the
    phase-curve inputs."""
    rng = np.random.default_rng(_SEED_BASE + 6)
    ktab_p = np.logspace(-6, 3, 20) * BAR
    ktab_t = np.linspace(100.0, 3000.0, 30)
    p1 = np.logspace(3, -3, N) * BAR
    edges = 0.3e-6 * (200.0 / 0.3) ** (np.arange(nb + 1) / nb)          # R = lam/dlam ~ 500 (Fig. 7)
    gw = np.array([1.0])
    ktab, z = _ktable(rng, ktab_p, ktab_t, nb, 1)
    lam_c = 0.5 * (edges[:-1] + edges[1:])
    # stellar spectrum: bin-mean blackbody; the bins are narrow, a 21-point Simpson rule is exact to 1e-10
    stellar = np.pi * _blackbody_bin_mean_quadrature(T_STAR, edges, n=21) * (R_STAR / SEMI_MAJOR) ** 2
    xyz = icosahedral_grid(n_col_level)
    mu = xyz[:, 0].copy()
    T = _guillot_like(p1, mu, 100.0)
    phi = rng.uniform(0.0, 2.0 * np.pi, 2)
    b = np.arange(nb)
    cloud_w0 = 0.5 + 0.499 * np.sin(3.0 * np.pi * b / nb + phi[0])
    cloud_g0 = 0.45 + 0.45 * np.cos(2.0 * np.pi * b / nb + phi[1])
    cloud_ext = 10.0 * np.exp(np.log(1e-4) + 2.0 * z[:, 0])
    scat_gas = 1e-6 * (lam_c / 1e-6) ** -4.0
    lon, lat, area = grid_geometry(n_col_level)
    p = np.broadcast_to(p1, (xyz.shape[0], N)).copy()
    if columns is not None:
        idx = np.arange(xyz.shape[0])[columns]
        p, T, mu, lon, lat, area = p[idx].copy(), T[idx].copy(), mu[idx].copy(), lon[idx].copy(), lat[idx].copy(), area[idx].copy()
    cfg = dict(n_layers=N + n_extra, ktab_p=ktab_p, ktab_t=ktab_t, ktab=ktab, bin_edges=edges, gauss_w=gw,
               scat_gas=scat_gas, cloud_ext=cloud_ext, cloud_w0=cloud_w0, cloud_g0=cloud_g0, cloud_p_top=1e-3 * BAR,
               cloud_p_bot=1.0 * BAR, gravity=GRAVITY, cp=CP, eps2=EPS2, e_tau=1e-4, gcrit_tol=1e-5, w0_transition=0.1,
               f_toa=0.0, flags=IMPROVED | TOA_SPECTRUM)
    inp = dict(p=np.ascontiguousarray(p), T=np.ascontiguousarray(T), mu_star=mu, stellar_flux=stellar,
               f_internal=SIGMA_SB * 100.0**4)
    meta = dict(config=6, n_columns=p.shape[0], n_layers=N + n_extra, n_model_layers=N, n_extra=n_extra, p_min=1e-6 * BAR,
                n_bins=nb, n_gauss=1, F_star_tot=float(np.sum(np.diff(edges) * stellar)), name="postproc-R500",
                lon=lon, lat=lat, area=area, alpha=np.linspace(-np.pi, np.pi, 64, endpoint=False),
                band=(1.1e-6, 1.7e-6))
    return cfg, inp, meta


def make_one_d(zenith_deg=(0.0, 30.0, 60.0, 89.0), cp: float = 2000.0):
    """Inputs of the "1-D mode" experiment (Sec. 3): one column per stellar zenith angle (the
    paper's 0, 30, 60, 89 degrees), config 1's column shape, table and spectrum (10 layers, 4 bins x 4 Gauss points),
    stepped with dt = 300 s (L384) from config 1's initial profile.  The steady state does not depend on the heat
    capacity, so c_P is lowered from Table 3's 12436 to `cp` J kg^-1 K^-1 as a pseudo-time acceleration (the paper
    integrates 800 days); the smaller the forcing, the smaller the c_P an explicit step tolerates: 2000 is stable at
    0-60 degrees, 500 at 89 degrees.  Returns (cfg, inp, meta, extra) with extra = dict(z, p_ref, R_d, dt): the fixed
    altitude grid (barometric, from the initial mean temperature), the reference pressure of Eq.(20), the gas constant
    of Table 3 and the time step."""
    cfg, inp, meta = make(1, columns=slice(0, len(zenith_deg)))
    mu = np.cos(np.radians(np.asarray(zenith_deg, dtype=np.float64)))
    R_d = 3553.0
    z = (R_d * inp["T"].mean() / cfg["gravity"]) * np.log(inp["p"][0, 0] / inp["p"][0])
    cfg = dict(cfg, cp=float(cp))
    inp = dict(inp, mu_star=mu)
    return cfg, inp, meta, dict(z=z, p_ref=float(inp["p"][0, 0]), R_d=R_d, dt=300.0)
