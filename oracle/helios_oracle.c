/*
 * helios_oracle.c -- plain, slow CPU oracle for the THOR+HELIOS radiative-transfer step.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2203_02293_b200/) may
 * import, link or execute this file; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs do.  It shares no code, header, table or helper with
 * the CUDA path.
 *
 * Every function restates a passage of /root/reference/PAPER.md (Deitrick et al., arXiv
 * 2203.02293) literally, in the paper's order and notation; where the paper is silent the
 * reading of DESIGN.md ("Readings", R1..R15 = SURVEY.md 8(c) Q1..Q18) is taken and named.
 * No blocking, fusion or algebraic rearrangement: chi, xi, psi, Pi, G+- are evaluated exactly
 * as printed in Eqs. (B1), (B2), (B5), (B8); the flux relations are Eqs. (2)-(10); the system
 * is the 2x2-block tridiagonal system of Eq. (12) solved by Eqs. (13)-(15).
 *
 * Precision: compiled twice.  -DORACLE_REAL="long double" (default) is the truth used for
 * parity; -DORACLE_REAL=double is the timed CPU baseline.  All array arguments are double.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): ODE integration of the two-stream equations
 * across one layer; dense LU of the assembled system; the converged pair-wise iteration the
 * paper replaces; pure-absorption closed form; conservative scattering; opaque isothermal
 * limit; layer-splitting exactness; BOA condition; Planck integrals vs quadrature and
 * sigma*T^4; bilinear reproduction; guard branches; 40-digit worked example.  The pair-wise
 * iteration (column_mono_iterative) is pinned by its limit (= dense LU of the system) and by
 * the non-scattering case, where one iteration is already the closed form.
 *
 * Index conventions (SURVEY.md "Conventions"): layer j (0..N-1) lies between interface j
 * (lower) and j+1 (upper); interface 0 = BOA, interface N = TOA; tau measured from the TOA
 * downward; API mu > 0 is the dayside and the paper's mu_star = -mu (App. B).
 */
#include <math.h>
#include <tgmath.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef ORACLE_REAL
#define ORACLE_REAL long double
#endif
typedef ORACLE_REAL real;

#define ORACLE_IMPROVED      1u
#define ORACLE_NONISOTHERMAL 2u
#define ORACLE_TOA_SPECTRUM  4u

/* CODATA-2019 exact SI constants. */
static const real H_PLANCK = (real)6.62607015e-34L;
static const real C_LIGHT  = (real)299792458.0L;
static const real K_BOLTZ  = (real)1.380649e-23L;
static const real PI_R     = (real)3.14159265358979323846264338327950288L;

/* ------------------------------------------------------------------------------------------
 * Planck (reading R8: exact bin-mean radiance per unit wavelength; paper silent, L171).
 * G(x) = int_x^inf t^3/(e^t-1) dt.
 *   x >= 1 : sum_{n>=1} e^{-n x} (x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4)
 *   x <  1 : pi^4/15 - sum_k B_k x^{k+3} / ((k+3) k!)   (Bernoulli series of t/(e^t-1))
 * ---------------------------------------------------------------------------------------- */
static real planck_G(real x)
{
    if (x <= 0) return PI_R * PI_R * PI_R * PI_R / 15;
    if (x >= 1) {
        real sum = 0;
        for (int n = 1; n < 20000; ++n) {
            real rn = (real)n;
            real term = exp(-rn * x) * (x * x * x / rn + 3 * x * x / (rn * rn)
                                        + 6 * x / (rn * rn * rn) + 6 / (rn * rn * rn * rn));
            sum += term;
            if (term < (real)1e-24L * sum) break;
        }
        return sum;
    }
    /* Bernoulli numbers B_0, B_1, B_2, B_4, ..., B_24 as exact fractions. */
    static const long double bnum[] = {1.0L, -1.0L, 1.0L, -1.0L, 1.0L, -1.0L, 5.0L, -691.0L, 7.0L,
                                       -3617.0L, 43867.0L, -174611.0L, 854513.0L, -236364091.0L};
    static const long double bden[] = {1.0L, 2.0L, 6.0L, 30.0L, 42.0L, 30.0L, 66.0L, 2730.0L, 6.0L,
                                       510.0L, 798.0L, 330.0L, 138.0L, 2730.0L};
    static const int bidx[] = {0, 1, 2, 4, 6, 8, 10, 12, 14, 16, 18, 20, 22, 24};
    real low = 0;  /* int_0^x t^3/(e^t-1) dt */
    for (int m = 0; m < 14; ++m) {
        int k = bidx[m];
        real fact = 1;
        for (int q = 2; q <= k; ++q) fact *= (real)q;
        real xp = 1;
        for (int q = 0; q < k + 3; ++q) xp *= x;
        low += (real)bnum[m] / (real)bden[m] * xp / ((real)(k + 3) * fact);
    }
    return PI_R * PI_R * PI_R * PI_R / 15 - low;
}

/* B_b(T) = [2 k^4 T^4 / (h^3 c^2)] [G(x_hi) - G(x_lo)] / (lam_hi - lam_lo), x = h c / (lam k T);
 * the short-wavelength edge has the larger x.  W m^-2 sr^-1 m^-1.  T <= 0 gives 0. */
static real planck_bin_mean(real T, real lam_lo, real lam_hi)
{
    if (!(T > 0)) return 0;
    real x_of_lo = H_PLANCK * C_LIGHT / (lam_lo * K_BOLTZ * T);  /* larger x */
    real x_of_hi = H_PLANCK * C_LIGHT / (lam_hi * K_BOLTZ * T);  /* smaller x */
    real pref = 2 * K_BOLTZ * K_BOLTZ * K_BOLTZ * K_BOLTZ * T * T * T * T
                / (H_PLANCK * H_PLANCK * H_PLANCK * C_LIGHT * C_LIGHT);
    return pref * (planck_G(x_of_hi) - planck_G(x_of_lo)) / (lam_hi - lam_lo);
}

double oracle_planck_G(double x) { return (double)planck_G((real)x); }
double oracle_planck_bin_mean(double T, double lam_lo, double lam_hi)
{
    return (double)planck_bin_mean((real)T, (real)lam_lo, (real)lam_hi);
}

/* ------------------------------------------------------------------------------------------
 * O1 levels (reading R9; "values at the interfaces are determined by linear
 * interpolation").  Interfaces in ln p: interior = midpoint of the adjacent centres, ends
 * extrapolated half a step; T interior = mean of adjacent centres, ends held constant.
 * Outputs: p_int[N+1], T_int[N+1].
 * ---------------------------------------------------------------------------------------- */
static void levels(int N, const double *p, const double *T, real *p_int, real *T_int)
{
    for (int i = 1; i < N; ++i) {
        p_int[i] = exp((log((real)p[i - 1]) + log((real)p[i])) / 2);
        T_int[i] = ((real)T[i - 1] + (real)T[i]) / 2;
    }
    if (N >= 2) {
        p_int[0] = exp(log((real)p[0]) + (log((real)p[0]) - log((real)p[1])) / 2);
        p_int[N] = exp(log((real)p[N - 1]) - (log((real)p[N - 2]) - log((real)p[N - 1])) / 2);
    } else { /* single layer: no neighbour to take a step from; half a decade each way */
        p_int[0] = (real)p[0] * sqrt((real)10);
        p_int[N] = (real)p[0] / sqrt((real)10);
    }
    T_int[0] = (real)T[0];
    T_int[N] = (real)T[N - 1];
}

void oracle_levels(int N, const double *p, const double *T, double *p_int, double *T_int)
{
    real *pi_ = malloc(sizeof(real) * (N + 1)), *ti_ = malloc(sizeof(real) * (N + 1));
    levels(N, p, T, pi_, ti_);
    for (int i = 0; i <= N; ++i) { p_int[i] = (double)pi_[i]; T_int[i] = (double)ti_[i]; }
    free(pi_); free(ti_);
}

/* ------------------------------------------------------------------------------------------
 * O2 opacity (reading R7; scheme not stated): bilinear interpolation of ln kappa
 * in (log10 P, T), coordinates clamped to the table range; grids strictly ascending.
 * ktab layout [nP][nT][nbin][ng].
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int nP, nT, nbin, ng;
    const double *ktab_p, *ktab_t, *ktab;
} ktable;

static void find_cell(int n, const double *grid, real x, int log10_coord, int *i0, real *w)
{
    real xc = x;
    if (xc < (real)grid[0]) xc = (real)grid[0];
    if (xc > (real)grid[n - 1]) xc = (real)grid[n - 1];
    int i = 0;
    while (i < n - 2 && xc > (real)grid[i + 1]) ++i;
    real a = (real)grid[i], b = (real)grid[i + 1];
    if (log10_coord) *w = (log10(xc) - log10(a)) / (log10(b) - log10(a));
    else             *w = (xc - a) / (b - a);
    *i0 = i;
}

static real kappa_abs(const ktable *kt, real p, real T, int b, int g)
{
    int ip, it; real wp, wt;
    find_cell(kt->nP, kt->ktab_p, p, 1, &ip, &wp);
    find_cell(kt->nT, kt->ktab_t, T, 0, &it, &wt);
    size_t sT = (size_t)kt->nbin * kt->ng, sP = sT * kt->nT, o = (size_t)b * kt->ng + g;
    real l00 = log((real)kt->ktab[ip * sP + it * sT + o]);
    real l01 = log((real)kt->ktab[ip * sP + (it + 1) * sT + o]);
    real l10 = log((real)kt->ktab[(ip + 1) * sP + it * sT + o]);
    real l11 = log((real)kt->ktab[(ip + 1) * sP + (it + 1) * sT + o]);
    real l = (1 - wp) * ((1 - wt) * l00 + wt * l01) + wp * ((1 - wt) * l10 + wt * l11);
    return exp(l);
}

double oracle_kappa(int nP, int nT, int nbin, int ng, const double *ktab_p, const double *ktab_t,
                    const double *ktab, double p, double T, int b, int g)
{
    ktable kt = {nP, nT, nbin, ng, ktab_p, ktab_t, ktab};
    return (double)kappa_abs(&kt, (real)p, (real)T, b, g);
}

/* ------------------------------------------------------------------------------------------
 * O7 layer coefficients, literal: E Eq.(19) L374 (readings R5: E <- max(1, fit); R6: strict
 * "omega0 > w0_transition"); zeta+-, T Eq.(B2); chi, xi, psi Eq.(B1);
 * Pi Eq.(B5); G+- Eq.(B8) L1091 with mu_star = -mu and the guard of L252 / Eq.(11)
 * (reading R4: test |D| < gcrit_tol, then D <- 2 mu_star).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    real E, zeta_p, zeta_m, trans, chi, xi, psi, Pi, G_p, G_m, twoE1mwg;
} coeffs;

static coeffs layer_coeffs(real w0, real g0, real dtau, real mu, real eps2, int improved,
                           real gcrit_tol, real w0_transition)
{
    coeffs c;
    real E = 1;
    if (improved && w0 > w0_transition) {
        E = (real)1.225L - (real)0.1582L * g0 - (real)0.1777L * w0 - (real)0.07465L * g0 * g0
            + (real)0.2351L * w0 * g0 - (real)0.05582L * w0 * w0;
        if (E < 1) E = 1;
    }
    c.E = E;
    real root = sqrt((E - w0) / (E * (1 - w0 * g0)));
    c.zeta_p = (1 + root) / 2;
    c.zeta_m = (1 - root) / 2;
    c.trans = exp(-2 * sqrt(E * (E - w0) * (1 - w0 * g0)) * dtau);
    c.chi = c.zeta_m * c.zeta_m * c.trans * c.trans - c.zeta_p * c.zeta_p;
    c.xi = c.zeta_p * c.zeta_m * (1 - c.trans * c.trans);
    c.psi = (c.zeta_m * c.zeta_m - c.zeta_p * c.zeta_p) * c.trans;
    c.Pi = PI_R * (1 - w0) / (E - w0);
    c.twoE1mwg = 2 * E * (1 - w0 * g0);
    c.G_p = 0; c.G_m = 0;
    if (mu > 0) {
        real mustar = -mu;
        real D = 4 * E * mustar * mustar * (E - w0) * (1 - w0 * g0) - 1;
        if (fabs(D) < gcrit_tol) D = 2 * mustar;
        real lead = w0 * (c.twoE1mwg + g0 / eps2) / D;
        real last = w0 * g0 / (eps2 * c.twoE1mwg);
        c.G_p = (lead * (mustar + 1 / c.twoE1mwg) + last) / 2;
        c.G_m = (lead * (mustar - 1 / c.twoE1mwg) - last) / 2;
    }
    return c;
}

/* out[10] = E, zeta+, zeta-, T, chi, xi, psi, Pi, G+, G- */
void oracle_layer_coeffs(double w0, double g0, double dtau, double mu, double eps2, int improved,
                         double gcrit_tol, double w0_transition, double *out)
{
    coeffs c = layer_coeffs((real)w0, (real)g0, (real)dtau, (real)mu, (real)eps2, improved,
                            (real)gcrit_tol, (real)w0_transition);
    out[0] = (double)c.E; out[1] = (double)c.zeta_p; out[2] = (double)c.zeta_m;
    out[3] = (double)c.trans; out[4] = (double)c.chi; out[5] = (double)c.xi;
    out[6] = (double)c.psi; out[7] = (double)c.Pi; out[8] = (double)c.G_p; out[9] = (double)c.G_m;
}

/* ------------------------------------------------------------------------------------------
 * O8: the block system of Eq.(12) (L286) for one monochromatic column of L "system layers"
 * (L = N isothermal; L = 2N sub-layers non-isothermal, L311-313), levels 0..L, level 0 = BOA.
 * System layer s lies between level s (lower, "a") and s+1 (upper, "b").
 *   row "F_up at b"  : Eq.(2) / Eq.(4),(7)   (L177-180, L190-200, L217)
 *   row "F_dn at a"  : Eq.(3) / Eq.(6),(9)   (L185, L211, L227-232)
 *   BOA: F_up0 - F_dn0 = F_BOA + F_beam0  Eq.(10);  TOA: F_dn,top = f_toa (Fig.5).
 * Reconstruction of the missing Figures 5/6 (reading R1).
 * Blocks stored row-major: A[l][4], Bm[l][4], C[l][4], D[l][2], l = 0..L.
 * B_lo[s], B_hi[s]: Planck function at the lower / upper end of system layer s.
 * linear_source = 0: isothermal rows (B' = 0, B* as given; pass B_lo = B_hi = B_centre).
 * linear_source = 1: B' = (B_lo - B_hi)/dtau, Theta Eqs.(5),(8), e_tau rule L209/L223
 * (reading R15: strict "<" on the sub-layer's own dtau).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    real eps2, e_tau, gcrit_tol, w0_transition, f_toa;
    int improved, linear_source;
} rt_opts;

static void assemble(int L, const real *dtau, const real *w0, const real *g0, const real *B_lo,
                     const real *B_hi, real mu, real Fstar, real F_boa, const rt_opts *o,
                     real *A, real *Bm, real *C, real *D, real *F_beam)
{
    /* optical depth from the TOA downward (O4) and the direct beam, Eq.(B6) L1080 with
     * mu_star = -mu:  F_beam = -mu_star F_star exp(tau/mu_star) = mu F_star exp(-tau/mu). */
    real *tau = malloc(sizeof(real) * (L + 1));
    tau[L] = 0;
    for (int s = L - 1; s >= 0; --s) tau[s] = tau[s + 1] + dtau[s];
    for (int l = 0; l <= L; ++l) F_beam[l] = (mu > 0) ? mu * Fstar * exp(-tau[l] / mu) : 0;

    memset(A, 0, sizeof(real) * 4 * (L + 1));
    memset(Bm, 0, sizeof(real) * 4 * (L + 1));
    memset(C, 0, sizeof(real) * 4 * (L + 1));
    memset(D, 0, sizeof(real) * 2 * (L + 1));

    /* boundary rows */
    Bm[0 * 4 + 0] = 1; Bm[0 * 4 + 1] = -1; D[0 * 2 + 0] = F_boa + F_beam[0];
    Bm[L * 4 + 2] = 0; Bm[L * 4 + 3] = 1;  D[L * 2 + 1] = o->f_toa;

    for (int s = 0; s < L; ++s) {
        coeffs c = layer_coeffs(w0[s], g0[s], dtau[s], mu, o->eps2, o->improved, o->gcrit_tol,
                                o->w0_transition);
        real Ba = B_lo[s], Bb = B_hi[s], Bprime = 0;
        if (o->linear_source) {
            if ((tau[s] - tau[s + 1]) < o->e_tau) { Ba = Bb = (B_lo[s] + B_hi[s]) / 2; Bprime = 0; }
            else Bprime = (B_lo[s] - B_hi[s]) / (tau[s] - tau[s + 1]);
        }
        real Theta = (c.chi - c.psi - c.xi) / c.twoE1mwg;
        real rhs_up = c.Pi * (Bb * (c.chi + c.xi) - c.psi * Ba + Bprime * Theta)
                      + c.psi * c.G_p * F_beam[s] - (c.xi * c.G_m + c.chi * c.G_p) * F_beam[s + 1];
        real rhs_dn = c.Pi * (Ba * (c.chi + c.xi) - c.psi * Bb - Bprime * Theta)
                      + c.psi * c.G_m * F_beam[s + 1] - (c.xi * c.G_p + c.chi * c.G_m) * F_beam[s];
        /* row 1 of block s+1: chi F_up[s+1] - psi F_up[s] + xi F_dn[s+1] = rhs_up */
        A[(s + 1) * 4 + 0] = -c.psi;
        Bm[(s + 1) * 4 + 0] = c.chi; Bm[(s + 1) * 4 + 1] = c.xi;
        D[(s + 1) * 2 + 0] = rhs_up;
        /* row 2 of block s: xi F_up[s] + chi F_dn[s] - psi F_dn[s+1] = rhs_dn */
        Bm[s * 4 + 2] = c.xi; Bm[s * 4 + 3] = c.chi;
        C[s * 4 + 3] = -c.psi;
        D[s * 2 + 1] = rhs_dn;
    }
    free(tau);
}

/* 2x2 helpers, row-major m = {m00, m01, m10, m11} */
static void inv2(const real *m, real *r)
{
    real det = m[0] * m[3] - m[1] * m[2];
    r[0] = m[3] / det; r[1] = -m[1] / det; r[2] = -m[2] / det; r[3] = m[0] / det;
}
static void mul22(const real *a, const real *b, real *r)
{
    r[0] = a[0] * b[0] + a[1] * b[2]; r[1] = a[0] * b[1] + a[1] * b[3];
    r[2] = a[2] * b[0] + a[3] * b[2]; r[3] = a[2] * b[1] + a[3] * b[3];
}
static void mul21(const real *a, const real *v, real *r)
{
    r[0] = a[0] * v[0] + a[1] * v[1]; r[1] = a[2] * v[0] + a[3] * v[1];
}

/* Thomas's algorithm on 2x2 blocks, Eqs.(13)-(15) (L300-309); "/" = left-multiplication by the
 * inverse.  n block rows.  X[n][2] = (F_up, F_dn) per level. */
static void block_thomas(int n, const real *A, const real *Bm, const real *C, const real *D, real *X)
{
    real *Cp = malloc(sizeof(real) * 4 * n), *Dp = malloc(sizeof(real) * 2 * n);
    real inv[4], t[4], v[2];
    inv2(&Bm[0], inv);
    mul22(inv, &C[0], &Cp[0]);                       /* C'_0 = C_0 / B_0 */
    mul21(inv, &D[0], &Dp[0]);                       /* D'_0 = D_0 / B_0 */
    for (int i = 1; i < n; ++i) {
        mul22(&A[i * 4], &Cp[(i - 1) * 4], t);       /* A_i C'_{i-1} */
        for (int k = 0; k < 4; ++k) t[k] = Bm[i * 4 + k] - t[k];
        inv2(t, inv);
        mul22(inv, &C[i * 4], &Cp[i * 4]);           /* C'_i, Eq.(13) */
        mul21(&A[i * 4], &Dp[(i - 1) * 2], v);       /* A_i D'_{i-1} */
        v[0] = D[i * 2 + 0] - v[0]; v[1] = D[i * 2 + 1] - v[1];
        mul21(inv, v, &Dp[i * 2]);                   /* D'_i, Eq.(14) */
    }
    X[(n - 1) * 2 + 0] = Dp[(n - 1) * 2 + 0];       /* Eq.(15) */
    X[(n - 1) * 2 + 1] = Dp[(n - 1) * 2 + 1];
    for (int i = n - 2; i >= 0; --i) {
        mul21(&Cp[i * 4], &X[(i + 1) * 2], v);
        X[i * 2 + 0] = Dp[i * 2 + 0] - v[0];
        X[i * 2 + 1] = Dp[i * 2 + 1] - v[1];
    }
    free(Cp); free(Dp);
}

static rt_opts make_opts(double eps2, double e_tau, double gcrit_tol, double w0_transition,
                         double f_toa, int improved, int linear_source)
{
    rt_opts o;
    o.eps2 = (real)eps2; o.e_tau = (real)e_tau; o.gcrit_tol = (real)gcrit_tol;
    o.w0_transition = (real)w0_transition; o.f_toa = (real)f_toa;
    o.improved = improved; o.linear_source = linear_source;
    return o;
}

/* Test hook: the assembled blocks of one monochromatic column, as doubles, so that a test can
 * build the dense 2(L+1) x 2(L+1) matrix and solve it with a library LU. */
void oracle_assemble_blocks(int L, const double *dtau, const double *w0, const double *g0,
                            const double *B_lo, const double *B_hi, double mu, double Fstar,
                            double F_boa, double eps2, double e_tau, double gcrit_tol,
                            double w0_transition, double f_toa, int improved, int linear_source,
                            double *A, double *Bm, double *C, double *D, double *F_beam)
{
    rt_opts o = make_opts(eps2, e_tau, gcrit_tol, w0_transition, f_toa, improved, linear_source);
    int n = L + 1;
    real *r = malloc(sizeof(real) * (5 * L + 15 * n));
    real *dt = r, *w = dt + L, *g = w + L, *bl = g + L, *bh = bl + L;
    real *rA = bh + L, *rB = rA + 4 * n, *rC = rB + 4 * n, *rD = rC + 4 * n, *rF = rD + 2 * n;
    for (int s = 0; s < L; ++s) {
        dt[s] = (real)dtau[s]; w[s] = (real)w0[s]; g[s] = (real)g0[s];
        bl[s] = (real)B_lo[s]; bh[s] = (real)B_hi[s];
    }
    assemble(L, dt, w, g, bl, bh, (real)mu, (real)Fstar, (real)F_boa, &o, rA, rB, rC, rD, rF);
    for (int k = 0; k < 4 * n; ++k) { A[k] = (double)rA[k]; Bm[k] = (double)rB[k]; C[k] = (double)rC[k]; }
    for (int k = 0; k < 2 * n; ++k) D[k] = (double)rD[k];
    for (int k = 0; k < n; ++k) F_beam[k] = (double)rF[k];
    free(r);
}

/* One monochromatic column: assemble + Thomas.  Outputs F_up[L+1], F_dn[L+1] (diffuse),
 * F_beam[L+1]. */
static void column_mono(int L, const real *dtau, const real *w0, const real *g0, const real *B_lo,
                        const real *B_hi, real mu, real Fstar, real F_boa, const rt_opts *o,
                        real *F_up, real *F_dn, real *F_beam)
{
    int n = L + 1;
    real *r = malloc(sizeof(real) * 16 * n);
    real *A = r, *Bm = A + 4 * n, *C = Bm + 4 * n, *D = C + 4 * n, *X = D + 2 * n;
    assemble(L, dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, o, A, Bm, C, D, F_beam);
    block_thomas(n, A, Bm, C, D, X);
    for (int l = 0; l < n; ++l) { F_up[l] = X[2 * l]; F_dn[l] = X[2 * l + 1]; }
    free(r);
}

/* The scheme Thomas's algorithm replaces (L258-270, L397): "iterate the two-stream solutions, across the
 * entire atmosphere, for a finite number of times" (N = 200 in HELIOS, ~10 in Oreshenko et al. 2016).
 * Reading R23 (the paper does not print the sweep): all diffuse fluxes start at 0; one iteration is one upward
 * pass -- Eq.(10) at the BOA, then Eq.(2)/(4),(7) layer by layer with the downward fluxes of the previous
 * iteration -- followed by one downward pass -- F_dn,top = f_toa, then Eq.(3)/(6),(9) with the upward fluxes just
 * computed.  The rows are exactly those of assemble():
 *   chi F_up[s+1] = psi F_up[s] - xi F_dn[s+1] + rhs_up[s],   chi F_dn[s] = psi F_dn[s+1] - xi F_up[s] + rhs_dn[s]. */
static void column_mono_iterative(int L, const real *dtau, const real *w0, const real *g0, const real *B_lo,
                                  const real *B_hi, real mu, real Fstar, real F_boa, const rt_opts *o,
                                  int n_iter, real *F_up, real *F_dn, real *F_beam)
{
    int n = L + 1;
    real *r = malloc(sizeof(real) * 14 * n);
    real *A = r, *Bm = A + 4 * n, *C = Bm + 4 * n, *D = C + 4 * n;
    assemble(L, dtau, w0, g0, B_lo, B_hi, mu, Fstar, F_boa, o, A, Bm, C, D, F_beam);
    for (int l = 0; l < n; ++l) { F_up[l] = 0; F_dn[l] = 0; }
    for (int it = 0; it < n_iter; ++it) {
        F_up[0] = F_dn[0] + D[0];                                   /* Eq.(10): D[0] = F_BOA + F_beam[0] */
        for (int s = 0; s < L; ++s) {                               /* upward pass */
            real chi = Bm[(s + 1) * 4 + 0], xi = Bm[(s + 1) * 4 + 1], psi = -A[(s + 1) * 4 + 0];
            F_up[s + 1] = (psi * F_up[s] - xi * F_dn[s + 1] + D[(s + 1) * 2 + 0]) / chi;
        }
        F_dn[L] = D[L * 2 + 1];                                     /* f_toa */
        for (int s = L - 1; s >= 0; --s) {                          /* downward pass */
            real xi = Bm[s * 4 + 2], chi = Bm[s * 4 + 3], psi = -C[s * 4 + 3];
            F_dn[s] = (psi * F_dn[s + 1] - xi * F_up[s] + D[s * 2 + 1]) / chi;
        }
    }
    free(r);
}

void oracle_column_mono_iter(int L, const double *dtau, const double *w0, const double *g0,
                             const double *B_lo, const double *B_hi, double mu, double Fstar,
                             double F_boa, double eps2, double e_tau, double gcrit_tol,
                             double w0_transition, double f_toa, int improved, int linear_source,
                             int n_iter, double *F_up, double *F_dn, double *F_beam)
{
    rt_opts o = make_opts(eps2, e_tau, gcrit_tol, w0_transition, f_toa, improved, linear_source);
    int n = L + 1;
    real *r = malloc(sizeof(real) * (5 * L + 3 * n));
    real *dt = r, *w = dt + L, *g = w + L, *bl = g + L, *bh = bl + L;
    real *fu = bh + L, *fd = fu + n, *fb = fd + n;
    for (int s = 0; s < L; ++s) {
        dt[s] = (real)dtau[s]; w[s] = (real)w0[s]; g[s] = (real)g0[s];
        bl[s] = (real)B_lo[s]; bh[s] = (real)B_hi[s];
    }
    column_mono_iterative(L, dt, w, g, bl, bh, (real)mu, (real)Fstar, (real)F_boa, &o, n_iter, fu, fd, fb);
    for (int l = 0; l < n; ++l) { F_up[l] = (double)fu[l]; F_dn[l] = (double)fd[l]; F_beam[l] = (double)fb[l]; }
    free(r);
}

void oracle_column_mono(int L, const double *dtau, const double *w0, const double *g0,
                        const double *B_lo, const double *B_hi, double mu, double Fstar,
                        double F_boa, double eps2, double e_tau, double gcrit_tol,
                        double w0_transition, double f_toa, int improved, int linear_source,
                        double *F_up, double *F_dn, double *F_beam)
{
    rt_opts o = make_opts(eps2, e_tau, gcrit_tol, w0_transition, f_toa, improved, linear_source);
    int n = L + 1;
    real *r = malloc(sizeof(real) * (5 * L + 3 * n));
    real *dt = r, *w = dt + L, *g = w + L, *bl = g + L, *bh = bl + L;
    real *fu = bh + L, *fd = fu + n, *fb = fd + n;
    for (int s = 0; s < L; ++s) {
        dt[s] = (real)dtau[s]; w[s] = (real)w0[s]; g[s] = (real)g0[s];
        bl[s] = (real)B_lo[s]; bh[s] = (real)B_hi[s];
    }
    column_mono(L, dt, w, g, bl, bh, (real)mu, (real)Fstar, (real)F_boa, &o, fu, fd, fb);
    for (int l = 0; l < n; ++l) { F_up[l] = (double)fu[l]; F_dn[l] = (double)fd[l]; F_beam[l] = (double)fb[l]; }
    free(r);
}

/* ------------------------------------------------------------------------------------------
 * The full step (O1..O9).  Config / inputs / outputs mirror include/helios_rt.h but with HOST
 * pointers; the struct is the oracle's own (no shared header).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int32_t n_layers, n_bins, n_gauss, n_ktab_p, n_ktab_t;
    const double *ktab_p, *ktab_t, *ktab, *bin_edges, *gauss_w;
    const double *scat_gas, *cloud_ext, *cloud_w0, *cloud_g0;
    double cloud_p_top, cloud_p_bot, gravity, cp, eps2, e_tau, gcrit_tol, w0_transition, f_toa;
    uint32_t flags;
    int32_t n_iterations;   /* 0: Thomas (Eqs. 13-15); > 0: that many pair-wise iterations (L258-270) instead */
} oracle_config;

typedef struct {
    int32_t n_columns;
    const double *p, *T, *mu_star, *stellar_flux;
    double f_internal;
} oracle_inputs;

typedef struct {
    double *F_up, *F_down, *F_net, *dTdt, *F_beam, *F_up_toa_bin;
    /* optional debug: per-point interface fluxes of column dbg_column,
     * [n_layers+1][n_bins*n_gauss] each; NULL = not wanted */
    int32_t dbg_column;
    double *dbg_F_up_pt, *dbg_F_dn_pt;
} oracle_outputs;

/* optical properties at one level, O3 (Eqs. 17-18, per unit mass) */
static void level_optics(const oracle_config *cfg, const ktable *kt, real p, real T, int b, int g,
                         real *k_ext, real *w0, real *g0)
{
    real k_abs = kappa_abs(kt, p, T, b, g);
    real s_gas = (real)cfg->scat_gas[b];
    real k_c = 0, s_c = 0;
    if (p >= (real)cfg->cloud_p_top && p <= (real)cfg->cloud_p_bot) {
        k_c = (real)cfg->cloud_ext[b];
        s_c = (real)cfg->cloud_w0[b] * k_c;
    }
    *k_ext = k_abs + s_gas + k_c;
    *w0 = (s_gas + s_c) / *k_ext;
    *g0 = (s_gas + s_c > 0) ? s_c * (real)cfg->cloud_g0[b] / (s_gas + s_c) : 0;
}

/* exported for the pins of Eqs. 17-18 (tests/test_oracle_pins.py): the same level_optics the step uses; out = {k_ext, w0, g0} */
void oracle_level_optics(const oracle_config *cfg, double p, double T, int b, int g, double *out3)
{
    const ktable kt = {cfg->n_ktab_p, cfg->n_ktab_t, cfg->n_bins, cfg->n_gauss, cfg->ktab_p, cfg->ktab_t, cfg->ktab};
    real k, w, gg;
    level_optics(cfg, &kt, (real)p, (real)T, b, g, &k, &w, &gg);
    out3[0] = (double)k; out3[1] = (double)w; out3[2] = (double)gg;
}

int oracle_rt_step(const oracle_config *cfg, const oracle_inputs *in, const oracle_outputs *out)
{
    const int N = cfg->n_layers, nb = cfg->n_bins, ng = cfg->n_gauss, npt = nb * ng;
    const int noniso = (cfg->flags & ORACLE_NONISOTHERMAL) != 0;
    const int improved = (cfg->flags & ORACLE_IMPROVED) != 0;
    const int L = noniso ? 2 * N : N;
    const ktable kt = {cfg->n_ktab_p, cfg->n_ktab_t, nb, ng, cfg->ktab_p, cfg->ktab_t, cfg->ktab};
    const rt_opts o = make_opts(cfg->eps2, cfg->e_tau, cfg->gcrit_tol, cfg->w0_transition,
                                cfg->f_toa, improved, noniso);
    const real grav = (real)cfg->gravity;
    /* sigma_SB from the exact constants: 2 pi^5 k^4 / (15 h^3 c^2) */
    const real sigma_sb = 2 * PI_R * PI_R * PI_R * PI_R * PI_R * K_BOLTZ * K_BOLTZ * K_BOLTZ * K_BOLTZ
                          / (15 * H_PLANCK * H_PLANCK * H_PLANCK * C_LIGHT * C_LIGHT);
    const real T_internal = (in->f_internal > 0) ? sqrt(sqrt((real)in->f_internal / sigma_sb)) : 0;

#pragma omp parallel for schedule(dynamic, 1)
    for (int c = 0; c < in->n_columns; ++c) {
        const double *p = in->p + (size_t)c * N, *T = in->T + (size_t)c * N;
        const real mu = (real)in->mu_star[c];
        real *buf = malloc(sizeof(real) * (size_t)(2 * (N + 1) + 2 * (L + 1) + 3 * (L + 1)
                                                   + 5 * L + 3 * (L + 1) + 3 * (L + 1) + 3 * (N + 1)));
        real *p_int = buf, *T_int = p_int + (N + 1);
        real *p_lev = T_int + (N + 1), *T_lev = p_lev + (L + 1);
        real *kx = T_lev + (L + 1), *wl = kx + (L + 1), *gl = wl + (L + 1);
        real *dtau = gl + (L + 1), *w0 = dtau + L, *g0 = w0 + L, *B_lo = g0 + L, *B_hi = B_lo + L;
        real *Fu = B_hi + L, *Fd = Fu + (L + 1), *Fb = Fd + (L + 1);
        real *B_lev = Fb + (L + 1), *dm_sys = B_lev + (L + 1), *spare = dm_sys + (L + 1);
        real *acc_up = spare + (L + 1), *acc_dn = acc_up + (N + 1), *acc_bm = acc_dn + (N + 1);
        (void)spare;

        levels(N, p, T, p_int, T_int);                       /* O1 */
        if (noniso) {
            for (int i = 0; i <= N; ++i) { p_lev[2 * i] = p_int[i]; T_lev[2 * i] = T_int[i]; }
            for (int i = 0; i < N; ++i) { p_lev[2 * i + 1] = (real)p[i]; T_lev[2 * i + 1] = (real)T[i]; }
            for (int s = 0; s < L; ++s) dm_sys[s] = (p_lev[s] - p_lev[s + 1]) / grav;
        } else {
            for (int i = 0; i < N; ++i) dm_sys[i] = (p_int[i] - p_int[i + 1]) / grav;
        }
        for (int i = 0; i <= N; ++i) { acc_up[i] = 0; acc_dn[i] = 0; acc_bm[i] = 0; }

        for (int b = 0; b < nb; ++b) {
            const real lam_lo = (real)cfg->bin_edges[b], lam_hi = (real)cfg->bin_edges[b + 1];
            const real dlam = lam_hi - lam_lo;
            const real F_boa = PI_R * planck_bin_mean(T_internal, lam_lo, lam_hi);   /* L239 */
            /* O5 Planck at the levels of the system */
            if (noniso) {
                for (int l = 0; l <= L; ++l) B_lev[l] = planck_bin_mean(T_lev[l], lam_lo, lam_hi);
                for (int s = 0; s < L; ++s) { B_lo[s] = B_lev[s]; B_hi[s] = B_lev[s + 1]; }
            } else {
                for (int i = 0; i < N; ++i) B_lo[i] = B_hi[i] = planck_bin_mean((real)T[i], lam_lo, lam_hi);
            }
            real toa_bin = 0;
            for (int g = 0; g < ng; ++g) {
                /* O3/O4 optical properties per system layer */
                if (noniso) {
                    for (int l = 0; l <= L; ++l)
                        level_optics(cfg, &kt, p_lev[l], T_lev[l], b, g, &kx[l], &wl[l], &gl[l]);
                    for (int s = 0; s < L; ++s) {            /* L171: arithmetic means (R10) */
                        real kbar = (kx[s] + kx[s + 1]) / 2;
                        w0[s] = (wl[s] + wl[s + 1]) / 2;
                        g0[s] = (gl[s] + gl[s + 1]) / 2;
                        dtau[s] = kbar * dm_sys[s];
                    }
                } else {
                    for (int i = 0; i < N; ++i) {
                        real k;
                        level_optics(cfg, &kt, (real)p[i], (real)T[i], b, g, &k, &w0[i], &g0[i]);
                        dtau[i] = k * dm_sys[i];
                    }
                }
                if (cfg->n_iterations > 0)
                    column_mono_iterative(L, dtau, w0, g0, B_lo, B_hi, mu, (real)in->stellar_flux[b], F_boa, &o,
                                          cfg->n_iterations, Fu, Fd, Fb);
                else
                    column_mono(L, dtau, w0, g0, B_lo, B_hi, mu, (real)in->stellar_flux[b], F_boa, &o,
                                Fu, Fd, Fb);
                /* O9 reduction: bin weight dlam, Gauss weight w_g; interfaces only */
                const real wgt = dlam * (real)cfg->gauss_w[g];
                const int stride = noniso ? 2 : 1;
                for (int i = 0; i <= N; ++i) {
                    acc_up[i] += wgt * Fu[i * stride];
                    acc_dn[i] += wgt * (Fd[i * stride] + Fb[i * stride]);   /* L235 */
                    acc_bm[i] += wgt * Fb[i * stride];
                }
                toa_bin += (real)cfg->gauss_w[g] * Fu[N * stride];
                if (out->dbg_F_up_pt && c == out->dbg_column)
                    for (int i = 0; i <= N; ++i) {
                        out->dbg_F_up_pt[(size_t)i * npt + b * ng + g] = (double)Fu[i * stride];
                        out->dbg_F_dn_pt[(size_t)i * npt + b * ng + g] = (double)Fd[i * stride];
                    }
            }
            if (out->F_up_toa_bin) out->F_up_toa_bin[(size_t)c * nb + b] = (double)toa_bin;
        }
        for (int i = 0; i <= N; ++i) {
            size_t k = (size_t)c * (N + 1) + i;
            if (out->F_up)   out->F_up[k] = (double)acc_up[i];
            if (out->F_down) out->F_down[k] = (double)acc_dn[i];
            if (out->F_net)  out->F_net[k] = (double)(acc_up[i] - acc_dn[i]);
            if (out->F_beam) out->F_beam[k] = (double)acc_bm[i];
        }
        if (out->dTdt)
            for (int j = 0; j < N; ++j) {                     /* reading R14 */
                real dm = (p_int[j] - p_int[j + 1]) / grav;
                real fn1 = acc_up[j + 1] - acc_dn[j + 1], fn0 = acc_up[j] - acc_dn[j];
                out->dTdt[(size_t)c * N + j] = (double)(-(fn1 - fn0) / ((real)cfg->cp * dm));
            }
        free(buf);
    }
    return 0;
}

int oracle_sizeof_real(void) { return (int)sizeof(real); }
