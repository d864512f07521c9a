// helios_rt.cu -- B200 (sm_100a) implementation of the THOR+HELIOS radiative-transfer step.
//
// C ABI: include/helios_rt.h.  Citations are PAPER.md lines (arXiv 2203.02293).
//
// Two launches per step, both on the caller's stream:
//
//   rt_prep_kernel   (per column) S1 level geometry -- interface p,T, layer masses, k-table cell + corner weights per
//                    level -- and S2 band Planck B_b(T_level); results go to the handle's workspace.
//   rt_solve*_kernel (per spectral point) S3-S7.  A thread block owns one atmospheric column and a tile of its
//                    (bin, Gauss point) spectral points; one thread = one spectral point = one monochromatic
//                    two-stream problem over the column (the unit the paper solves independently, L449/L592) --
//                    or two / four adjacent points of one bin (rt_solve2_kernel / rt_solvem_kernel):
//     sweep 1 (TOA -> BOA): S3 bilinear ln(kappa) interpolation + exp, S4 omega0/g0/dtau, tau prefix and direct beam
//              (Eq. B6), S5 layer coefficients (Eq. 19, B1, B2, B5, B8, Eq. 11 guard) and the forward elimination
//              of S6.  The block-tridiagonal system of Eq.(12) has one non-zero in each off-diagonal 2x2 block, so
//              Eqs.(13)-(14) reduce to the scalar recurrences (R, U, c, d) below; they are carried in registers.
//     sweep 2 (BOA -> TOA): back-substitution Eq.(15) fused with S7, the Gauss-/bin-weighted reduction (warp
//              shuffles, then shared memory, then a fixed-order sum over tiles).
//   rt_iter_kernel   the pair-wise iterative scheme the paper replaces (helios_rt_step_iterative; comparison only).
//
// The layer relations are used in transmission/reflection form.  With zeta+- and T of Eq.(B2),
//   t = psi/chi = s T / (a b),  r = -xi/chi = zeta+ zeta- (1 - T^2) / (a b),
//   a = zeta+ - zeta- T,  b = zeta+ + zeta- T,  s = zeta+ - zeta-,  1 - t - r = s (1 - T) / b,
// Eqs.(2),(3) read  F_up[j+1] = t F_up[j] + r F_dn[j+1] + S_up,  F_dn[j] = t F_dn[j+1] + r F_up[j] + S_dn.
// These forms avoid the cancellations of chi + xi - psi and 1 - T^2.
//
// fp64 throughout.  Reciprocals, reciprocal square roots and exponentials are done with the
// MUFU seed instructions plus Newton/polynomial refinement in FMA (the fp64 pipe is the binding
// resource); helios_rt_selftest_math exposes them to the tests.

#include "../../include/helios_rt.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <type_traits>

namespace {

constexpr int MAXL = HELIOS_RT_MAX_LAYERS;
// unroll factors of the isothermal sweep-1 loop, measured on B200: with the back-substitution
// stack 1 is best (config 2: 0.760 / 0.787 / 0.891 ms at 1 / 2 / 4), the stack-free TOA mode prefers 4 (config 5:
// 5.31 / 5.13 / 4.98 ms)
constexpr int kIsoUnroll = 1, kIsoUnrollToa = 4;
#ifndef HRT_U2
#define HRT_U2 1
#endif
constexpr int kIsoUnrollToa2 = HRT_U2;   // rt_solve2_kernel, TOA mode
constexpr double kPi = 3.14159265358979323846;
constexpr double kH = 6.62607015e-34, kC = 299792458.0, kKB = 1.380649e-23;  // CODATA 2019 (exact)
constexpr double kSigmaSB =
    2.0 * kPi * kPi * kPi * kPi * kPi * kKB * kKB * kKB * kKB / (15.0 * kH * kH * kH * kC * kC);
constexpr double kPlanckC1 = 2.0 * kKB * kKB * kKB * kKB / (kH * kH * kH * kC * kC);  // 2 k^4 / (h^3 c^2)
constexpr double kPlanckC2 = kH * kC / kKB;                                            // h c / k

// --------------------------------------------------------------------------------------------
// fp64 primitives
// --------------------------------------------------------------------------------------------
// MUFU.RCP64H seed (~20 good bits), then y (1 + e + e^2) = (1/x)(1 - e^3): <= 1.5 ulp
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  e = fma(e, e, e);
  return fma(y, e, y);
}

// MUFU.RSQ64H seed, then y (1 + e/2 + 3 e^2/8), e = 1 - x y^2: error O(e^3)
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  const double p = fma(0.375, e, 0.5) * e;
  return fma(y, p, y);
}

// positive, non-NaN doubles order like their bit patterns: comparisons on the integer pipes keep the
// fp64 pipe (the binding resource) for arithmetic
__device__ __forceinline__ bool gt_pos(double a, double b) { return __double_as_longlong(a) > __double_as_longlong(b); }
__device__ __forceinline__ bool abs_lt(double a, double b_pos) {
  return (__double_as_longlong(a) & 0x7fffffffffffffffLL) < __double_as_longlong(b_pos);
}
// min(x, c) for x >= 0, c > 0 on the integer pipes
__device__ __forceinline__ double min_pos(double x, double c) { return gt_pos(x, c) ? c : x; }

// exp by table: e^x = 2^m T[j] (1 + p(r)), k = 32 m + j = round(32 x / ln 2), r = x - k ln2/32, |r| <= ln2/64,
// T[j] = 2^(j/32) (32 doubles in shared memory), p = expm1(r) by its degree-6 Taylor polynomial (remainder
// r^7/5040 < 4e-18).  10 fp64 instructions.  The single-constant reduction k * fl(ln2/32) is exact to
// |k| 2.4e-18, i.e. <= 8e-14 relative at |x| = 700 and <= 3e-15 for |x| <= 30 (far inside the 1e-9 budget).
//   MODE 0: e^x for |x| <= 708;  MODE 1: e^-a, 0 <= a <= 708;  MODE 2: e^-2a, 0 <= a <= 354, and, if OM,
//   *om = 1 - e^-2a without cancellation.
__constant__ double kExp2Tab[32] = {
    1.0, 1.0218971486541166, 1.0442737824274138, 1.0671404006768237,
    1.0905077326652577, 1.1143867425958924, 1.1387886347566916, 1.1637248587775775,
    1.189207115002721, 1.215247359980469, 1.241857812073484, 1.2690509571917332,
    1.2968395546510096, 1.3252366431597413, 1.3542555469368927, 1.383909881963832,
    1.4142135623730951, 1.4451808069770467, 1.4768261459394993, 1.5091644275934228,
    1.5422108254079407, 1.5759808451078865, 1.6104903319492543, 1.645755478153965,
    1.681792830507429, 1.718619298122478, 1.7562521603732995, 1.7947090750031072,
    1.8340080864093424, 1.8741676341103, 1.9152065613971474, 1.9571441241754002};

// --------------------------------------------------------------------------------------------
// S2: band Planck.  G(x) = int_x^inf t^3/(e^t - 1) dt (reading R8).
//   x >= 1.5 : sum_n e^{-n x} (x^3/n + 3 x^2/n^2 + 6 x/n^3 + 6/n^4)
//   x <  1.5 : pi^4/15 - sum_k B_k x^{k+3} / ((k+3) k!)   (Bernoulli numbers B_k)
// --------------------------------------------------------------------------------------------
// *low receives int_0^x t^3/(e^t-1) dt when x < 1.5 (else -1): a bin whose two edges both lie there is
// differenced on `low`, which avoids the cancellation against pi^4/15 for narrow Rayleigh-Jeans bins.
__constant__ double kInvN[33] = {
    0.0, 1.0, 1.0 / 2, 1.0 / 3, 1.0 / 4, 1.0 / 5, 1.0 / 6, 1.0 / 7, 1.0 / 8, 1.0 / 9, 1.0 / 10, 1.0 / 11, 1.0 / 12, 1.0 / 13,
    1.0 / 14, 1.0 / 15, 1.0 / 16, 1.0 / 17, 1.0 / 18, 1.0 / 19, 1.0 / 20, 1.0 / 21, 1.0 / 22, 1.0 / 23, 1.0 / 24, 1.0 / 25,
    1.0 / 26, 1.0 / 27, 1.0 / 28, 1.0 / 29, 1.0 / 30, 1.0 / 31, 1.0 / 32};

__device__ double planck_G(double x, double *low_out) {
  *low_out = -1.0;
  if (!(x > 0.0)) { *low_out = 0.0; return kPi * kPi * kPi * kPi / 15.0; }
  if (x >= 1.5) {
    if (x > 745.0) return 0.0;
    const double u = exp(-x);
    const double x2 = x * x, x3 = x2 * x, c1 = 6.0 * x, c2 = 3.0 * x2;
    double un = 1.0, sum = 0.0;
    // two terms per trip, one convergence test per trip (the terms decrease monotonically)
    for (int n = 1; n <= 32; n += 2) {
      const double in1 = kInvN[n], in2 = kInvN[n + 1];   // 1/n, correctly rounded: same value as the division
      const double un1 = un * u;
      un = un1 * u;
      // x^3/n + 3 x^2/n^2 + 6 x/n^3 + 6/n^4
      const double t1 = un1 * (in1 * fma(in1, fma(in1, fma(in1, 6.0, c1), c2), x3));
      const double t2 = un * (in2 * fma(in2, fma(in2, fma(in2, 6.0, c1), c2), x3));
      sum += t1;
      sum += t2;
      if (t2 < 1e-18 * sum) break;
    }
    return sum;
  }
  // coefficients B_k / ((k+3) k!), k = 0,1,2,4,...,30
  const double c0 = 1.0 / 3.0, c1 = -1.0 / 8.0;
  const double ce[15] = {
      1.0 / 60.0,                                   // k=2 : (1/6)/(5*2)
      -1.0 / 5040.0,                                // k=4 : (-1/30)/(7*24)
      1.0 / 272160.0,                               // k=6 : (1/42)/(9*720)
      -1.0 / 13305600.0,                            // k=8
      1.0 / 622702080.0,                            // k=10
      -691.0 / (2730.0 * 15.0 * 479001600.0),       // k=12
      7.0 / (6.0 * 17.0 * 87178291200.0),           // k=14
      -3617.0 / (510.0 * 19.0 * 20922789888000.0),  // k=16
      43867.0 / (798.0 * 21.0 * 6402373705728000.0),            // k=18
      -174611.0 / (330.0 * 23.0 * 2432902008176640000.0),       // k=20
      854513.0 / (138.0 * 25.0 * 1124000727777607680000.0),     // k=22
      -236364091.0 / (2730.0 * 27.0 * 620448401733239439360000.0),   // k=24
      8553103.0 / (6.0 * 29.0 * 403291461126605635584000000.0),      // k=26
      -23749461029.0 / (870.0 * 31.0 * 304888344611713860501504000000.0),   // k=28
      8615841276005.0 / (14322.0 * 33.0 * 265252859812191058636308480000000.0)  // k=30
  };
  const double x2 = x * x;
  double s = ce[14];
#pragma unroll
  for (int i = 13; i >= 0; --i) s = fma(s, x2, ce[i]);
  // low = x^3 (c0 + c1 x + x^2 s)
  const double low = x2 * x * fma(x2, s, fma(c1, x, c0));
  *low_out = low;
  return kPi * kPi * kPi * kPi / 15.0 - low;
}

// G(x_hi_edge) - G(x_lo_edge) for one bin from the per-edge (G, low) pairs (edge e = lam_lo: larger x)
__device__ __forceinline__ double planck_dG(double G_lo_edge, double low_lo_edge, double G_hi_edge, double low_hi_edge) {
  return (low_lo_edge >= 0.0 && low_hi_edge >= 0.0) ? (low_lo_edge - low_hi_edge) : (G_hi_edge - G_lo_edge);
}

// --------------------------------------------------------------------------------------------
// kernel parameters
// --------------------------------------------------------------------------------------------
struct BinConst {   // per bin, built at create time from scat_gas / cloud_* (Eqs. 17-18)
  double dlam;      // lam_hi - lam_lo
  double inv_dlam;
  double sb[2];     // kappa_ext = kappa_abs + sb[cloudy]
  double ss[2];     // omega0 = ss[cloudy] / kappa_ext
  double gg[2];     // g0 at a clear / cloudy level
};

// S1 result per (column, level), written by rt_prep_kernel, staged in shared memory by rt_solve_kernel
struct __align__(16) LevelRec {
  double c00, c01, c10, c11;  // bilinear weights of the corners (iP,iT), (iP,iT+1), (iP+1,iT), (iP+1,iT+1)
  unsigned o00, o01, o10, o11;  // offsets of the four corner rows (spectral point 0) in the ln(kappa) table, doubles
  double dm;                  // column mass of the (sub-)layer whose lower level this is, kg m^-2
  int cloud;                  // cloud_p_top <= p <= cloud_p_bot
  int pad;
};
static_assert(sizeof(LevelRec) == 64, "LevelRec layout");

struct KParams {
  // create-time tables (device)
  const double *lnk;      // [nP][nT][npt] ln(kappa)
  const double *tab_lp;   // [nP] log10(p)
  const double *tab_t;    // [nT]
  const double *edges;    // [nb+1]
  const double *gauss_w;  // [ng]
  const BinConst *bins;   // [nb]
  int nP, nT, N, nlev, nb, ng, npt, tiles;
  double cloud_p_top, cloud_p_bot, inv_g, inv_cp, inv_eps2, e_tau, gcrit_tol, w0_transition, f_toa;
  int improved;
  // per-step
  const double *p, *T, *mu, *fstar;
  double T_int;
  double *F_up, *F_down, *F_net, *dTdt, *F_beam, *F_toa_bin;
  // workspace
  LevelRec *ws_lev;       // [ncol][nlev+1]   record 0 pads the one-level-ahead prefetch (copy of level 0)
  double *ws_B;           // [ncol][nlev+1][nb] band Planck per level; last row pi B_b(T_int)
  double *ws_dm;          // [ncol][N]        full-layer column mass (heating rate)
  int *ws_nan;            // [ncol]           NaN in p, T of the column
  double *partial;        // [ncol][tiles][4][N+1]
  unsigned *counter;      // [ncol]
};

// constants of the hot loop live in constant memory: an fp64 instruction takes one operand straight from
// the constant bank, so none of them costs a register, a move or a uniform-register rematerialisation
struct HotConst {
  double S, nS, n2S;      // 32/ln2, -32/ln2, -64/ln2
  double nL, hL;          // -ln2/32, ln2/64
  double e6, e5, e4, e3;  // 1/720, 1/120, 1/24, 1/6
  double q4, q3, q2, q1;  // 4/45, -4/15, 2/3, -4/3
  double fa, fb, fc;      // Eq.(19): 1.225 - 0.1582 g - 0.07465 g^2
  double fd, fe, ff;      //          + w (-0.1777 + 0.2351 g - 0.05582 w)
  double pi, npi;
};
__constant__ HotConst kHC = {
    46.16624130844683,     -46.16624130844683,   -92.33248261689366,
    -0.02166084939249829,  0.010830424696249145,
    1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0,
    4.0 / 45.0, -4.0 / 15.0, 2.0 / 3.0, -4.0 / 3.0,
    1.225, -0.1582, -0.07465,
    -0.1777, 0.2351, -0.05582,
    3.14159265358979323846, -3.14159265358979323846};

// exp by table (see kExp2Tab), constants from kHC.
//   MODE 0: e^x for |x| <= 708;  MODE 1: e^-a, 0 <= a <= 708;  MODE 2: e^-2a, 0 <= a <= 354, and, if OM,
//   *om = 1 - e^-2a without cancellation.
template <int MODE, bool OM>
__device__ __forceinline__ double exp_hot(double x, const double *__restrict__ T32, double *om) {
  const double kMagic = 6755399441055744.0;      // 1.5 * 2^52: round-to-nearest-integer trick
  double kd, p;
  if (MODE == 0) kd = fma(x, kHC.S, kMagic);
  else if (MODE == 1) kd = fma(x, kHC.nS, kMagic);
  else kd = fma(x, kHC.n2S, kMagic);
  const int ki = __double2loint(kd);
  const double kf = kd - kMagic;
  if (MODE == 2) {
    // r = -2 x - kf L; with h = -r/2 = x + kf L/2:  p = expm1(-2 h) = h (-2 + h q(h))
    const double h = fma(kf, kHC.hL, x);
    double q = fma(h, kHC.q4, kHC.q3);
    q = fma(q, h, kHC.q2);
    q = fma(q, h, kHC.q1);
    q = fma(q, h, 2.0);
    p = h * fma(h, q, -2.0);
  } else {
    const double r = (MODE == 0) ? fma(kf, kHC.nL, x) : fma(kf, kHC.nL, -x);
    double q = fma(r, kHC.e6, kHC.e5);
    q = fma(q, r, kHC.e4);
    q = fma(q, r, kHC.e3);
    q = fma(q, r, 0.5);
    p = fma(r * r, q, r);
  }
  const double Tj = T32[ki & 31];
  const double Ts = __hiloint2double(__double2hiint(Tj) + ((ki >> 5) << 20), __double2loint(Tj));   // 2^m T[j]
  if (OM) *om = fma(-Ts, p, 1.0 - Ts);
  return fma(Ts, p, Ts);
}


// --------------------------------------------------------------------------------------------
// S5 for one (sub-)layer between a lower level "a" and an upper level "b": transmission t = psi/chi, reflection
// r = -xi/chi and the sources of  F_up[b] = t F_up[a] + r F_dn[b] + S_up,  F_dn[a] = t F_dn[b] + r F_up[a] + S_dn.
// --------------------------------------------------------------------------------------------
// the terms of S5 that depend on the asymmetry factor g0 alone.  On isothermal columns g0 is a per-(bin, cloud flag)
// constant, so they are built once at staging time (BinOpt); non-isothermal sub-layers average g0 and build them here.
struct G0Terms {
  double g0;
  double fg;   // Eq.(19): 1.225 - 0.1582 g0 - 0.07465 g0^2
  double fA;   // Eq.(19): -0.1777 + 0.2351 g0   (fit = fg + w0 (fA - 0.05582 w0))
  double ge;   // g0 / eps2, (B8)
};
__device__ __forceinline__ G0Terms g0_terms(double g0, double inv_eps2) {
  G0Terms t;
  t.g0 = g0;
  t.fg = fma(g0, fma(kHC.fc, g0, kHC.fb), kHC.fa);
  t.fA = fma(g0, kHC.fe, kHC.fd);
  t.ge = g0 * inv_eps2;
  return t;
}

template <bool DAY, bool LINSRC>
__device__ __forceinline__ void layer_coeffs(const KParams &P, const double *__restrict__ T32, double w0, const G0Terms &gt,
                                             double dtau, double Ba, double Bb, double mu, double Fa, double Fb,
                                             double &t_out, double &r_out, double &Sup_out, double &Sdn_out) {
  // E, Eq.(19) L374 (readings R5, R6): E = max(1, fit) if w0 > 0.1 else 1
  const double g0 = gt.g0;
  const double fit = fma(w0, fma(kHC.ff, w0, gt.fA), gt.fg);
  const double E = (P.improved && gt_pos(w0, P.w0_transition) && gt_pos(fit, 1.0)) ? fit : 1.0;
  const double wg = w0 * g0;
  const double num = E - w0;             // E - omega0
  const double den = E * (1.0 - wg);     // E (1 - omega0 g0)
  const double X = num * den;
  const double rs = rsqrt_fast(X);       // 1/sqrt(E (E-w0)(1-w0 g0))
  const double s = num * rs;             // sqrt((E-w0)/(E(1-w0 g0))) = zeta+ - zeta-   (B2)
  const double ha = X * rs;              // alpha / 2 = sqrt(E (E-w0)(1-w0 g0))
  const double rs2 = rs * rs;
  const double zp = fma(0.5, s, 0.5), zm = fma(-0.5, s, 0.5);
  double omT;
  const double Tr = exp_hot<2, true>(min_pos(ha * dtau, 354.0), T32, &omT);   // transmission function (B2), 1 - T
  const double zmT = zm * Tr;
  const double a = zp - zmT, b = zp + zmT;
  const double inv_ab = rcp_fast(a * b);
  const double u = omT * inv_ab;
  const double t = (s * Tr) * inv_ab;                        // psi/chi
  const double r = (zp * zm) * (1.0 + Tr) * u;               // -xi/chi
  const double emis = (s * a) * u;                           // 1 - t - r
  const double Pi = fma(kHC.npi, w0, kHC.pi) * (den * rs2);  // (B5): pi (1-w0)/(E-w0)
  double Sup, Sdn;
  if (LINSRC) {
    // Eqs.(4)-(9): B* (1-r) - t B*' +- B' (1 - t + r)/(2E(1-w0 g0)), B' = (Ba - Bb)/dtau; e_tau rule L209
    const bool thin = !gt_pos(dtau, P.e_tau) && dtau != P.e_tau;   // dtau < e_tau
    const double Bm = 0.5 * (Ba + Bb);
    const double dB = thin ? 0.0 : (Ba - Bb);
    const double Bal = thin ? Bm : Ba, Bbl = thin ? Bm : Bb;
    const double invP = 0.5 * (num * rs2);                   // 1 / (2 E (1 - w0 g0))
    const double grad = (1.0 - t + r) * invP * rcp_fast(dtau);
    const double k = dB * (t - grad);
    Sup = Pi * fma(Bbl, emis, -k);
    Sdn = Pi * fma(Bal, emis, k);
  } else {
    Sup = Sdn = (Pi * Bb) * emis;                            // Eqs.(2),(3)
  }
  if (DAY) {
    // (B8) with mu_star = -mu; guard of Eq.(11)/L252 (reading R4)
    const double ma = mu * (2.0 * ha);
    double D = (ma - 1.0) * (ma + 1.0);                      // 4 E mu^2 (E-w0)(1-w0 g0) - 1
    D = abs_lt(D, P.gcrit_tol) ? -2.0 * mu : D;
    const double invD = rcp_fast(D);
    const double hP = 0.5 * (num * rs2);                     // 1 / (2 E (1 - w0 g0))
    const double ge = gt.ge;
    const double lead = (0.5 * w0) * fma(2.0, den, ge) * invD;
    const double last = (0.5 * w0) * ge * hP;
    const double Gp = fma(lead, hP - mu, last);
    const double Gm = -fma(lead, hP + mu, last);
    // (B7): S_up += t G+ Fa + r G- Fb - G+ Fb ; S_dn += t G- Fb + r G+ Fa - G- Fa
    const double rGm = r * Gm, rGp = r * Gp;
    Sup = fma(rGm, Fb, fma(Gp, fma(t, Fa, -Fb), Sup));
    Sdn = fma(rGp, Fa, fma(Gm, fma(t, Fb, -Fa), Sdn));
  }
  t_out = t; r_out = r; Sup_out = Sup; Sdn_out = Sdn;
}

// S5 + S6 forward step: layer_coeffs, then the forward elimination.
// In: (R, U) at the upper level: F_dn[b] = R F_up[b] + U.   Out: (R, U) at the lower level and the
// back-substitution pair (c, d): F_up[b] = c F_up[a] + d.
template <bool DAY, bool LINSRC>
__device__ __forceinline__ void layer_forward(const KParams &P, const double *__restrict__ T32, double w0, const G0Terms &gt,
                                              double dtau, double Ba, double Bb, double mu, double Fa, double Fb,
                                              double &R, double &U, double &c, double &d) {
  double t, r, Sup, Sdn;
  layer_coeffs<DAY, LINSRC>(P, T32, w0, gt, dtau, Ba, Bb, mu, Fa, Fb, t, r, Sup, Sdn);
  // forward elimination (Eqs. 13-14 specialised): F_up[b] (1 - r R) = t F_up[a] + r U + S_up
  const double q = rcp_fast(fma(-r, R, 1.0));
  c = t * q;
  d = fma(r, U, Sup) * q;
  const double Rn = fma(t * c, R, r);
  const double Un = fma(c, fma(R, Sup, U), Sdn);
  R = Rn;
  U = Un;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum each of the 16 values v[0..15] over the 32 lanes of the warp by recursive halving: 16 shuffle+add
// steps instead of 16 x 5.  Returns, in lanes L and L^1, the total of v[L >> 1].  Fixed order: deterministic.
__device__ __forceinline__ double warp_reduce16(double (&v)[16], int lane) {
  const unsigned full = 0xffffffffu;
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4, b1 = lane & 2;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const double send = b4 ? v[i] : v[i + 8], keep = b4 ? v[i + 8] : v[i];
    v[i] = keep + __shfl_xor_sync(full, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const double send = b3 ? v[i] : v[i + 4], keep = b3 ? v[i + 4] : v[i];
    v[i] = keep + __shfl_xor_sync(full, send, 8);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const double send = b2 ? v[i] : v[i + 2], keep = b2 ? v[i + 2] : v[i];
    v[i] = keep + __shfl_xor_sync(full, send, 4);
  }
  {
    const double send = b1 ? v[0] : v[1], keep = b1 ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(full, send, 2);
  }
  return v[0] + __shfl_xor_sync(full, v[0], 1);
}

template <bool DAY, bool LINSRC>
__device__ __forceinline__ void layer_forward(const KParams &P, const double *__restrict__ T32, double w0, double g0,
                                              double dtau, double Ba, double Bb, double mu, double Fa, double Fb,
                                              double &R, double &U, double &c, double &d) {
  layer_forward<DAY, LINSRC>(P, T32, w0, g0_terms(g0, P.inv_eps2), dtau, Ba, Bb, mu, Fa, Fb, R, U, c, d);
}
template <bool DAY, bool LINSRC>
__device__ __forceinline__ void layer_coeffs(const KParams &P, const double *__restrict__ T32, double w0, double g0,
                                             double dtau, double Ba, double Bb, double mu, double Fa, double Fb,
                                             double &t_out, double &r_out, double &Sup_out, double &Sdn_out) {
  layer_coeffs<DAY, LINSRC>(P, T32, w0, g0_terms(g0, P.inv_eps2), dtau, Ba, Bb, mu, Fa, Fb, t_out, r_out, Sup_out, Sdn_out);
}

// --------------------------------------------------------------------------------------------
// rt_prep_kernel: S1 (level geometry, k-table cell + weights per level) and S2 (band Planck per level
// and bin) for every column.  Grid = (bin chunks of PREP_BINS, columns).  Results go to the handle's
// workspace (a few tens of MB, L2-resident when rt_solve_kernel reads them back).
// --------------------------------------------------------------------------------------------
constexpr int PREP_BLOCK = 256, PREP_BINS = 32;

__host__ __device__ inline size_t prep_smem_bytes(int N, int nlev) {
  return sizeof(double) * ((size_t)N + 2 * (N + 1) + (nlev + 1) + 2 * (size_t)(nlev + 1) * (PREP_BINS + 1));
}

template <bool NONISO>
__global__ void __launch_bounds__(PREP_BLOCK) rt_prep_kernel(const KParams P) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int N = P.N, nlev = P.nlev;
  double *s_lnp = (double *)smem;                       // [N]
  double *s_pint = s_lnp + N;                           // [N+1]
  double *s_tint = s_pint + (N + 1);                    // [N+1]
  double *s_tlev = s_tint + (N + 1);                    // [nlev+1], last = internal temperature
  double *s_G = s_tlev + (nlev + 1);                    // [nlev+1][PREP_BINS+1]
  double *s_Glow = s_G + (size_t)(nlev + 1) * (PREP_BINS + 1);
  __shared__ int s_nan;
  __shared__ short s_rep[2 * MAXL + 2];

  const int tid = threadIdx.x;
  const int chunk = blockIdx.x, col = blockIdx.y;
  const double *pc = P.p + (size_t)col * N;
  const double *Tc = P.T + (size_t)col * N;
  const int b0 = chunk * PREP_BINS;
  const int nbc = (P.nb - b0 < PREP_BINS) ? (P.nb - b0) : PREP_BINS;

  // NaN in p, T or mu of this column poisons the column's outputs (and only them): the clamps and
  // selects below would otherwise swallow it.
  if (tid == 0) { const double mu = P.mu[col]; s_nan = (mu != mu) ? 1 : 0; }
  __syncthreads();
  // ---------------- S1: level geometry (reading R9; L171) ----------------
  for (int j = tid; j < N; j += PREP_BLOCK) {
    const double pj = pc[j], tj = Tc[j];
    if (pj != pj || tj != tj) s_nan = 1;
    s_lnp[j] = log(pj);
  }
  __syncthreads();
  for (int i = tid; i <= N; i += PREP_BLOCK) {
    double lp, ti;
    if (N == 1) {
      lp = s_lnp[0] + (i == 0 ? 0.5 : -0.5) * 2.302585092994045684;
      ti = Tc[0];
    } else if (i == 0) {
      lp = s_lnp[0] + 0.5 * (s_lnp[0] - s_lnp[1]);
      ti = Tc[0];
    } else if (i == N) {
      lp = s_lnp[N - 1] - 0.5 * (s_lnp[N - 2] - s_lnp[N - 1]);
      ti = Tc[N - 1];
    } else {
      lp = 0.5 * (s_lnp[i - 1] + s_lnp[i]);
      ti = 0.5 * (Tc[i - 1] + Tc[i]);
    }
    s_pint[i] = exp(lp);
    s_tint[i] = ti;
  }
  __syncthreads();
  auto p_level = [&](int l) -> double {
    if (NONISO) return (l & 1) ? pc[l >> 1] : s_pint[l >> 1];
    return pc[l];
  };
  for (int l = tid; l <= nlev; l += PREP_BLOCK) {
    if (l == nlev) { s_tlev[l] = P.T_int; continue; }
    const double pl = p_level(l);
    const double tl = NONISO ? ((l & 1) ? Tc[l >> 1] : s_tint[l >> 1]) : Tc[l];
    s_tlev[l] = tl;
    if (chunk != 0) continue;
    LevelRec rec;
    rec.cloud = (pl >= P.cloud_p_top && pl <= P.cloud_p_bot) ? 1 : 0;
    // table cell + weights: bilinear in (log10 p, T), clamped (reading R7)
    double xp = log10(pl);
    xp = fmin(fmax(xp, P.tab_lp[0]), P.tab_lp[P.nP - 1]);
    int ip = 0;
    while (ip < P.nP - 2 && xp > P.tab_lp[ip + 1]) ++ip;
    const double wp = (xp - P.tab_lp[ip]) / (P.tab_lp[ip + 1] - P.tab_lp[ip]);
    const double xt = fmin(fmax(tl, P.tab_t[0]), P.tab_t[P.nT - 1]);
    int it = 0;
    while (it < P.nT - 2 && xt > P.tab_t[it + 1]) ++it;
    const double wt = (xt - P.tab_t[it]) / (P.tab_t[it + 1] - P.tab_t[it]);
    rec.c00 = (1.0 - wp) * (1.0 - wt);
    rec.c01 = (1.0 - wp) * wt;
    rec.c10 = wp * (1.0 - wt);
    rec.c11 = wp * wt;
    rec.o00 = (unsigned)(ip * P.nT + it) * (unsigned)P.npt;
    rec.o01 = rec.o00 + (unsigned)P.npt;
    rec.o10 = rec.o00 + (unsigned)P.nT * (unsigned)P.npt;
    rec.o11 = rec.o10 + (unsigned)P.npt;
    rec.pad = 0;
    // column mass below this level down to the next level: full layer (isothermal: level = layer centre,
    // mass between its two interfaces) or sub-layer (non-isothermal: levels alternate interface / centre)
    if (NONISO) rec.dm = (l < nlev - 1) ? (pl - p_level(l + 1)) * P.inv_g : 0.0;
    else rec.dm = (s_pint[l] - s_pint[l + 1]) * P.inv_g;
    LevelRec *dst = P.ws_lev + (size_t)col * (nlev + 1) + 1 + l;
    *dst = rec;
    if (l == 0) dst[-1] = rec;
  }
  if (chunk == 0)
    for (int j = tid; j < N; j += PREP_BLOCK) P.ws_dm[(size_t)col * N + j] = (s_pint[j] - s_pint[j + 1]) * P.inv_g;
  __syncthreads();
  if (chunk == 0 && tid == 0) P.ws_nan[col] = s_nan;

  // ---------------- S2: band Planck for this chunk's bins (reading R8) ----------------
  // a level whose temperature equals that of the level below it (an isothermal stretch, e.g. the extension above the
  // model top, L385) shares that level's cumulative integrals: s_rep[l] = first level of the run
  const int nedge = nbc + 1;
  if (tid == 0) {
    s_rep[0] = 0;
    for (int l = 1; l <= nlev; ++l) s_rep[l] = (s_tlev[l] == s_tlev[l - 1]) ? s_rep[l - 1] : l;
  }
  __syncthreads();
  // warp w takes levels w, w + 8, ...; lane e takes edge e of the chunk (no integer division, one edge per lane);
  // the chunk's last edge (index 32) is done afterwards, one level per thread
  const int wrp = tid >> 5, lane = tid & 31;
  {
    const double lam_e = (lane < nedge) ? P.edges[b0 + lane] : 1.0;
    for (int l = wrp; l <= nlev; l += PREP_BLOCK / 32) {
      if (s_rep[l] != l || lane >= nedge) continue;
      const double Tl = s_tlev[l];
      double low = 0.0;
      s_G[l * (PREP_BINS + 1) + lane] = (Tl > 0.0) ? planck_G(kPlanckC2 / (lam_e * Tl), &low) : 0.0;
      s_Glow[l * (PREP_BINS + 1) + lane] = low;
    }
    if (nedge == PREP_BINS + 1) {
      const double lam_last = P.edges[b0 + PREP_BINS];
      for (int l = tid; l <= nlev; l += PREP_BLOCK) {
        if (s_rep[l] != l) continue;
        const double Tl = s_tlev[l];
        double low = 0.0;
        s_G[l * (PREP_BINS + 1) + PREP_BINS] = (Tl > 0.0) ? planck_G(kPlanckC2 / (lam_last * Tl), &low) : 0.0;
        s_Glow[l * (PREP_BINS + 1) + PREP_BINS] = low;
      }
    }
  }
  __syncthreads();
  if (lane < nbc) {
    const double inv_dlam = P.bins[b0 + lane].inv_dlam;
    double *dst = P.ws_B + (size_t)col * (nlev + 1) * P.nb + b0 + lane;
    for (int l = wrp; l <= nlev; l += PREP_BLOCK / 32) {
      const double Tl = s_tlev[l];
      const double T2 = Tl * Tl;
      const double *g = s_G + s_rep[l] * (PREP_BINS + 1) + lane;
      const double *gl = s_Glow + s_rep[l] * (PREP_BINS + 1) + lane;
      double B = kPlanckC1 * T2 * T2 * planck_dG(g[0], gl[0], g[1], gl[1]) * inv_dlam;
      if (l == nlev) B *= kPi;   // F_BOA = pi B(T_int), L239
      dst[(size_t)l * P.nb] = (Tl > 0.0) ? B : 0.0;
    }
  }
}

// --------------------------------------------------------------------------------------------
// rt_solve_kernel: S3-S7.  Grid = (tiles per column, columns); a block owns one column and a tile of
// BLOCK consecutive spectral points (bin-major, Gauss point fastest); one thread = one spectral point.
// --------------------------------------------------------------------------------------------
constexpr int STAGE_LD = 36;   // row stride (doubles) of the per-warp 8 x 32 staging tile: conflict-free transpose

// per bin of the tile: [0][bin] clear level, [1][bin] cloudy level.  gt: the g0-only terms of S5 (G0Terms)
struct __align__(16) BinOpt { double sb, ss; G0Terms gt; double pad[2]; };
static_assert(sizeof(BinOpt) == 64, "BinOpt layout");

struct SolveSmem {
  int nbt;         // max bins per tile
  int LP;          // N + 1 rounded up to a multiple of 8 (the reductions handle 8 levels at a time)
  size_t off_lev, off_B, off_bin, off_red, off_stage, off_fin, off_vals, total;
};

__host__ __device__ inline SolveSmem solve_smem(int N, int nlev, int block, int ng, int nb, bool toa, bool bdirect = false,
                                                int ppt = 1) {
  SolveSmem L;
  int nbt = (block * ppt + ng - 1) / ng + 1;   // ppt: spectral points per thread (rt_solve2_kernel: 2)
  L.nbt = nbt < nb ? nbt : nb;
  L.LP = (N + 1 + 7) & ~7;
  const int nwarp = (block + 31) / 32;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o += (bytes + 15) & ~size_t(15); return r; };
  L.off_lev = take(sizeof(LevelRec) * (nlev + 1));
  L.off_B = take(bdirect ? 0 : sizeof(double) * (nlev + 1) * L.nbt);   // bdirect: B read straight from the workspace
  L.off_bin = take(sizeof(BinOpt) * 2 * L.nbt);
  L.off_red = take(toa ? 0 : sizeof(double) * nwarp * 4 * L.LP);       // F_up, R F_up, U + beam, beam
  L.off_stage = take(toa ? 0 : sizeof(double) * nwarp * 8 * STAGE_LD);
  L.off_fin = take(toa ? 0 : sizeof(double) * 4 * (N + 1));
  L.off_vals = take(sizeof(double) * block * ppt);
  L.total = o;
  return L;
}

struct Rows { double l00, l01, l10, l11; };   // the four k-table corner values of one (level, point)

// address of element `off` (32-bit, unsigned) of a double array: one IMAD.WIDE.U32
__device__ __forceinline__ const double *elem_addr(const double *base, unsigned off) {
  unsigned long long a;
  asm("mad.wide.u32 %0, %1, 8, %2;" : "=l"(a) : "r"(off), "l"((unsigned long long)base));
  return (const double *)a;
}

__device__ __forceinline__ Rows load_rows(const double *__restrict__ lnk_pt, const LevelRec *lv) {
  const uint4 o = *reinterpret_cast<const uint4 *>(&lv->o00);
  Rows r;
  r.l00 = __ldg(elem_addr(lnk_pt, o.x));
  r.l01 = __ldg(elem_addr(lnk_pt, o.y));
  r.l10 = __ldg(elem_addr(lnk_pt, o.z));
  r.l11 = __ldg(elem_addr(lnk_pt, o.w));
  return r;
}


// optical properties at one level (S3 + Eqs. 17-18): bilinear ln(kappa) from the four corner rows with the
// level's corner weights, exp, then kappa_ext, omega0, g0.  bin0 / bin1: the point's BinOpt for clear / cloudy.
__device__ __forceinline__ void level_optics(const Rows &rw, const double *__restrict__ T32, const LevelRec *lv,
                                             const BinOpt *bin0, const BinOpt *bin1, double &kx, double &w0,
                                             double &g0) {
  const double2 ca = *reinterpret_cast<const double2 *>(&lv->c00);
  const double2 cb = *reinterpret_cast<const double2 *>(&lv->c10);
  const double lk = fma(cb.y, rw.l11, fma(cb.x, rw.l10, fma(ca.y, rw.l01, ca.x * rw.l00)));
  const double kabs = exp_hot<0, false>(lk, T32, nullptr);
  const BinOpt *bo = lv->cloud ? bin1 : bin0;
  const double2 sbss = *reinterpret_cast<const double2 *>(&bo->sb);
  kx = kabs + sbss.x;
  w0 = sbss.y * rcp_fast(kx);
  g0 = bo->gt.g0;
}

// sum over the warp's lanes of the 8 staged rows (one per interface); row k of the tile belongs to interface
// base + k.  Lane L sums 8 entries of row L >> 2, two shuffle steps finish the row.  Fixed order.
__device__ __forceinline__ void flush_stage(const double *__restrict__ stage_w, double *__restrict__ dst, int lane) {
  __syncwarp();
  const double *row = stage_w + (lane >> 2) * STAGE_LD + (lane & 3);
  double s = row[0];
#pragma unroll
  for (int i = 1; i < 8; ++i) s += row[4 * i];
  s += __shfl_xor_sync(0xffffffffu, s, 1);
  s += __shfl_xor_sync(0xffffffffu, s, 2);
  if ((lane & 3) == 0) dst[lane >> 2] = s;
  __syncwarp();
}

// stage the column's level records, the tile's Planck values and per-bin optical constants in shared memory
template <int BLOCK>
__device__ __forceinline__ void stage_column(const KParams &P, const SolveSmem &L, unsigned char *smem, double *s_T32,
                                             int col, int b_first, int nbt, int tid, bool stage_B = true) {
  const int nlev = P.nlev, nbtS = L.nbt;
  double *s_B = (double *)(smem + L.off_B);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  if (tid < 32) s_T32[tid] = kExp2Tab[tid];
  {
    const double *src = (const double *)(P.ws_lev + (size_t)col * (nlev + 1));
    double *dst = (double *)(smem + L.off_lev);
    for (int i = tid; i < 8 * (nlev + 1); i += BLOCK) dst[i] = src[i];
    const double *gB = P.ws_B + (size_t)col * (nlev + 1) * P.nb + b_first;
    if (stage_B)
      for (int i = tid; i < (nlev + 1) * nbt; i += BLOCK) {
        const int l = i / nbt, k = i - l * nbt;
        s_B[l * nbtS + k] = gB[(size_t)l * P.nb + k];
      }
    for (int i = tid; i < 2 * nbt; i += BLOCK) {
      const int cl = i / nbt, k = i - cl * nbt;
      const BinConst bc = P.bins[b_first + k];
      BinOpt bo;
      bo.sb = bc.sb[cl]; bo.ss = bc.ss[cl]; bo.gt = g0_terms(bc.gg[cl], P.inv_eps2); bo.pad[0] = bo.pad[1] = 0.0;
      s_bin[cl * nbtS + k] = bo;
    }
  }
}

// cross-warp sum of the per-warp interface sums (s_red: [warp][4][LP] = F_up, diffuse F_dn part 1, part 2 (+ beam),
// beam), tile partials in fixed order, and the column's outputs written by its last tile
template <int BLOCK>
__device__ __forceinline__ void column_epilogue(const KParams &P, const SolveSmem &L, double *s_red, double *s_fin,
                                                int *s_is_last_p, int nwa, bool want_beam, int col, int tile, int col_nan) {
  const int N = P.N, LP = L.LP, tid = threadIdx.x;
  int &s_is_last = *s_is_last_p;
  // cross-warp sum in fixed order -> tile partial: F_up, R F_up, U + beam, beam
  const int nq = want_beam ? 4 : 3;
  const int nred = nq * (N + 1);
  for (int k = tid; k < nred; k += BLOCK) {
    const int q = k / (N + 1), lev = k - q * (N + 1);
    double sum = 0.0;
    for (int w = 0; w < nwa; ++w) sum += s_red[(size_t)w * 4 * LP + q * LP + lev];
    s_fin[k] = sum;
  }
  __syncthreads();

  if (P.tiles > 1) {
    // publish the tile partial; the last tile of the column to arrive sums them in tile order
    double *part = P.partial + ((size_t)col * P.tiles + tile) * 4 * (N + 1);
    for (int k = tid; k < nred; k += BLOCK) part[k] = s_fin[k];
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      const unsigned prev = atomicAdd(P.counter + col, 1u);
      s_is_last = (prev == (unsigned)(P.tiles - 1));
      if (s_is_last) P.counter[col] = 0;   // re-arm for the next step
    }
    __syncthreads();
    if (!s_is_last) return;
    __threadfence();
    const double *pall = P.partial + (size_t)col * P.tiles * 4 * (N + 1);
    for (int k = tid; k < nred; k += BLOCK) {
      double sum = 0.0;
      for (int t = 0; t < P.tiles; ++t) sum += __ldcg(pall + (size_t)t * 4 * (N + 1) + k);
      s_fin[k] = sum;
    }
    __syncthreads();
  }

  // final outputs of the column: F_down = sum W R F_up + sum W (U + beam)
  const double poison = col_nan ? nan("") : 0.0;
  for (int i = tid; i <= N; i += BLOCK) {
    const size_t o = (size_t)col * (N + 1) + i;
    const double fu = s_fin[i] + poison, fd = s_fin[N + 1 + i] + s_fin[2 * (N + 1) + i] + poison;
    if (P.F_up) P.F_up[o] = fu;
    if (P.F_down) P.F_down[o] = fd;
    if (P.F_net) P.F_net[o] = fu - fd;
    if (want_beam) P.F_beam[o] = s_fin[3 * (N + 1) + i] + poison;
  }
  if (P.dTdt) {
    const double *dm = P.ws_dm + (size_t)col * N;
    for (int j = tid; j < N; j += BLOCK) {
      const double fn1 = s_fin[j + 1] - (s_fin[N + 1 + j + 1] + s_fin[2 * (N + 1) + j + 1]);
      const double fn0 = s_fin[j] - (s_fin[N + 1 + j] + s_fin[2 * (N + 1) + j]);
      P.dTdt[(size_t)col * N + j] = -(fn1 - fn0) * P.inv_cp / dm[j] + poison;   // reading R14
    }
  }
}

template <bool NONISO, bool TOA, bool BDIRECT, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) rt_solve_kernel(const KParams P) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ double s_T32[32];
  __shared__ int s_is_last;
  const int N = P.N, nlev = P.nlev;
  // one Gauss point per bin (opacity sampling, L385): every thread has its own bin, so the Planck values are read
  // coalesced straight from the workspace instead of being staged (64 KB per block otherwise)
  constexpr bool bdirect = BDIRECT;   // host: n_gauss == 1
  const SolveSmem L = solve_smem(N, nlev, BLOCK, P.ng, P.nb, TOA, bdirect);
  const LevelRec *s_lev = (const LevelRec *)(smem + L.off_lev) + 1;   // s_lev[-1] pads the prefetch
  double *s_B = (double *)(smem + L.off_B);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  double *s_red = (double *)(smem + L.off_red);
  double *s_stage = (double *)(smem + L.off_stage);
  double *s_fin = (double *)(smem + L.off_fin);
  double *s_vals = (double *)(smem + L.off_vals);

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, col = blockIdx.y;
  const int LP = L.LP, nbtS = L.nbt;
  const double mu = P.mu[col];
  const bool day = mu > 0.0;

  const int pt0 = tile * BLOCK;
  const int b_first = pt0 / P.ng;
  int pt_last = pt0 + BLOCK - 1;
  if (pt_last > P.npt - 1) pt_last = P.npt - 1;
  const int nbt = pt_last / P.ng - b_first + 1;   // bins touched by this tile (<= L.nbt)
  const int nwa = ((pt_last - pt0) >> 5) + 1;     // warps of this tile that own at least one spectral point

  stage_column<BLOCK>(P, L, smem, s_T32, col, b_first, nbt, tid, !bdirect);
  const int col_nan = P.ws_nan[col];
  __syncthreads();

  // ---------------- per-thread constants ----------------
  int pt = pt0 + tid;
  const bool active = pt < P.npt;
  if (!active) pt = P.npt - 1;
  const int b = pt / P.ng, gidx = pt - b * P.ng;
  const int bl = b - b_first;
  const int warp = tid >> 5, lane = tid & 31;
  const bool warp_on = warp < nwa;          // a warp without any spectral point only joins the barriers
  double *red_w = s_red + (size_t)warp * 4 * LP;
  double *stage_w = s_stage + (size_t)warp * 8 * STAGE_LD;
  const bool want_beam = !TOA && (P.F_beam != nullptr);

  if (warp_on) {
    const double W = active ? P.bins[b].dlam * P.gauss_w[gidx] : 0.0;    // dlam_b * w_g
    const double muF = day ? mu * P.fstar[b] : 0.0;                      // mu * F_star[b]
    const double inv_mu = day ? 1.0 / mu : 0.0;
    const double *lnk_pt = P.lnk + pt;
    const BinOpt *bin0 = s_bin + bl, *bin1 = s_bin + nbtS + bl;
    const double *T32 = s_T32;
    double *stage_wr = stage_w + lane;
    // B of level l: Bbase[l * Bstride] (global workspace row, or the staged tile in shared memory)
    const double *Bbase = s_B + bl;
    if (BDIRECT) Bbase = P.ws_B + (size_t)col * (nlev + 1) * P.nb + b;
    const int Bstride = BDIRECT ? P.nb : nbtS;

    // back-substitution state per interface i = 0..N (thread-private stack in local memory, written top-down,
    // read bottom-up): F_up[i] = c F_up[i-1] + d (weight folded into d) and R with F_dn[i] = R F_up[i] + U.
    // U itself is not kept: sum_points W (U + beam) is reduced on the way down (flush_stage).
    // Entries N+1 .. LP-1 pad the last group of 8 in sweep 2 with the identity (c = 1, d = 0, R = 0).
    constexpr int STK = TOA ? 1 : ((MAXL + 1 + 7) & ~7);
    double2 st_cd[STK];
    double st_R[STK];

    double R = 0.0, U = P.f_toa;       // F_dn[N] = f_toa (Fig. 5)
    double Fb = muF;                   // beam at the TOA (full strength, L235)
    double Ctoa = 1.0, Dtoa = 0.0;     // TOA mode: F_up[N] = Ctoa F_up[j] + Dtoa

    // bookkeeping of interface i with (R, U, Fb) at that interface
    auto push_interface = [&](int i, double Ri, double Ui, double Fbi) {
      if (!TOA) {
        st_R[i] = Ri;
        stage_wr[(i & 7) * STAGE_LD] = W * (Ui + Fbi);
        if ((i & 7) == 0) flush_stage(stage_w, red_w + 2 * LP + i, lane);
        if (want_beam) {
          const double wb = warp_sum(W * Fbi);
          if (lane == 0) red_w[3 * LP + i] = wb;
        }
      }
    };

    // ---------------- sweep 1: TOA -> BOA (one instantiation per day / night: the loop body has no branch) ------
    auto sweep1 = [&](auto day_tag) {
      constexpr bool DAY = decltype(day_tag)::value;
      double tau = 0.0;
      if (!NONISO) {
        const LevelRec *lv = s_lev + (N - 1);
        const double *Bp = Bbase + (size_t)(N - 1) * Bstride;
        Rows nx = load_rows(lnk_pt, lv);   // rows of the next level, loaded one level ahead
#pragma unroll (TOA ? kIsoUnrollToa : kIsoUnroll)
        for (int j = N - 1; j >= 0; --j, --lv, Bp -= Bstride) {
          const Rows cur = nx;
          nx = load_rows(lnk_pt, lv - 1);
          push_interface(j + 1, R, U, Fb);
          double kx, w0, g0, c, d;
          level_optics(cur, T32, lv, bin0, bin1, kx, w0, g0);
          const double dtau = kx * lv->dm;
          const double Bj = *Bp;
          double Fa = 0.0;
          if (DAY) {
            tau += dtau;
            Fa = muF * exp_hot<1, false>(min_pos(tau * inv_mu, 708.0), T32, nullptr);   // (B6)
          }
          layer_forward<DAY, false>(P, T32, w0, g0, dtau, Bj, Bj, mu, Fa, Fb, R, U, c, d);
          Fb = Fa;
          if (TOA) {
            Dtoa = fma(Ctoa, d, Dtoa);
            Ctoa *= c;
          } else {
            st_cd[j + 1] = make_double2(c, W * d);
          }
        }
      } else {
        // levels alternate interface (even) / centre (odd); sub-layer s lies between levels s and s+1 and takes
        // the arithmetic mean of the two levels' kappa_ext, omega0, g0 (L171, reading R10).  The centre unknowns
        // are eliminated on the fly: F_up[j+1] = cu F_up[centre] + du, F_up[centre] = cl F_up[j] + dl.
        const LevelRec *lv = s_lev + (nlev - 1);
        const double *Bp = Bbase + (size_t)(nlev - 1) * Bstride;
        double kx_up, w0_up, g0_up;
        {
          const Rows top = load_rows(lnk_pt, lv);
          level_optics(top, T32, lv, bin0, bin1, kx_up, w0_up, g0_up);
        }
        double B_up = *Bp;
        Rows nxc = load_rows(lnk_pt, lv - 1);   // centre and lower interface of the next layer, one layer ahead
        Rows nxl = load_rows(lnk_pt, lv - 2);
#pragma unroll 1
        for (int j = N - 1; j >= 0; --j, lv -= 2, Bp -= 2 * Bstride) {
          const Rows rc = nxc, rl = nxl;
          nxc = load_rows(lnk_pt, lv - 3);
          nxl = load_rows(lnk_pt, (j > 0) ? lv - 4 : lv - 3);
          push_interface(j + 1, R, U, Fb);
          double kx_c, w0_c, g0_c, kx_lo, w0_lo, g0_lo, cu, du, cl, dl;
          level_optics(rc, T32, lv - 1, bin0, bin1, kx_c, w0_c, g0_c);
          level_optics(rl, T32, lv - 2, bin0, bin1, kx_lo, w0_lo, g0_lo);
          const double B_c = Bp[-Bstride], B_lo = Bp[-2 * Bstride];
          const double dtau_u = 0.5 * (kx_c + kx_up) * lv[-1].dm;
          const double dtau_l = 0.5 * (kx_lo + kx_c) * lv[-2].dm;
          double Fc = 0.0, Fa = 0.0;
          if (DAY) {
            const double tau_c = tau + dtau_u;
            tau = tau_c + dtau_l;
            Fc = muF * exp_hot<1, false>(min_pos(tau_c * inv_mu, 708.0), T32, nullptr);   // (B6)
            Fa = muF * exp_hot<1, false>(min_pos(tau * inv_mu, 708.0), T32, nullptr);
          }
          layer_forward<DAY, true>(P, T32, 0.5 * (w0_c + w0_up), 0.5 * (g0_c + g0_up), dtau_u, B_c, B_up, mu, Fc, Fb,
                                   R, U, cu, du);
          layer_forward<DAY, true>(P, T32, 0.5 * (w0_lo + w0_c), 0.5 * (g0_lo + g0_c), dtau_l, B_lo, B_c, mu, Fa, Fc,
                                   R, U, cl, dl);
          Fb = Fa;
          kx_up = kx_lo; w0_up = w0_lo; g0_up = g0_lo; B_up = B_lo;
          const double cc = cu * cl, dd = fma(cu, dl, du);
          if (TOA) {
            Dtoa = fma(Ctoa, dd, Dtoa);
            Ctoa *= cc;
          } else {
            st_cd[j + 1] = make_double2(cc, W * dd);
          }
        }
      }
    };
    if (day) sweep1(std::true_type{}); else sweep1(std::false_type{});

    // ---------------- BOA, Eq.(10) L237 ----------------
    const double F_boa = Bbase[(size_t)nlev * Bstride];
    const double Fup0 = (U + F_boa + Fb) * rcp_fast(1.0 - R);

    if (TOA) {
      // S7 (spectrum shape): F_up_toa_bin[b] = sum_g w_g F_up[N]
      const double FupN = fma(Ctoa, Fup0, Dtoa);
      s_vals[tid] = active ? P.gauss_w[gidx] * FupN : 0.0;
    } else {
      push_interface(0, R, U, Fb);
      st_cd[0] = make_double2(0.0, W * Fup0);
      // ---------------- sweep 2: back-substitution Eq.(15) + S7 reduction, 8 interfaces at a time ----------------
      for (int i = N + 1; i < LP; ++i) { st_cd[i] = make_double2(1.0, 0.0); st_R[i] = 0.0; }
      double wFup = 0.0;
#pragma unroll 1
      for (int base = 0; base <= N; base += 8) {
        double v[16];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          // levels beyond N repeat F_up[N] into rows of the reduction buffer that are never read
          const double2 cd = st_cd[base + k];
          const double Ri = st_R[base + k];
          wFup = fma(cd.x, wFup, cd.y);
          v[k] = wFup;
          v[8 + k] = Ri * wFup;
        }
        const double tot = warp_reduce16(v, lane);
        const int idx = lane >> 1;
        if (!(lane & 1)) red_w[(idx >> 3) * LP + base + (idx & 7)] = tot;
      }
      if (P.F_toa_bin != nullptr) s_vals[tid] = active ? wFup * P.bins[b].inv_dlam : 0.0;
    }
  } else if (TOA || P.F_toa_bin != nullptr) {
    s_vals[tid] = 0.0;
  }
  __syncthreads();

  if (TOA || P.F_toa_bin != nullptr) {
    for (int k = tid; k < nbt; k += BLOCK) {
      const int bb = b_first + k;
      int g_lo = bb * P.ng - pt0, g_hi = g_lo + P.ng;
      // a bin may straddle two tiles: every tile adds its own part
      const bool whole = (g_lo >= 0) && (g_hi <= BLOCK);
      if (g_lo < 0) g_lo = 0;
      if (g_hi > BLOCK) g_hi = BLOCK;
      double sum = col_nan ? nan("") : 0.0;
      for (int q = g_lo; q < g_hi; ++q) sum += s_vals[q];
      double *dst = P.F_toa_bin + (size_t)col * P.nb + bb;
      if (whole) *dst = sum; else atomicAdd(dst, sum);
    }
  }
  if (TOA) return;

  column_epilogue<BLOCK>(P, L, s_red, s_fin, &s_is_last, nwa, want_beam, col, tile, col_nan);
}

// --------------------------------------------------------------------------------------------
// rt_solve2_kernel: the isothermal S3-S7 path with TWO adjacent spectral points per thread (same bin: needs an even
// number of Gauss points).  Same algorithm and arithmetic as rt_solve_kernel<false, TOA, false, ...>; what changes is
// the instruction mix: everything that depends only on (column, level, bin) -- the level record, corner weights, row
// addresses (one 16-byte load per corner instead of two 8-byte ones), Planck value, bin constants, hot constants,
// loop control -- is issued once for the two points, the two dependence chains interleave in one warp (ILP 2), and
// the staging / butterfly reductions handle the pair's sum.  A tile is 2 x BLOCK points.
// --------------------------------------------------------------------------------------------
struct Rows2 { double2 l00, l01, l10, l11; };

__device__ __forceinline__ Rows2 load_rows2(const double *__restrict__ lnk_pt, const LevelRec *lv) {
  const uint4 o = *reinterpret_cast<const uint4 *>(&lv->o00);
  Rows2 r;
  r.l00 = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.x)));
  r.l01 = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.y)));
  r.l10 = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.z)));
  r.l11 = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.w)));
  return r;
}

template <bool TOA, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) rt_solve2_kernel(const KParams P) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ double s_T32[32];
  __shared__ int s_is_last;
  constexpr int TP = 2 * BLOCK;   // points per tile
  const int N = P.N, nlev = P.nlev;
  const SolveSmem L = solve_smem(N, nlev, BLOCK, P.ng, P.nb, TOA, false, 2);
  const LevelRec *s_lev = (const LevelRec *)(smem + L.off_lev) + 1;
  double *s_B = (double *)(smem + L.off_B);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  double *s_red = (double *)(smem + L.off_red);
  double *s_stage = (double *)(smem + L.off_stage);
  double *s_fin = (double *)(smem + L.off_fin);
  double *s_vals = (double *)(smem + L.off_vals);

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, col = blockIdx.y;
  const int LP = L.LP, nbtS = L.nbt;
  const double mu = P.mu[col];
  const bool day = mu > 0.0;

  const int pt0 = tile * TP;
  const int b_first = pt0 / P.ng;
  int pt_last = pt0 + TP - 1;
  if (pt_last > P.npt - 1) pt_last = P.npt - 1;
  const int nbt = pt_last / P.ng - b_first + 1;
  const int nwa = ((pt_last - pt0) >> 6) + 1;     // warps that own at least one pair of points

  stage_column<BLOCK>(P, L, smem, s_T32, col, b_first, nbt, tid, true);
  const int col_nan = P.ws_nan[col];
  __syncthreads();

  // the pair (pt, pt + 1): pt is even and n_gauss is even, so both points lie in bin b
  int pt = pt0 + 2 * tid;
  const bool active = pt < P.npt;
  if (!active) pt = P.npt - 2;
  const int b = pt / P.ng, gidx = pt - b * P.ng;
  const int bl = b - b_first;
  const int warp = tid >> 5, lane = tid & 31;
  const bool warp_on = warp < nwa;
  double *red_w = s_red + (size_t)warp * 4 * LP;
  double *stage_w = s_stage + (size_t)warp * 8 * STAGE_LD;
  const bool want_beam = !TOA && (P.F_beam != nullptr);

  if (warp_on) {
    const double dlam = P.bins[b].dlam;
    const double W0 = active ? dlam * P.gauss_w[gidx] : 0.0, W1 = active ? dlam * P.gauss_w[gidx + 1] : 0.0;
    const double muF = day ? mu * P.fstar[b] : 0.0;
    const double inv_mu = day ? 1.0 / mu : 0.0;
    const double *lnk_pt = P.lnk + pt;
    const BinOpt *bin0 = s_bin + bl, *bin1 = s_bin + nbtS + bl;
    const double *T32 = s_T32;
    double *stage_wr = stage_w + lane;

    constexpr int STK = TOA ? 1 : ((MAXL + 1 + 7) & ~7);
    double2 st_cd0[STK], st_cd1[STK];   // (c, W d) of the two points
    double2 st_R[STK];                  // (R0, R1)

    double R0 = 0.0, R1 = 0.0, U0 = P.f_toa, U1 = P.f_toa;
    double Fb0 = muF, Fb1 = muF;
    double Ct0 = 1.0, Dt0 = 0.0, Ct1 = 1.0, Dt1 = 0.0;

    auto push_interface = [&](int i) {
      if (!TOA) {
        st_R[i] = make_double2(R0, R1);
        stage_wr[(i & 7) * STAGE_LD] = fma(W0, U0 + Fb0, W1 * (U1 + Fb1));
        if ((i & 7) == 0) flush_stage(stage_w, red_w + 2 * LP + i, lane);
        if (want_beam) {
          const double wb = warp_sum(fma(W0, Fb0, W1 * Fb1));
          if (lane == 0) red_w[3 * LP + i] = wb;
        }
      }
    };

    auto sweep1 = [&](auto day_tag) {
      constexpr bool DAY = decltype(day_tag)::value;
      double tau0 = 0.0, tau1 = 0.0;
      const LevelRec *lv = s_lev + (N - 1);
      const double *Bp = s_B + (size_t)(N - 1) * nbtS + bl;
      Rows2 nx = load_rows2(lnk_pt, lv);
#pragma unroll (TOA ? kIsoUnrollToa2 : 1)
      for (int j = N - 1; j >= 0; --j, --lv, Bp -= nbtS) {
        const Rows2 cur = nx;
        nx = load_rows2(lnk_pt, lv - 1);
        push_interface(j + 1);
        // S3 + Eqs. 17-18 for the pair: shared corner weights and bin constants
        const double2 ca = *reinterpret_cast<const double2 *>(&lv->c00);
        const double2 cb = *reinterpret_cast<const double2 *>(&lv->c10);
        const double lk0 = fma(cb.y, cur.l11.x, fma(cb.x, cur.l10.x, fma(ca.y, cur.l01.x, ca.x * cur.l00.x)));
        const double lk1 = fma(cb.y, cur.l11.y, fma(cb.x, cur.l10.y, fma(ca.y, cur.l01.y, ca.x * cur.l00.y)));
        const double ka0 = exp_hot<0, false>(lk0, T32, nullptr), ka1 = exp_hot<0, false>(lk1, T32, nullptr);
        const BinOpt *bo = lv->cloud ? bin1 : bin0;
        const double2 sbss = *reinterpret_cast<const double2 *>(&bo->sb);
        const G0Terms gt = bo->gt;
        const double dm = lv->dm, Bj = *Bp;
        const double kx0 = ka0 + sbss.x, kx1 = ka1 + sbss.x;
        const double w00 = sbss.y * rcp_fast(kx0), w01 = sbss.y * rcp_fast(kx1);
        const double dtau0 = kx0 * dm, dtau1 = kx1 * dm;
        double Fa0 = 0.0, Fa1 = 0.0;
        if (DAY) {
          tau0 += dtau0;
          tau1 += dtau1;
          Fa0 = muF * exp_hot<1, false>(min_pos(tau0 * inv_mu, 708.0), T32, nullptr);   // (B6)
          Fa1 = muF * exp_hot<1, false>(min_pos(tau1 * inv_mu, 708.0), T32, nullptr);
        }
        double c0, d0, c1, d1;
        layer_forward<DAY, false>(P, T32, w00, gt, dtau0, Bj, Bj, mu, Fa0, Fb0, R0, U0, c0, d0);
        layer_forward<DAY, false>(P, T32, w01, gt, dtau1, Bj, Bj, mu, Fa1, Fb1, R1, U1, c1, d1);
        Fb0 = Fa0;
        Fb1 = Fa1;
        if (TOA) {
          Dt0 = fma(Ct0, d0, Dt0); Ct0 *= c0;
          Dt1 = fma(Ct1, d1, Dt1); Ct1 *= c1;
        } else {
          st_cd0[j + 1] = make_double2(c0, W0 * d0);
          st_cd1[j + 1] = make_double2(c1, W1 * d1);
        }
      }
    };
    if (day) sweep1(std::true_type{}); else sweep1(std::false_type{});

    // BOA, Eq.(10)
    const double F_boa = s_B[(size_t)nlev * nbtS + bl];
    const double Fup00 = (U0 + F_boa + Fb0) * rcp_fast(1.0 - R0), Fup01 = (U1 + F_boa + Fb1) * rcp_fast(1.0 - R1);

    if (TOA) {
      const double2 gw = make_double2(P.gauss_w[gidx], P.gauss_w[gidx + 1]);
      s_vals[2 * tid] = active ? gw.x * fma(Ct0, Fup00, Dt0) : 0.0;
      s_vals[2 * tid + 1] = active ? gw.y * fma(Ct1, Fup01, Dt1) : 0.0;
    } else {
      push_interface(0);
      st_cd0[0] = make_double2(0.0, W0 * Fup00);
      st_cd1[0] = make_double2(0.0, W1 * Fup01);
      for (int i = N + 1; i < LP; ++i) {
        st_cd0[i] = make_double2(1.0, 0.0); st_cd1[i] = make_double2(1.0, 0.0); st_R[i] = make_double2(0.0, 0.0);
      }
      double wF0 = 0.0, wF1 = 0.0;
#pragma unroll 1
      for (int base = 0; base <= N; base += 8) {
        double v[16];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const double2 a0 = st_cd0[base + k], a1 = st_cd1[base + k], r = st_R[base + k];
          wF0 = fma(a0.x, wF0, a0.y);
          wF1 = fma(a1.x, wF1, a1.y);
          v[k] = wF0 + wF1;
          v[8 + k] = fma(r.x, wF0, r.y * wF1);
        }
        const double tot = warp_reduce16(v, lane);
        const int idx = lane >> 1;
        if (!(lane & 1)) red_w[(idx >> 3) * LP + base + (idx & 7)] = tot;
      }
      if (P.F_toa_bin != nullptr) {
        const double inv_dlam = P.bins[b].inv_dlam;
        s_vals[2 * tid] = active ? wF0 * inv_dlam : 0.0;
        s_vals[2 * tid + 1] = active ? wF1 * inv_dlam : 0.0;
      }
    }
  } else if (TOA || P.F_toa_bin != nullptr) {
    s_vals[2 * tid] = 0.0;
    s_vals[2 * tid + 1] = 0.0;
  }
  __syncthreads();

  if (TOA || P.F_toa_bin != nullptr) {
    for (int k = tid; k < nbt; k += BLOCK) {
      const int bb = b_first + k;
      int g_lo = bb * P.ng - pt0, g_hi = g_lo + P.ng;
      const bool whole = (g_lo >= 0) && (g_hi <= TP);
      if (g_lo < 0) g_lo = 0;
      if (g_hi > TP) g_hi = TP;
      double sum = col_nan ? nan("") : 0.0;
      for (int q = g_lo; q < g_hi; ++q) sum += s_vals[q];
      double *dst = P.F_toa_bin + (size_t)col * P.nb + bb;
      if (whole) *dst = sum; else atomicAdd(dst, sum);
    }
  }
  if (TOA) return;

  column_epilogue<BLOCK>(P, L, s_red, s_fin, &s_is_last, nwa, want_beam, col, tile, col_nan);
}

template <bool TOA, int PPT, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB) rt_solvem_kernel(const KParams P) {
  static_assert(PPT == 2 || PPT == 4, "points per thread");
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ double s_T32[32];
  __shared__ int s_is_last;
  constexpr int TP = PPT * BLOCK;   // points per tile
  constexpr int H = PPT / 2;        // 16-byte loads per corner row
  const int N = P.N, nlev = P.nlev;
  const SolveSmem L = solve_smem(N, nlev, BLOCK, P.ng, P.nb, TOA, false, PPT);
  const LevelRec *s_lev = (const LevelRec *)(smem + L.off_lev) + 1;
  double *s_B = (double *)(smem + L.off_B);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  double *s_red = (double *)(smem + L.off_red);
  double *s_stage = (double *)(smem + L.off_stage);
  double *s_fin = (double *)(smem + L.off_fin);
  double *s_vals = (double *)(smem + L.off_vals);

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, col = blockIdx.y;
  const int LP = L.LP, nbtS = L.nbt;
  const double mu = P.mu[col];
  const bool day = mu > 0.0;

  const int pt0 = tile * TP;
  const int b_first = pt0 / P.ng;
  int pt_last = pt0 + TP - 1;
  if (pt_last > P.npt - 1) pt_last = P.npt - 1;
  const int nbt = pt_last / P.ng - b_first + 1;
  const int nwa = ((pt_last - pt0) / (32 * PPT)) + 1;     // warps that own at least one group of points

  stage_column<BLOCK>(P, L, smem, s_T32, col, b_first, nbt, tid, true);
  const int col_nan = P.ws_nan[col];
  __syncthreads();

  // the group pt .. pt + PPT - 1: pt and n_gauss are multiples of PPT, so all its points lie in bin b
  int pt = pt0 + PPT * tid;
  const bool active = pt < P.npt;
  if (!active) pt = P.npt - PPT;
  const int b = pt / P.ng, gidx = pt - b * P.ng;
  const int bl = b - b_first;
  const int warp = tid >> 5, lane = tid & 31;
  const bool warp_on = warp < nwa;
  double *red_w = s_red + (size_t)warp * 4 * LP;
  double *stage_w = s_stage + (size_t)warp * 8 * STAGE_LD;
  const bool want_beam = !TOA && (P.F_beam != nullptr);

  if (warp_on) {
    const double dlam = P.bins[b].dlam;
    double W[PPT];
#pragma unroll
    for (int q = 0; q < PPT; ++q) W[q] = active ? dlam * P.gauss_w[gidx + q] : 0.0;
    const double muF = day ? mu * P.fstar[b] : 0.0;
    const double inv_mu = day ? 1.0 / mu : 0.0;
    const double *lnk_pt = P.lnk + pt;
    const BinOpt *bin0 = s_bin + bl, *bin1 = s_bin + nbtS + bl;
    const double *T32 = s_T32;
    double *stage_wr = stage_w + lane;

    constexpr int STK = TOA ? 1 : ((MAXL + 1 + 7) & ~7);
    double2 st_cd[STK][PPT];   // (c, W d) per point
    double st_R[STK][PPT];

    double R[PPT], U[PPT], Fb[PPT], Ct[PPT], Dt[PPT];
#pragma unroll
    for (int q = 0; q < PPT; ++q) { R[q] = 0.0; U[q] = P.f_toa; Fb[q] = muF; Ct[q] = 1.0; Dt[q] = 0.0; }

    auto push_interface = [&](int i) {
      if (!TOA) {
        double su = 0.0, sb = 0.0;
#pragma unroll
        for (int q = 0; q < PPT; ++q) { st_R[i][q] = R[q]; su = fma(W[q], U[q] + Fb[q], su); sb = fma(W[q], Fb[q], sb); }
        stage_wr[(i & 7) * STAGE_LD] = su;
        if ((i & 7) == 0) flush_stage(stage_w, red_w + 2 * LP + i, lane);
        if (want_beam) {
          const double wb = warp_sum(sb);
          if (lane == 0) red_w[3 * LP + i] = wb;
        }
      }
    };

    struct RowsM { double2 l00[H], l01[H], l10[H], l11[H]; };
    auto load_rows_m = [&](const LevelRec *lv) {
      const uint4 o = *reinterpret_cast<const uint4 *>(&lv->o00);
      RowsM r;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        r.l00[h] = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.x)) + h);
        r.l01[h] = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.y)) + h);
        r.l10[h] = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.z)) + h);
        r.l11[h] = __ldg(reinterpret_cast<const double2 *>(elem_addr(lnk_pt, o.w)) + h);
      }
      return r;
    };

    auto sweep1 = [&](auto day_tag) {
      constexpr bool DAY = decltype(day_tag)::value;
      double tau[PPT];
#pragma unroll
      for (int q = 0; q < PPT; ++q) tau[q] = 0.0;
      const LevelRec *lv = s_lev + (N - 1);
      const double *Bp = s_B + (size_t)(N - 1) * nbtS + bl;
      RowsM nx = load_rows_m(lv);
#pragma unroll 1
      for (int j = N - 1; j >= 0; --j, --lv, Bp -= nbtS) {
        const RowsM cur = nx;
        nx = load_rows_m(lv - 1);
        push_interface(j + 1);
        const double2 ca = *reinterpret_cast<const double2 *>(&lv->c00);
        const double2 cb = *reinterpret_cast<const double2 *>(&lv->c10);
        const BinOpt *bo = lv->cloud ? bin1 : bin0;
        const double2 sbss = *reinterpret_cast<const double2 *>(&bo->sb);
        const G0Terms gt = bo->gt;
        const double dm = lv->dm, Bj = *Bp;
#pragma unroll
        for (int q = 0; q < PPT; ++q) {
          const int h = q >> 1;
          const double r00 = (q & 1) ? cur.l00[h].y : cur.l00[h].x, r01 = (q & 1) ? cur.l01[h].y : cur.l01[h].x;
          const double r10 = (q & 1) ? cur.l10[h].y : cur.l10[h].x, r11 = (q & 1) ? cur.l11[h].y : cur.l11[h].x;
          const double lk = fma(cb.y, r11, fma(cb.x, r10, fma(ca.y, r01, ca.x * r00)));
          const double kx = exp_hot<0, false>(lk, T32, nullptr) + sbss.x;
          const double w0 = sbss.y * rcp_fast(kx);
          const double dtau = kx * dm;
          double Fa = 0.0;
          if (DAY) {
            tau[q] += dtau;
            Fa = muF * exp_hot<1, false>(min_pos(tau[q] * inv_mu, 708.0), T32, nullptr);   // (B6)
          }
          double c, d;
          layer_forward<DAY, false>(P, T32, w0, gt, dtau, Bj, Bj, mu, Fa, Fb[q], R[q], U[q], c, d);
          Fb[q] = Fa;
          if (TOA) {
            Dt[q] = fma(Ct[q], d, Dt[q]);
            Ct[q] *= c;
          } else {
            st_cd[j + 1][q] = make_double2(c, W[q] * d);
          }
        }
      }
    };
    if (day) sweep1(std::true_type{}); else sweep1(std::false_type{});

    // BOA, Eq.(10)
    const double F_boa = s_B[(size_t)nlev * nbtS + bl];
    double Fup0[PPT];
#pragma unroll
    for (int q = 0; q < PPT; ++q) Fup0[q] = (U[q] + F_boa + Fb[q]) * rcp_fast(1.0 - R[q]);

    if (TOA) {
#pragma unroll
      for (int q = 0; q < PPT; ++q) s_vals[PPT * tid + q] = active ? P.gauss_w[gidx + q] * fma(Ct[q], Fup0[q], Dt[q]) : 0.0;
    } else {
      push_interface(0);
#pragma unroll
      for (int q = 0; q < PPT; ++q) st_cd[0][q] = make_double2(0.0, W[q] * Fup0[q]);
      for (int i = N + 1; i < LP; ++i)
#pragma unroll
        for (int q = 0; q < PPT; ++q) { st_cd[i][q] = make_double2(1.0, 0.0); st_R[i][q] = 0.0; }
      double wF[PPT];
#pragma unroll
      for (int q = 0; q < PPT; ++q) wF[q] = 0.0;
#pragma unroll 1
      for (int base = 0; base <= N; base += 8) {
        double v[16];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          double su = 0.0, sd = 0.0;
#pragma unroll
          for (int q = 0; q < PPT; ++q) {
            const double2 a = st_cd[base + k][q];
            wF[q] = fma(a.x, wF[q], a.y);
            su += wF[q];
            sd = fma(st_R[base + k][q], wF[q], sd);
          }
          v[k] = su;
          v[8 + k] = sd;
        }
        const double tot = warp_reduce16(v, lane);
        const int idx = lane >> 1;
        if (!(lane & 1)) red_w[(idx >> 3) * LP + base + (idx & 7)] = tot;
      }
      if (P.F_toa_bin != nullptr) {
        const double inv_dlam = P.bins[b].inv_dlam;
#pragma unroll
        for (int q = 0; q < PPT; ++q) s_vals[PPT * tid + q] = active ? wF[q] * inv_dlam : 0.0;
      }
    }
  } else if (TOA || P.F_toa_bin != nullptr) {
#pragma unroll
    for (int q = 0; q < PPT; ++q) s_vals[PPT * tid + q] = 0.0;
  }
  __syncthreads();

  if (TOA || P.F_toa_bin != nullptr) {
    for (int k = tid; k < nbt; k += BLOCK) {
      const int bb = b_first + k;
      int g_lo = bb * P.ng - pt0, g_hi = g_lo + P.ng;
      const bool whole = (g_lo >= 0) && (g_hi <= TP);
      if (g_lo < 0) g_lo = 0;
      if (g_hi > TP) g_hi = TP;
      double sum = col_nan ? nan("") : 0.0;
      for (int q = g_lo; q < g_hi; ++q) sum += s_vals[q];
      double *dst = P.F_toa_bin + (size_t)col * P.nb + bb;
      if (whole) *dst = sum; else atomicAdd(dst, sum);
    }
  }
  if (TOA) return;

  column_epilogue<BLOCK>(P, L, s_red, s_fin, &s_is_last, nwa, want_beam, col, tile, col_nan);
}

// --------------------------------------------------------------------------------------------
// rt_iter_kernel: the scheme Thomas's algorithm replaces (L258-270, L397), as a measured
// comparison.  Same decomposition, staging and S3-S5 arithmetic as rt_solve_kernel; instead of the forward
// elimination the (t, r, S_up, S_dn) of every system layer go to thread-private arrays, and the flux arrays are
// swept n_iter times: upward pass Eq.(10) + Eq.(2) with the previous downward fluxes, downward pass Eq.(3) with the
// upward fluxes just computed; all diffuse fluxes start at 0 (reading R23).  The non-isothermal system keeps its
// centre levels as unknowns (2N system layers, L311-313).  S7 as in the Thomas path (column_epilogue).
// --------------------------------------------------------------------------------------------
template <bool NONISO, int BLOCK>
__global__ void __launch_bounds__(BLOCK) rt_iter_kernel(const KParams P, const int n_iter) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ double s_T32[32];
  __shared__ int s_is_last;
  constexpr int MAXS = NONISO ? 2 * MAXL : MAXL;   // system layers
  const int N = P.N, nlev = P.nlev;
  const SolveSmem L = solve_smem(N, nlev, BLOCK, P.ng, P.nb, false);
  const LevelRec *s_lev = (const LevelRec *)(smem + L.off_lev) + 1;
  double *s_B = (double *)(smem + L.off_B);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  double *s_red = (double *)(smem + L.off_red);
  double *s_fin = (double *)(smem + L.off_fin);

  const int tid = threadIdx.x;
  const int tile = blockIdx.x, col = blockIdx.y;
  const int LP = L.LP, nbtS = L.nbt;
  const double mu = P.mu[col];
  const bool day = mu > 0.0;
  const int pt0 = tile * BLOCK;
  const int b_first = pt0 / P.ng;
  int pt_last = pt0 + BLOCK - 1;
  if (pt_last > P.npt - 1) pt_last = P.npt - 1;
  const int nbt = pt_last / P.ng - b_first + 1;
  const int nwa = ((pt_last - pt0) >> 5) + 1;
  stage_column<BLOCK>(P, L, smem, s_T32, col, b_first, nbt, tid);
  const int col_nan = P.ws_nan[col];
  __syncthreads();

  int pt = pt0 + tid;
  const bool active = pt < P.npt;
  if (!active) pt = P.npt - 1;
  const int b = pt / P.ng, gidx = pt - b * P.ng;
  const int bl = b - b_first;
  const int warp = tid >> 5, lane = tid & 31;
  double *red_w = s_red + (size_t)warp * 4 * LP;

  if (warp < nwa) {
    const double W = active ? P.bins[b].dlam * P.gauss_w[gidx] : 0.0;
    const double muF = day ? mu * P.fstar[b] : 0.0;
    const double inv_mu = day ? 1.0 / mu : 0.0;
    const double *lnk_pt = P.lnk + pt;
    const BinOpt *bin0 = s_bin + bl, *bin1 = s_bin + nbtS + bl;
    const double *T32 = s_T32;
    const int LS = NONISO ? 2 * N : N;             // system layers; level s = lower end of system layer s

    double a_t[MAXS], a_r[MAXS], a_su[MAXS], a_sd[MAXS];
    double fu[MAXS + 1], fd[MAXS + 1], bm[MAXS + 1];

    // ---- S3-S5 per system layer, TOA -> BOA (tau and the beam are running prefixes) ----
    auto coeffs = [&](auto day_tag) {
      constexpr bool DAY = decltype(day_tag)::value;
      double tau = 0.0, Fb = muF;
      bm[LS] = Fb;
      if (!NONISO) {
        for (int j = N - 1; j >= 0; --j) {
          const LevelRec *lv = s_lev + j;
          double kx, w0, g0;
          level_optics(load_rows(lnk_pt, lv), T32, lv, bin0, bin1, kx, w0, g0);
          const double dtau = kx * lv->dm;
          const double Bj = s_B[(size_t)j * nbtS + bl];
          double Fa = 0.0;
          if (DAY) {
            tau += dtau;
            Fa = muF * exp_hot<1, false>(min_pos(tau * inv_mu, 708.0), T32, nullptr);
          }
          layer_coeffs<DAY, false>(P, T32, w0, g0, dtau, Bj, Bj, mu, Fa, Fb, a_t[j], a_r[j], a_su[j], a_sd[j]);
          bm[j] = Fa;
          Fb = Fa;
        }
      } else {
        double kx_up, w0_up, g0_up;
        {
          const LevelRec *lv = s_lev + LS;
          level_optics(load_rows(lnk_pt, lv), T32, lv, bin0, bin1, kx_up, w0_up, g0_up);
        }
        double B_up = s_B[(size_t)LS * nbtS + bl];
        for (int sl = LS - 1; sl >= 0; --sl) {
          const LevelRec *lv = s_lev + sl;
          double kx_lo, w0_lo, g0_lo;
          level_optics(load_rows(lnk_pt, lv), T32, lv, bin0, bin1, kx_lo, w0_lo, g0_lo);
          const double B_lo = s_B[(size_t)sl * nbtS + bl];
          const double dtau = 0.5 * (kx_lo + kx_up) * lv->dm;
          double Fa = 0.0;
          if (DAY) {
            tau += dtau;
            Fa = muF * exp_hot<1, false>(min_pos(tau * inv_mu, 708.0), T32, nullptr);
          }
          layer_coeffs<DAY, true>(P, T32, 0.5 * (w0_lo + w0_up), 0.5 * (g0_lo + g0_up), dtau, B_lo, B_up, mu, Fa, Fb,
                                  a_t[sl], a_r[sl], a_su[sl], a_sd[sl]);
          bm[sl] = Fa;
          Fb = Fa;
          kx_up = kx_lo; w0_up = w0_lo; g0_up = g0_lo; B_up = B_lo;
        }
      }
    };
    if (day) coeffs(std::true_type{}); else coeffs(std::false_type{});

    // ---- n_iter pair-wise sweeps over the whole atmosphere ----
    for (int l = 0; l <= LS; ++l) { fu[l] = 0.0; fd[l] = 0.0; }
    const double F_boa = s_B[(size_t)nlev * nbtS + bl];
    for (int it = 0; it < n_iter; ++it) {
      fu[0] = fd[0] + F_boa + bm[0];                                        // Eq.(10)
      for (int sl = 0; sl < LS; ++sl) fu[sl + 1] = fma(a_t[sl], fu[sl], fma(a_r[sl], fd[sl + 1], a_su[sl]));   // Eq.(2)
      fd[LS] = P.f_toa;
      for (int sl = LS - 1; sl >= 0; --sl) fd[sl] = fma(a_t[sl], fd[sl + 1], fma(a_r[sl], fu[sl], a_sd[sl]));  // Eq.(3)
    }

    // ---- S7: weighted sums over the warp at the interfaces ----
    const int stride = NONISO ? 2 : 1;
    for (int i = 0; i <= N; ++i) {
      const double su = warp_sum(W * fu[i * stride]);
      const double sd = warp_sum(W * fd[i * stride]);
      const double sb = warp_sum(W * bm[i * stride]);
      if (lane == 0) { red_w[i] = su; red_w[LP + i] = sd; red_w[2 * LP + i] = sb; red_w[3 * LP + i] = sb; }
    }
  }
  __syncthreads();
  column_epilogue<BLOCK>(P, L, s_red, s_fin, &s_is_last, nwa, P.F_beam != nullptr, col, tile, col_nan);
}

// --------------------------------------------------------------------------------------------
// small utility kernels
// --------------------------------------------------------------------------------------------
__global__ void zero_kernel(double *p, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    p[i] = 0.0;
}

__global__ void selftest_math_kernel(int n, const double *x, double *rcp, double *rsq, double *ex, double *omx) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  __shared__ double T32[32];
  if (threadIdx.x < 32) T32[threadIdx.x] = kExp2Tab[threadIdx.x];
  __syncthreads();
  if (i >= n) return;
  const double v = x[i];
  rcp[i] = rcp_fast(v);
  rsq[i] = rsqrt_fast(fabs(v));
  // e^-|x| through the three entry points the step kernel uses: e^-a, e^-2(a/2) (+ 1 - e^-a), e^(-a)
  const double a = fmin(fabs(v), 708.0);
  double om;
  const double e2 = exp_hot<2, true>(0.5 * a, T32, &om);
  const double e1 = exp_hot<1, false>(a, T32, nullptr);
  const double e0 = exp_hot<0, false>(-a, T32, nullptr);
  ex[i] = (i % 3 == 0) ? e0 : ((i % 3 == 1) ? e1 : e2);
  omx[i] = om;
}

__global__ void selftest_planck_kernel(int n, const double *T, const double *lo, const double *hi, double *out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double t = T[i];
  if (!(t > 0.0)) { out[i] = 0.0; return; }
  double l_hi, l_lo;
  const double g_hi = planck_G(kPlanckC2 / (hi[i] * t), &l_hi), g_lo = planck_G(kPlanckC2 / (lo[i] * t), &l_lo);
  const double t2 = t * t;
  out[i] = kPlanckC1 * t2 * t2 * planck_dG(g_lo, l_lo, g_hi, l_hi) / (hi[i] - lo[i]);
}

__global__ void dfma_peak_kernel(int iters, double seed, double *sink, long long *cycles) {
  double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6,
         a7 = seed + 7;
  const double m = 0.999999, k = 1e-9;
  const long long t0 = clock64();
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, k); a1 = fma(a1, m, k); a2 = fma(a2, m, k); a3 = fma(a3, m, k);
    a4 = fma(a4, m, k); a5 = fma(a5, m, k); a6 = fma(a6, m, k); a7 = fma(a7, m, k);
  }
  const long long t1 = clock64();
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) sink[0] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) cycles[0] = t1 - t0;
}

// --------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------
typedef void (*kernel_fn)(const KParams);

struct KernelChoice {
  kernel_fn fn;
  int block;
};

template <bool NONISO, bool TOA, bool BDIRECT>
KernelChoice pick_kernel(int block, int minb) {
#define HRT_VARIANT(B, M) if (block == B && (minb == M || minb == 0)) return {rt_solve_kernel<NONISO, TOA, BDIRECT, B, M>, B};
  HRT_VARIANT(32, 16) HRT_VARIANT(64, 8) HRT_VARIANT(96, 7) HRT_VARIANT(128, 4) HRT_VARIANT(128, 5) HRT_VARIANT(128, 6)
#undef HRT_VARIANT
  return {nullptr, 0};
}

template <bool BDIRECT>
KernelChoice pick_b(bool noniso, bool toa, int block, int minb) {
  if (noniso) return toa ? pick_kernel<true, true, BDIRECT>(block, minb) : pick_kernel<true, false, BDIRECT>(block, minb);
  return toa ? pick_kernel<false, true, BDIRECT>(block, minb) : pick_kernel<false, false, BDIRECT>(block, minb);
}

KernelChoice pick(bool noniso, bool toa, bool bdirect, int block, int minb) {
  return bdirect ? pick_b<true>(noniso, toa, block, minb) : pick_b<false>(noniso, toa, block, minb);
}

KernelChoice pick2(bool toa, int minb) {
#define HRT_VARIANT2(M) if (minb == M) return {toa ? rt_solve2_kernel<true, 64, M> : rt_solve2_kernel<false, 64, M>, 64};
  HRT_VARIANT2(5) HRT_VARIANT2(6) HRT_VARIANT2(7) HRT_VARIANT2(8)
#undef HRT_VARIANT2
  return {nullptr, 0};
}

// four points per thread: TOA mode only (no stack), 12 warp-sized blocks per SM at 164 registers
KernelChoice pick4() { return {rt_solvem_kernel<true, 4, 32, 9>, 32}; }

typedef void (*iter_fn)(const KParams, const int);
iter_fn pick_iter(bool noniso, int block) {
  switch (block) {
    case 32: return noniso ? rt_iter_kernel<true, 32> : rt_iter_kernel<false, 32>;
    case 64: return noniso ? rt_iter_kernel<true, 64> : rt_iter_kernel<false, 64>;
    case 96: return noniso ? rt_iter_kernel<true, 96> : rt_iter_kernel<false, 96>;
    case 128: return noniso ? rt_iter_kernel<true, 128> : rt_iter_kernel<false, 128>;
  }
  return nullptr;
}

const int kBlocks[] = {32, 64, 96, 128};

// block size of the one-point-per-thread kernels: columns with many spectral points use 128-thread tiles, except the
// non-isothermal solve kernel, which runs best as 16 warp-sized blocks per SM at 128 registers (config 3 / 4:
// 1.390 / 5.41 ms against 1.427 / 5.60 at 128 x 4 and 1.460 / 5.73 at 64 x 8); small columns take the block with the
// fewest padded lanes, ties -> larger block (fewer tiles)
int choose_block(int npt, bool noniso_solve = false) {
  const char *env = getenv("HELIOS_RT_BLOCK");
  if (env) {
    const int v = atoi(env);
    for (int b : kBlocks) if (b == v) return v;
  }
  if (npt >= 256) return noniso_solve ? 32 : 128;
  int best = 32;
  long best_waste = -1;
  for (int b : {32, 64, 96, 128}) {
    const long tiles = (npt + b - 1) / b;
    const long waste = tiles * (long)(((b + 31) / 32) * 32) - npt;
    if (best_waste < 0 || waste < best_waste || (waste == best_waste && b > best)) { best = b; best_waste = waste; }
  }
  return best;
}

// resident blocks per SM the kernel is compiled for (register cap), measured on B200: isothermal with the
// back-substitution stack 128 x 6 (80 registers, no spills: config 2 0.718 ms against 0.762 at 5 and 0.747 at 7),
// TOA mode 128 x 5 (96 registers), non-isothermal 128 x 4 (128 registers)
int choose_minb(int block, bool noniso, bool toa) {
  const char *mb = getenv("HELIOS_RT_MINB");
  if (mb) return atoi(mb);
  if (block == 128) return noniso ? 4 : (toa ? 5 : 6);
  return 0;
}

// spectral points per thread: isothermal columns whose number of Gauss points is a multiple of it, with enough points
// to fill the tiles.  2 (rt_solve2_kernel) with the back-substitution stack; 4 (rt_solvem_kernel) in TOA mode, where no
// stack competes for the load/store path (measured, config 2 / config 5 solve kernel: 1: 0.716 / 4.97 ms, 2: 0.67 / 4.73,
// 4: 0.80 / 4.52).  HELIOS_RT_PPT=1|2|4 overrides.
int choose_ppt(int npt, int ng, bool noniso, bool toa) {
  const bool can2 = !noniso && ng > 1 && (ng % 2) == 0, can4 = can2 && toa && (ng % 4) == 0;
  const char *env = getenv("HELIOS_RT_PPT");
  if (env) { const int v = atoi(env); return (v == 4 && can4) ? 4 : ((v >= 2 && can2) ? 2 : 1); }
  if (npt < 256) return 1;
  return can4 ? 4 : (can2 ? 2 : 1);
}

int choose_minb2() {
  const char *mb = getenv("HELIOS_RT_MINB");
  if (mb) { const int v = atoi(mb); if (v >= 5 && v <= 8) return v; }
  return 8;   // 126 registers, no spills: 8 x 64 threads x 2 points per SM
}

}  // namespace

struct helios_rt {
  helios_rt_config cfg;   // pointers nulled
  int npt, block, tiles, ppt;      // solve kernel: threads per block, tiles per column, points per thread
  int iter_block, iter_tiles;      // rt_iter_kernel keeps one point per thread
  bool noniso, toa;
  KernelChoice kc;
  SolveSmem lay;
  int nlev;
  // device tables
  double *d_lnk, *d_tab_lp, *d_tab_t, *d_edges, *d_gw;
  BinConst *d_bins;
  double *d_partial;
  unsigned *d_counter;
  LevelRec *d_ws_lev;
  double *d_ws_B, *d_ws_dm;
  int *d_ws_nan;
  // device staging for step_host
  double *d_p, *d_T, *d_mu, *d_fstar, *d_out;   // d_out: 5*(N+1)+N+nb per column, carved per output
  cudaStream_t own_stream;
  int regs, lmem, occ, sm_count;
  cudaError_t last_err;
  // per-kernel timing (helios_rt_set_profiling): a ring of event triples (before prep, between, after solve)
  int profiling;
  cudaEvent_t *prof_ev;      // [kProfRing][3]
  long long prof_head;       // triples recorded since the last read
};

constexpr int kProfRing = 256;

#define CK(h, call)                                                   \
  do {                                                                \
    cudaError_t e_ = (call);                                          \
    if (e_ != cudaSuccess) { if (h) (h)->last_err = e_; return HELIOS_RT_ECUDA; } \
  } while (0)

extern "C" const char *helios_rt_strerror(int code) {
  switch (code) {
    case HELIOS_RT_OK: return "success";
    case HELIOS_RT_EINVAL: return "invalid argument";
    case HELIOS_RT_ENOMEM: return "out of memory";
    case HELIOS_RT_ECUDA: return "CUDA runtime error (see helios_rt_last_cuda_error)";
    case HELIOS_RT_ENODEV: return "no usable CUDA device (compute capability 10.x required)";
    default: return "unknown error code";
  }
}

extern "C" const char *helios_rt_last_cuda_error(const helios_rt *h) {
  if (!h || h->last_err == cudaSuccess) return "";
  return cudaGetErrorString(h->last_err);
}

static int check_device() {
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || n == 0) { cudaGetLastError(); return HELIOS_RT_ENODEV; }
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return HELIOS_RT_ENODEV;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  return major == 10 ? HELIOS_RT_OK : HELIOS_RT_ENODEV;
}

static bool strictly_ascending(const double *a, int n) {
  for (int i = 0; i < n; ++i) if (!(a[i] == a[i])) return false;
  for (int i = 1; i < n; ++i) if (!(a[i] > a[i - 1])) return false;
  return true;
}

static int validate_config(const helios_rt_config *c) {
  if (!c) return HELIOS_RT_EINVAL;
  if (c->n_layers < 1 || c->n_layers > MAXL || c->n_bins < 1 || c->n_gauss < 1 || c->n_ktab_p < 2 ||
      c->n_ktab_t < 2 || c->max_columns < 1)
    return HELIOS_RT_EINVAL;
  if ((long long)c->n_bins * c->n_gauss > (1 << 24)) return HELIOS_RT_EINVAL;
  if ((long long)c->n_ktab_p * c->n_ktab_t * c->n_bins * c->n_gauss >= (1LL << 31)) return HELIOS_RT_EINVAL;   // 32-bit table offsets
  if (!c->ktab_p || !c->ktab_t || !c->ktab || !c->bin_edges || !c->gauss_w || !c->scat_gas || !c->cloud_ext ||
      !c->cloud_w0 || !c->cloud_g0)
    return HELIOS_RT_EINVAL;
  if (c->flags & ~(HELIOS_RT_IMPROVED | HELIOS_RT_NONISOTHERMAL | HELIOS_RT_TOA_SPECTRUM)) return HELIOS_RT_EINVAL;
  if (!strictly_ascending(c->ktab_p, c->n_ktab_p) || !(c->ktab_p[0] > 0)) return HELIOS_RT_EINVAL;
  if (!strictly_ascending(c->ktab_t, c->n_ktab_t)) return HELIOS_RT_EINVAL;
  if (!strictly_ascending(c->bin_edges, c->n_bins + 1) || !(c->bin_edges[0] > 0)) return HELIOS_RT_EINVAL;
  double sw = 0;
  for (int g = 0; g < c->n_gauss; ++g) { if (!(c->gauss_w[g] > 0)) return HELIOS_RT_EINVAL; sw += c->gauss_w[g]; }
  if (!(fabs(sw - 1.0) <= 1e-10)) return HELIOS_RT_EINVAL;
  for (int b = 0; b < c->n_bins; ++b) {
    if (!(c->scat_gas[b] >= 0) || !(c->cloud_ext[b] >= 0)) return HELIOS_RT_EINVAL;
    if (!(c->cloud_w0[b] >= 0 && c->cloud_w0[b] <= 1)) return HELIOS_RT_EINVAL;
    if (!(c->cloud_g0[b] >= 0 && c->cloud_g0[b] < 1)) return HELIOS_RT_EINVAL;
  }
  if (!(c->gravity > 0) || !(c->cp > 0) || !(c->eps2 > 0) || !(c->e_tau >= 0) || !(c->gcrit_tol >= 0) ||
      !(c->w0_transition >= 0) || !(c->f_toa >= 0))
    return HELIOS_RT_EINVAL;
  if (!(c->cloud_p_top == c->cloud_p_top) || !(c->cloud_p_bot == c->cloud_p_bot)) return HELIOS_RT_EINVAL;
  const size_t nk = (size_t)c->n_ktab_p * c->n_ktab_t * c->n_bins * c->n_gauss;
  for (size_t i = 0; i < nk; ++i) if (!(c->ktab[i] > 0) || !(c->ktab[i] < 1e300)) return HELIOS_RT_EINVAL;
  return HELIOS_RT_OK;
}

template <class T>
static cudaError_t upload(T **dst, const T *src, size_t n) {
  cudaError_t e = cudaMalloc((void **)dst, sizeof(T) * n);
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, src, sizeof(T) * n, cudaMemcpyHostToDevice);
}

extern "C" int helios_rt_destroy(helios_rt *h) {
  if (!h) return HELIOS_RT_OK;
  cudaFree(h->d_lnk); cudaFree(h->d_tab_lp); cudaFree(h->d_tab_t); cudaFree(h->d_edges); cudaFree(h->d_gw);
  cudaFree(h->d_bins); cudaFree(h->d_partial); cudaFree(h->d_counter);
  cudaFree(h->d_ws_lev); cudaFree(h->d_ws_B); cudaFree(h->d_ws_dm); cudaFree(h->d_ws_nan);
  cudaFree(h->d_p); cudaFree(h->d_T); cudaFree(h->d_mu); cudaFree(h->d_fstar); cudaFree(h->d_out);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  if (h->prof_ev) {
    for (int i = 0; i < 3 * kProfRing; ++i) if (h->prof_ev[i]) cudaEventDestroy(h->prof_ev[i]);
    free(h->prof_ev);
  }
  delete h;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_create(const helios_rt_config *cfg, helios_rt **out) {
  if (!out) return HELIOS_RT_EINVAL;
  *out = nullptr;
  int rc = validate_config(cfg);
  if (rc) return rc;
  rc = check_device();
  if (rc) return rc;
  helios_rt *h = new (std::nothrow) helios_rt();
  if (!h) return HELIOS_RT_ENOMEM;
  memset(h, 0, sizeof(*h));
  h->cfg = *cfg;
  h->cfg.ktab_p = h->cfg.ktab_t = h->cfg.ktab = h->cfg.bin_edges = h->cfg.gauss_w = nullptr;
  h->cfg.scat_gas = h->cfg.cloud_ext = h->cfg.cloud_w0 = h->cfg.cloud_g0 = nullptr;
  const int N = cfg->n_layers, nb = cfg->n_bins, ng = cfg->n_gauss;
  h->npt = nb * ng;
  h->noniso = (cfg->flags & HELIOS_RT_NONISOTHERMAL) != 0;
  h->toa = (cfg->flags & HELIOS_RT_TOA_SPECTRUM) != 0;
  h->iter_block = choose_block(h->npt);
  h->iter_tiles = (h->npt + h->iter_block - 1) / h->iter_block;
  h->nlev = h->noniso ? 2 * N + 1 : N;
  h->ppt = choose_ppt(h->npt, ng, h->noniso, h->toa);
  if (h->ppt == 4) {
    h->block = 32;
    h->kc = pick4();
  } else if (h->ppt == 2) {
    h->block = 64;
    h->kc = pick2(h->toa, choose_minb2());
  } else {
    h->block = choose_block(h->npt, h->noniso);
    h->kc = pick(h->noniso, h->toa, ng == 1, h->block, choose_minb(h->block, h->noniso, h->toa));
  }
  h->tiles = (h->npt + h->block * h->ppt - 1) / (h->block * h->ppt);
  h->lay = solve_smem(N, h->nlev, h->block, ng, nb, h->toa, ng == 1, h->ppt);
  cudaGetDevice(&rc);
  cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, rc);

  // ln(kappa) table, log10 pressure grid, per-bin constants
  const size_t nk = (size_t)cfg->n_ktab_p * cfg->n_ktab_t * h->npt;
  double *lnk = (double *)malloc(sizeof(double) * nk);
  double *lp = (double *)malloc(sizeof(double) * cfg->n_ktab_p);
  BinConst *bins = (BinConst *)malloc(sizeof(BinConst) * nb);
  if (!lnk || !lp || !bins) { free(lnk); free(lp); free(bins); helios_rt_destroy(h); return HELIOS_RT_ENOMEM; }
  for (size_t i = 0; i < nk; ++i) lnk[i] = log(cfg->ktab[i]);
  for (int i = 0; i < cfg->n_ktab_p; ++i) lp[i] = log10(cfg->ktab_p[i]);
  for (int b = 0; b < nb; ++b) {
    BinConst &bc = bins[b];
    bc.dlam = cfg->bin_edges[b + 1] - cfg->bin_edges[b];
    bc.inv_dlam = 1.0 / bc.dlam;
    const double sg = cfg->scat_gas[b], kc = cfg->cloud_ext[b], sc = cfg->cloud_w0[b] * kc;
    bc.sb[0] = sg;            bc.sb[1] = sg + kc;
    bc.ss[0] = sg;            bc.ss[1] = sg + sc;
    bc.gg[0] = 0.0;           bc.gg[1] = (sg + sc > 0.0) ? sc * cfg->cloud_g0[b] / (sg + sc) : 0.0;
  }
  cudaError_t e = cudaSuccess;
  auto step = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  step(upload(&h->d_lnk, lnk, nk));
  step(upload(&h->d_tab_lp, lp, (size_t)cfg->n_ktab_p));
  step(upload(&h->d_tab_t, cfg->ktab_t, (size_t)cfg->n_ktab_t));
  step(upload(&h->d_edges, cfg->bin_edges, (size_t)nb + 1));
  step(upload(&h->d_gw, cfg->gauss_w, (size_t)ng));
  step(upload(&h->d_bins, bins, (size_t)nb));
  free(lnk); free(lp); free(bins);
  const size_t ncol = (size_t)cfg->max_columns;
  step(cudaMalloc((void **)&h->d_partial, sizeof(double) * ncol * (h->tiles > h->iter_tiles ? h->tiles : h->iter_tiles) * 4 * (N + 1)));
  step(cudaMalloc((void **)&h->d_ws_lev, sizeof(LevelRec) * ncol * (h->nlev + 1)));
  step(cudaMalloc((void **)&h->d_ws_B, sizeof(double) * ncol * (h->nlev + 1) * nb));
  step(cudaMalloc((void **)&h->d_ws_dm, sizeof(double) * ncol * N));
  step(cudaMalloc((void **)&h->d_ws_nan, sizeof(int) * ncol));
  step(cudaMalloc((void **)&h->d_counter, sizeof(unsigned) * ncol));
  if (e == cudaSuccess) step(cudaMemset(h->d_counter, 0, sizeof(unsigned) * ncol));
  step(cudaMalloc((void **)&h->d_p, sizeof(double) * ncol * N));
  step(cudaMalloc((void **)&h->d_T, sizeof(double) * ncol * N));
  step(cudaMalloc((void **)&h->d_mu, sizeof(double) * ncol));
  step(cudaMalloc((void **)&h->d_fstar, sizeof(double) * nb));
  step(cudaMalloc((void **)&h->d_out, sizeof(double) * ncol * (4 * (N + 1) + N + nb)));
  step(cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking));
  if (e == cudaSuccess && h->kc.fn) {
    step(cudaFuncSetAttribute(h->kc.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->lay.total));
    step(cudaFuncSetAttribute(h->noniso ? rt_prep_kernel<true> : rt_prep_kernel<false>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prep_smem_bytes(N, h->nlev)));
    if (!h->toa && pick_iter(h->noniso, h->iter_block))
      step(cudaFuncSetAttribute(pick_iter(h->noniso, h->iter_block), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)solve_smem(N, h->nlev, h->iter_block, ng, nb, false).total));
    cudaFuncAttributes fa;
    step(cudaFuncGetAttributes(&fa, h->kc.fn));
    if (e == cudaSuccess) { h->regs = fa.numRegs; h->lmem = (int)fa.localSizeBytes; }
    step(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ, h->kc.fn, h->block, h->lay.total));
  }
  if (e != cudaSuccess || !h->kc.fn) {
    const bool oom = (e == cudaErrorMemoryAllocation);
    helios_rt_destroy(h);
    cudaGetLastError();
    return !oom && e == cudaSuccess ? HELIOS_RT_EINVAL : (oom ? HELIOS_RT_ENOMEM : HELIOS_RT_ECUDA);
  }
  *out = h;
  return HELIOS_RT_OK;
}

static int validate_step(const helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out) {
  if (!h || !in || !out) return HELIOS_RT_EINVAL;
  if (in->n_columns < 0 || in->n_columns > h->cfg.max_columns) return HELIOS_RT_EINVAL;
  if (in->n_columns == 0) return in->f_internal >= 0 ? HELIOS_RT_OK : HELIOS_RT_EINVAL;   // nothing to do
  if (in->n_columns > 0 && (!in->p || !in->T || !in->mu_star || !in->stellar_flux)) return HELIOS_RT_EINVAL;
  if (!(in->f_internal >= 0)) return HELIOS_RT_EINVAL;
  const bool any_flux = out->F_up || out->F_down || out->F_net || out->dTdt || out->F_beam;
  if (h->toa) { if (!out->F_up_toa_bin || any_flux) return HELIOS_RT_EINVAL; }
  else if (!any_flux && !out->F_up_toa_bin) return HELIOS_RT_EINVAL;
  return HELIOS_RT_OK;
}

static int launch_step(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out, cudaStream_t st,
                       int n_iter = 0) {
  const helios_rt_config &c = h->cfg;
  if (in->n_columns == 0) return HELIOS_RT_OK;
  KParams P;
  P.lnk = h->d_lnk; P.tab_lp = h->d_tab_lp; P.tab_t = h->d_tab_t; P.edges = h->d_edges; P.gauss_w = h->d_gw;
  P.bins = h->d_bins;
  P.nP = c.n_ktab_p; P.nT = c.n_ktab_t; P.N = c.n_layers; P.nlev = h->nlev; P.nb = c.n_bins; P.ng = c.n_gauss; P.npt = h->npt;
  P.tiles = n_iter > 0 ? h->iter_tiles : h->tiles;
  P.cloud_p_top = c.cloud_p_top; P.cloud_p_bot = c.cloud_p_bot; P.inv_g = 1.0 / c.gravity; P.inv_cp = 1.0 / c.cp;
  P.inv_eps2 = 1.0 / c.eps2; P.e_tau = c.e_tau; P.gcrit_tol = c.gcrit_tol; P.w0_transition = c.w0_transition;
  P.f_toa = c.f_toa; P.improved = (c.flags & HELIOS_RT_IMPROVED) ? 1 : 0;
  P.p = in->p; P.T = in->T; P.mu = in->mu_star; P.fstar = in->stellar_flux;
  P.T_int = in->f_internal > 0 ? sqrt(sqrt(in->f_internal / kSigmaSB)) : 0.0;
  P.F_up = out->F_up; P.F_down = out->F_down; P.F_net = out->F_net; P.dTdt = out->dTdt; P.F_beam = out->F_beam;
  P.F_toa_bin = out->F_up_toa_bin;
  P.partial = h->d_partial; P.counter = h->d_counter;
  P.ws_lev = h->d_ws_lev; P.ws_B = h->d_ws_B; P.ws_dm = h->d_ws_dm; P.ws_nan = h->d_ws_nan;
  // bins that straddle two tiles are accumulated with atomics: start from zero
  if (P.F_toa_bin && h->tiles > 1 && ((h->block * h->ppt) % c.n_gauss) != 0) {
    const size_t n = (size_t)in->n_columns * c.n_bins;
    zero_kernel<<<(unsigned)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024), 256, 0, st>>>(P.F_toa_bin, n);
  }
  cudaEvent_t *ev = h->profiling ? h->prof_ev + 3 * (h->prof_head % kProfRing) : nullptr;
  if (ev) CK(h, cudaEventRecord(ev[0], st));
  dim3 pgrid((unsigned)((c.n_bins + PREP_BINS - 1) / PREP_BINS), (unsigned)in->n_columns);
  const size_t psm = prep_smem_bytes(c.n_layers, h->nlev);
  if (h->noniso) rt_prep_kernel<true><<<pgrid, PREP_BLOCK, psm, st>>>(P);
  else rt_prep_kernel<false><<<pgrid, PREP_BLOCK, psm, st>>>(P);
  CK(h, cudaGetLastError());
  if (ev) CK(h, cudaEventRecord(ev[1], st));
  dim3 grid((unsigned)P.tiles, (unsigned)in->n_columns);
  if (n_iter > 0) {
    iter_fn fn = pick_iter(h->noniso, h->iter_block);
    if (!fn) return HELIOS_RT_EINVAL;
    const SolveSmem lay = solve_smem(c.n_layers, h->nlev, h->iter_block, c.n_gauss, c.n_bins, false);
    fn<<<grid, h->iter_block, lay.total, st>>>(P, n_iter);
  } else {
    h->kc.fn<<<grid, h->block, h->lay.total, st>>>(P);
  }
  CK(h, cudaGetLastError());
  if (ev) { CK(h, cudaEventRecord(ev[2], st)); ++h->prof_head; }
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_step(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out,
                              void *cuda_stream) {
  const int rc = validate_step(h, in, out);
  if (rc) return rc;
  return launch_step(h, in, out, (cudaStream_t)cuda_stream);
}

extern "C" int helios_rt_step_iterative(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out,
                                        int32_t n_iterations, void *cuda_stream) {
  const int rc = validate_step(h, in, out);
  if (rc) return rc;
  if (n_iterations < 1 || h->toa || out->F_up_toa_bin) return HELIOS_RT_EINVAL;
  return launch_step(h, in, out, (cudaStream_t)cuda_stream, n_iterations);
}

extern "C" int helios_rt_step_host(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out) {
  int rc = validate_step(h, in, out);
  if (rc) return rc;
  if (in->n_columns == 0) return HELIOS_RT_OK;
  const size_t ncol = (size_t)in->n_columns, N = (size_t)h->cfg.n_layers, nb = (size_t)h->cfg.n_bins;
  cudaStream_t st = h->own_stream;
  CK(h, cudaMemcpyAsync(h->d_p, in->p, sizeof(double) * ncol * N, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(h->d_T, in->T, sizeof(double) * ncol * N, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(h->d_mu, in->mu_star, sizeof(double) * ncol, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(h->d_fstar, in->stellar_flux, sizeof(double) * nb, cudaMemcpyHostToDevice, st));
  helios_rt_inputs din = *in;
  din.p = h->d_p; din.T = h->d_T; din.mu_star = h->d_mu; din.stellar_flux = h->d_fstar;
  helios_rt_outputs dout;
  double *o = h->d_out;
  const size_t ni = ncol * (N + 1);
  dout.F_up = out->F_up ? o : nullptr;                 o += ni;
  dout.F_down = out->F_down ? o : nullptr;             o += ni;
  dout.F_net = out->F_net ? o : nullptr;               o += ni;
  dout.F_beam = out->F_beam ? o : nullptr;             o += ni;
  dout.dTdt = out->dTdt ? o : nullptr;                 o += ncol * N;
  dout.F_up_toa_bin = out->F_up_toa_bin ? o : nullptr;
  rc = launch_step(h, &din, &dout, st);
  if (rc) return rc;
  if (out->F_up) CK(h, cudaMemcpyAsync(out->F_up, dout.F_up, sizeof(double) * ni, cudaMemcpyDeviceToHost, st));
  if (out->F_down) CK(h, cudaMemcpyAsync(out->F_down, dout.F_down, sizeof(double) * ni, cudaMemcpyDeviceToHost, st));
  if (out->F_net) CK(h, cudaMemcpyAsync(out->F_net, dout.F_net, sizeof(double) * ni, cudaMemcpyDeviceToHost, st));
  if (out->F_beam) CK(h, cudaMemcpyAsync(out->F_beam, dout.F_beam, sizeof(double) * ni, cudaMemcpyDeviceToHost, st));
  if (out->dTdt) CK(h, cudaMemcpyAsync(out->dTdt, dout.dTdt, sizeof(double) * ncol * N, cudaMemcpyDeviceToHost, st));
  if (out->F_up_toa_bin)
    CK(h, cudaMemcpyAsync(out->F_up_toa_bin, dout.F_up_toa_bin, sizeof(double) * ncol * nb, cudaMemcpyDeviceToHost, st));
  CK(h, cudaStreamSynchronize(st));
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_set_profiling(helios_rt *h, int32_t on) {
  if (!h) return HELIOS_RT_EINVAL;
  if (on && !h->prof_ev) {
    h->prof_ev = (cudaEvent_t *)calloc(3 * kProfRing, sizeof(cudaEvent_t));
    if (!h->prof_ev) return HELIOS_RT_ENOMEM;
    for (int i = 0; i < 3 * kProfRing; ++i) CK(h, cudaEventCreate(&h->prof_ev[i]));
  }
  h->profiling = on ? 1 : 0;
  h->prof_head = 0;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_kernel_times(helios_rt *h, int32_t *n_steps, double *prep_ms, double *solve_ms) {
  if (!h || !n_steps || !prep_ms || !solve_ms) return HELIOS_RT_EINVAL;
  *n_steps = 0; *prep_ms = 0.0; *solve_ms = 0.0;
  if (!h->prof_ev) return HELIOS_RT_OK;
  const long long n = h->prof_head < kProfRing ? h->prof_head : kProfRing;
  for (long long k = h->prof_head - n; k < h->prof_head; ++k) {
    cudaEvent_t *ev = h->prof_ev + 3 * (k % kProfRing);
    CK(h, cudaEventSynchronize(ev[2]));
    float a = 0.f, b = 0.f;
    CK(h, cudaEventElapsedTime(&a, ev[0], ev[1]));
    CK(h, cudaEventElapsedTime(&b, ev[1], ev[2]));
    *prep_ms += a; *solve_ms += b;
  }
  *n_steps = (int32_t)n;
  h->prof_head = 0;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_launch_info(const helios_rt *h, int32_t info[8]) {
  if (!h || !info) return HELIOS_RT_EINVAL;
  info[0] = h->block; info[1] = h->tiles; info[2] = (int32_t)h->lay.total; info[3] = h->regs; info[4] = h->occ;
  info[5] = h->lmem;
  info[6] = 2;   // rt_prep_kernel + rt_solve_kernel (+1 zero-fill launch when F_up_toa_bin bins straddle tiles)
  info[7] = h->sm_count;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_selftest_math(int32_t n, const double *x, double *rcp, double *rsq, double *ex, double *omx) {
  if (n < 0 || (n > 0 && (!x || !rcp || !rsq || !ex || !omx))) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  if (n == 0) return HELIOS_RT_OK;
  double *d = nullptr;
  if (cudaMalloc((void **)&d, sizeof(double) * 5 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return HELIOS_RT_ENOMEM; }
  cudaError_t e = cudaMemcpy(d, x, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    selftest_math_kernel<<<(n + 127) / 128, 128>>>(n, d, d + n, d + 2 * (size_t)n, d + 3 * (size_t)n, d + 4 * (size_t)n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(rcp, d + n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(rsq, d + 2 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(ex, d + 3 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(omx, d + 4 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  return e == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}

extern "C" int helios_rt_selftest_planck(int32_t n, const double *T, const double *lam_lo, const double *lam_hi,
                                         double *out) {
  if (n < 0 || (n > 0 && (!T || !lam_lo || !lam_hi || !out))) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  if (n == 0) return HELIOS_RT_OK;
  double *d = nullptr;
  if (cudaMalloc((void **)&d, sizeof(double) * 4 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return HELIOS_RT_ENOMEM; }
  cudaError_t e = cudaMemcpy(d, T, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d + n, lam_lo, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d + 2 * (size_t)n, lam_hi, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    selftest_planck_kernel<<<(n + 127) / 128, 128>>>(n, d, d + n, d + 2 * (size_t)n, d + 3 * (size_t)n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(out, d + 3 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  return e == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}

extern "C" int helios_rt_measure_dfma_peak(int32_t iters, double *dfma_per_s, double *sm_clock_mhz) {
  if (iters < 1 || !dfma_per_s) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double *sink = nullptr;
  long long *cyc = nullptr;
  if (cudaMalloc((void **)&sink, sizeof(double)) != cudaSuccess) return HELIOS_RT_ENOMEM;
  if (cudaMalloc((void **)&cyc, sizeof(long long)) != cudaSuccess) { cudaFree(sink); return HELIOS_RT_ENOMEM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = sms * 2, threads = 1024;
  dfma_peak_kernel<<<blocks, threads>>>(iters / 8 + 1, 1.0, sink, cyc);   // warm-up
  float best = 1e30f;
  long long hc = 0;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0);
    dfma_peak_kernel<<<blocks, threads>>>(iters, 1.0, sink, cyc);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { rc = HELIOS_RT_ECUDA; break; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) { best = ms; cudaMemcpy(&hc, cyc, sizeof(hc), cudaMemcpyDeviceToHost); }
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink); cudaFree(cyc);
  if (rc) return rc;
  *dfma_per_s = 8.0 * (double)iters * (double)blocks * threads / (best * 1e-3);
  if (sm_clock_mhz) *sm_clock_mhz = (double)hc / (best * 1e-3) * 1e-6;
  return HELIOS_RT_OK;
}
