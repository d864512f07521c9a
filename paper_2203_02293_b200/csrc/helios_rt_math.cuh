// helios_rt_math.cuh -- fp64 device primitives and the band-Planck integral of the helios_rt kernels (sm_100a).
//
// Shared by helios_rt.cu (the product kernels) and helios_rt_selftest.cu (the test-only library that exposes them
// to tests/ and bench.py).  Citations are PAPER.md lines (arXiv 2203.02293); R-numbers are DESIGN.md readings.
#pragma once

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace hrt {

constexpr double kPi = 3.14159265358979323846;
constexpr double kH = 6.62607015e-34, kC = 299792458.0, kKB = 1.380649e-23;  // CODATA 2019 (exact)
constexpr double kSigmaSB =
    2.0 * kPi * kPi * kPi * kPi * kPi * kKB * kKB * kKB * kKB / (15.0 * kH * kH * kH * kC * kC);
constexpr double kPlanckC1 = 2.0 * kKB * kKB * kKB * kKB / (kH * kH * kH * kC * kC);  // 2 k^4 / (h^3 c^2)
constexpr double kPlanckC2 = kH * kC / kKB;                                            // h c / k

// --------------------------------------------------------------------------------------------
// fp64 primitives.  Reciprocals, reciprocal square roots and exponentials are MUFU seeds refined in FMA: the fp64
// pipe is the binding resource of the step.
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
// fp64 pipe for arithmetic
__device__ __forceinline__ bool gt_pos(double a, double b) { return __double_as_longlong(a) > __double_as_longlong(b); }
__device__ __forceinline__ bool abs_lt(double a, double b_pos) {
  return (__double_as_longlong(a) & 0x7fffffffffffffffLL) < __double_as_longlong(b_pos);
}
// min(x, c) for x >= 0, c > 0 on the integer pipes
__device__ __forceinline__ double min_pos(double x, double c) { return gt_pos(x, c) ? c : x; }
// Cap of an exponential's argument, x >= 0, in ONE integer instruction: only the high word is limited to HI (the high
// word of the cap c, whose low word is 0), so the result is x for x < c and lies in [c, c (1 + 2^-20)) beyond.  Used
// where anything >= c gives e^-x = 0 to the last bit that matters (c = 354 for e^-2x, 708 for e^-x: >= 2^-1022).
template <int HI>
__device__ __forceinline__ double cap_pos(double x) {
  return __hiloint2double(min(__double2hiint(x), HI), __double2loint(x));
}

// exp by table: e^x = 2^m T[j] (1 + p(r)), k = 32 m + j = round(32 x / ln 2), r = x - k ln2/32, |r| <= ln2/64,
// T[j] = 2^(j/32) (32 doubles in shared memory), p = expm1(r) by its degree-6 Taylor polynomial (remainder
// r^7/5040 < 4e-18).  10 fp64 instructions.  The single-constant reduction k * fl(ln2/32) is exact to
// |k| 2.4e-18, i.e. <= 8e-14 relative at |x| = 700 and <= 3e-15 for |x| <= 30 (far inside the 1e-9 budget).
static __constant__ double kExp2Tab[32] = {
    1.0, 1.0218971486541166, 1.0442737824274138, 1.0671404006768237,
    1.0905077326652577, 1.1143867425958924, 1.1387886347566916, 1.1637248587775775,
    1.189207115002721, 1.215247359980469, 1.241857812073484, 1.2690509571917332,
    1.2968395546510096, 1.3252366431597413, 1.3542555469368927, 1.383909881963832,
    1.4142135623730951, 1.4451808069770467, 1.4768261459394993, 1.5091644275934228,
    1.5422108254079407, 1.5759808451078865, 1.6104903319492543, 1.645755478153965,
    1.681792830507429, 1.718619298122478, 1.7562521603732995, 1.7947090750031072,
    1.8340080864093424, 1.8741676341103, 1.9152065613971474, 1.9571441241754002};

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
static __constant__ HotConst kHC = {
    46.16624130844683,     -46.16624130844683,   -92.33248261689366,
    -0.02166084939249829,  0.010830424696249145,
    1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0,
    4.0 / 45.0, -4.0 / 15.0, 2.0 / 3.0, -4.0 / 3.0,
    1.225, -0.1582, -0.07465,
    -0.1777, 0.2351, -0.05582,
    3.14159265358979323846, -3.14159265358979323846};

//   MODE 0: e^x for |x| <= 708;  MODE 1: e^-a, 0 <= a <= 708;  MODE 2: e^-2a, 0 <= a <= 354, and, if OM,
//   *om = 1 - e^-2a without cancellation.  T32: the 2^(j/32) table (kExp2Tab) staged in shared memory.
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
  int hi;                                              // high word of 2^m T[j]: + ((ki >> 5) << 20), one LOP3 + one IMAD
  asm("mad.lo.s32 %0, %1, 32768, %2;" : "=r"(hi) : "r"(ki & ~31), "r"(__double2hiint(Tj)));
  const double Ts = __hiloint2double(hi, __double2loint(Tj));
  if (OM) *om = fma(-Ts, p, 1.0 - Ts);
  return fma(Ts, p, Ts);
}

// --------------------------------------------------------------------------------------------
// S2: band Planck (reading R8).  B_b(T) = [2 k^4 T^4 / (h^3 c^2)] [G(x_hi) - G(x_lo)] / (lam_hi - lam_lo),
// x = h c / (lam k T), G(x) = int_x^inf t^3/(e^t - 1) dt.  Evaluation (any method accurate to <= 1e-13 is allowed,
// SURVEY.md O5; this one is good to a few 1e-16):
//   x <  1.5       : G = pi^4/15 - low,  low = int_0^x = sum_k B_k x^{k+3} / ((k+3) k!)  (Bernoulli series; a bin
//                    with both edges here is differenced on `low`: no cancellation against pi^4/15)
//   1.5 <= x < 22  : G = e^{-x} P(x), P(x) = sum_{n>=1} e^{-(n-1)x} (x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4), which is
//                    analytic with its nearest singularities at +-2 pi i: degree-9 polynomial pieces on 41 intervals
//                    of width 1/2 (Chebyshev interpolation of the long-double series, built at create time by
//                    build_planck_table) reproduce it to 2e-16 (checked against 40-digit arithmetic)
//   x >= 22        : the n = 1, 2 terms of the series (the n = 3 term is < e^{-44} relative)
// --------------------------------------------------------------------------------------------
constexpr double kGX0 = 1.5, kGX1 = 22.0, kGH = 0.5;
constexpr int kGIntervals = 41, kGCoef = 10;   // (22 - 1.5) / 0.5 intervals, degree 9

// host: coefficients of P about each interval's midpoint, [kGIntervals][kGCoef], ascending powers of t = x - mid
inline void build_planck_table(double *tab) {
  const long double PI_L = 3.14159265358979323846264338327950288L;
  const int m = kGCoef;
  for (int iv = 0; iv < kGIntervals; ++iv) {
    const long double mid = (long double)kGX0 + (long double)kGH * (iv + 0.5L), hh = (long double)kGH * 0.5L;
    long double y[kGCoef], c[kGCoef];
    for (int k = 0; k < m; ++k) {
      const long double u = cosl(PI_L * (2 * k + 1) / (2 * m));
      const long double x = mid + hh * u;
      long double s = 0;
      for (int n = 1; n < 200; ++n) {
        const long double in = 1.0L / n;
        const long double term = expl(-(n - 1) * x) * in * (x * x * x + in * (3 * x * x + in * (6 * x + in * 6)));
        s += term;
        if (term < 1e-22L * s) break;
      }
      y[k] = s;
    }
    for (int j = 0; j < m; ++j) {          // Chebyshev coefficients
      long double a = 0;
      for (int k = 0; k < m; ++k) a += y[k] * cosl(j * PI_L * (2 * k + 1) / (2 * m));
      c[j] = a * 2 / m;
    }
    c[0] *= 0.5L;
    // Chebyshev -> monomial in u via T_{j} = 2 u T_{j-1} - T_{j-2}
    long double Tm2[kGCoef] = {0}, Tm1[kGCoef] = {0}, mono[kGCoef] = {0};
    Tm2[0] = 1; Tm1[1] = 1;
    mono[0] += c[0];
    if (m > 1) mono[1] += c[1];
    for (int j = 2; j < m; ++j) {
      long double Tj[kGCoef];
      for (int i = 0; i < m; ++i) Tj[i] = (i > 0 ? 2 * Tm1[i - 1] : 0) - Tm2[i];
      for (int i = 0; i < m; ++i) { mono[i] += c[j] * Tj[i]; Tm2[i] = Tm1[i]; Tm1[i] = Tj[i]; }
    }
    long double sc = 1;
    for (int i = 0; i < m; ++i) { tab[iv * m + i] = (double)(mono[i] / sc); sc *= hh; }
  }
}

// *low receives int_0^x t^3/(e^t-1) dt when x < 1.5 (else -1).  T32: the 2^(j/32) table in shared memory (exp_hot).
// Branch-free per lane: the forms are evaluated on clamped arguments and selected (the polynomial piece uses Estrin's
// scheme: dependence depth 4 instead of 9).  VOTE: a form that no active lane of the warp needs is skipped (warp-uniform
// branches; phase A's lanes are consecutive levels of a column at one bin edge, so their x lie within a factor ~2.5 and
// usually share one form).  x <= 0 (T = inf) is not special-cased: callers pass T > 0.
template <bool VOTE = false>
__device__ __forceinline__ double planck_G(double x, const double *__restrict__ gtab, const double *__restrict__ T32,
                                           double *low_out) {
  const bool is_low = x < kGX0;
  const double xc = fmin(x, 708.0);                                                        // beyond: G < 1e-298
  const bool is_mid = !is_low && xc < kGX1;
  bool need_low = true, need_mid = true, need_hi = true;
  if (VOTE) {
    const unsigned act = __activemask();
    need_low = __any_sync(act, is_low);
    need_mid = __any_sync(act, is_mid);
    need_hi = __any_sync(act, !is_low && !is_mid);
  }
  double low = 0.0;
  if (need_low) {
    // x < 1.5: Bernoulli series of int_0^x; coefficients B_k / ((k+3) k!), k = 0,1,2,4,...,30
    const double xs = fmin(x, kGX0);
    const double x2 = xs * xs;
    double s = 8615841276005.0 / (14322.0 * 33.0 * 265252859812191058636308480000000.0);    // k=30
    s = fma(s, x2, -23749461029.0 / (870.0 * 31.0 * 304888344611713860501504000000.0));      // k=28
    s = fma(s, x2, 8553103.0 / (6.0 * 29.0 * 403291461126605635584000000.0));                // k=26
    s = fma(s, x2, -236364091.0 / (2730.0 * 27.0 * 620448401733239439360000.0));             // k=24
    s = fma(s, x2, 854513.0 / (138.0 * 25.0 * 1124000727777607680000.0));                    // k=22
    s = fma(s, x2, -174611.0 / (330.0 * 23.0 * 2432902008176640000.0));                      // k=20
    s = fma(s, x2, 43867.0 / (798.0 * 21.0 * 6402373705728000.0));                           // k=18
    s = fma(s, x2, -3617.0 / (510.0 * 19.0 * 20922789888000.0));                             // k=16
    s = fma(s, x2, 7.0 / (6.0 * 17.0 * 87178291200.0));                                      // k=14
    s = fma(s, x2, -691.0 / (2730.0 * 15.0 * 479001600.0));                                  // k=12
    s = fma(s, x2, 1.0 / 622702080.0);                                                       // k=10
    s = fma(s, x2, -1.0 / 13305600.0);                                                       // k=8
    s = fma(s, x2, 1.0 / 272160.0);                                                          // k=6 : (1/42)/(9*720)
    s = fma(s, x2, -1.0 / 5040.0);                                                           // k=4 : (-1/30)/(7*24)
    s = fma(s, x2, 1.0 / 60.0);                                                              // k=2 : (1/6)/(5*2)
    low = x2 * xs * fma(x2, s, fma(-1.0 / 8.0, xs, 1.0 / 3.0));                              // x^3 (1/3 - x/8 + x^2 s)
  }
  // x >= 1.5: e^-x times a polynomial
  double G_big = 0.0;
  if (need_mid || need_hi) {
    const double u = exp_hot<1, false>(xc, T32, nullptr);
    double p_mid = 0.0, p_hi = 0.0;
    if (need_mid) {
      int iv = (int)((xc - kGX0) * (1.0 / kGH));
      iv = iv < 0 ? 0 : (iv > kGIntervals - 1 ? kGIntervals - 1 : iv);
      const double t = fmin(fmax(xc - (kGX0 + kGH * 0.5 + kGH * (double)iv), -kGH), kGH);
      const double2 *c = reinterpret_cast<const double2 *>(gtab + iv * kGCoef);
      const double2 c01 = __ldg(c), c23 = __ldg(c + 1), c45 = __ldg(c + 2), c67 = __ldg(c + 3), c89 = __ldg(c + 4);
      const double t2 = t * t, t4 = t2 * t2, t8 = t4 * t4;
      const double p01 = fma(c01.y, t, c01.x), p23 = fma(c23.y, t, c23.x), p45 = fma(c45.y, t, c45.x),
                   p67 = fma(c67.y, t, c67.x), p89 = fma(c89.y, t, c89.x);
      const double q0 = fma(p23, t2, p01), q1 = fma(p67, t2, p45);
      p_mid = fma(p89, t8, fma(q1, t4, q0));
    }
    if (need_hi) {
      const double p1 = fma(fma(fma(xc, 1.0, 3.0), xc, 6.0), xc, 6.0);               // x^3 + 3x^2 + 6x + 6
      const double p2 = fma(fma(fma(xc, 0.5, 0.75), xc, 0.75), xc, 0.375);           // x^3/2 + 3x^2/4 + 6x/8 + 6/16
      p_hi = fma(u, p2, p1);
    }
    G_big = u * (is_mid ? p_mid : p_hi);
  }
  *low_out = is_low ? low : -1.0;
  return is_low ? (kPi * kPi * kPi * kPi / 15.0 - low) : (x > 708.0 ? 0.0 : G_big);
}

// G(x_hi_edge) - G(x_lo_edge) for one bin from the per-edge (G, low) pairs (edge e = lam_lo: larger x)
__device__ __forceinline__ double planck_dG(double G_lo_edge, double low_lo_edge, double G_hi_edge, double low_hi_edge) {
  return (low_lo_edge >= 0.0 && low_hi_edge >= 0.0) ? (low_lo_edge - low_hi_edge) : (G_hi_edge - G_lo_edge);
}

}  // namespace hrt
