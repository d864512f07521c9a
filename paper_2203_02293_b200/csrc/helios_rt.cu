// helios_rt.cu -- B200 (sm_100a) implementation of the THOR+HELIOS radiative-transfer step.
//
// C ABI: include/helios_rt.h.  Citations are PAPER.md lines (arXiv 2203.02293); R-numbers are DESIGN.md readings.
//
// ONE launch per step: rt_step_kernel, a persistent grid of (tiles per column) x (workers) thread blocks.  A block
// is bound to one tile of the (bin, Gauss point) axis for the whole launch -- so its per-bin optical constants,
// weights and table addresses are built once -- and pulls atmospheric columns from its tile's queue.  Per column:
//
//   S1  level geometry: interface p, T (R9), layer masses, k-table cell + bilinear corner weights per level
//   S2  band Planck B_b(T_level) for the tile's bins (piecewise-polynomial G, helios_rt_math.cuh), pi B_b(T_int)
//       -- both computed by the block itself into shared memory (no second kernel, no workspace round trip)
//   sweep 1 (TOA -> BOA), one thread = PPT adjacent spectral points of one bin, each a monochromatic two-stream
//       problem (the unit the paper solves independently, L449/L592): S3 bilinear ln(kappa) + exp (the four
//       k-table corner rows of a level reach shared memory by one-dimensional bulk async copies -- TMA -- into a
//       per-warp two-stage ring guarded by mbarriers, or by register-prefetched loads), S4 omega0/g0/dtau, tau
//       prefix and direct beam (Eq. B6), S5 layer coefficients (Eq. 19, B1, B2, B5, B8, Eq. 11 guard) and the
//       forward elimination of S6.  The block-tridiagonal system of Eq.(12) has one non-zero in each off-diagonal
//       2x2 block, so Eqs.(13)-(14) reduce to the scalar recurrences (R, U, c, d) below, carried in registers.
//       The back-substitution coefficients (c, W d, R) of every interface go to a per-block slab of a global
//       workspace sized to the resident grid (coalesced 16-byte stores), which the persistent block reuses column
//       after column, so it lives in L2; its lines are discarded (discard.global.L2) once sweep 2 has read them.
//   sweep 2 (BOA -> TOA): back-substitution Eq.(15) fused with S7, the Gauss-/bin-weighted reduction (shared-memory
//       transposes + warp shuffles, then a fixed-order sum over warps and tiles).
//
//   rt_iter_kernel   the pair-wise iterative scheme the paper replaces (helios_rt_step_iterative; comparison only).
//
// The layer relations are used in transmission/reflection form.  With zeta+- and T of Eq.(B2),
//   t = psi/chi = s T / (a b),  r = -xi/chi = zeta+ zeta- (1 - T^2) / (a b),
//   a = zeta+ - zeta- T,  b = zeta+ + zeta- T,  s = zeta+ - zeta-,  1 - t - r = s (1 - T) / b,
// Eqs.(2),(3) read  F_up[j+1] = t F_up[j] + r F_dn[j+1] + S_up,  F_dn[j] = t F_dn[j+1] + r F_up[j] + S_dn.
// These forms avoid the cancellations of chi + xi - psi and 1 - T^2.

#include "../../include/helios_rt.h"
#include "../../include/helios_rt_debug.h"
#include "helios_rt_math.cuh"

#include <stdlib.h>
#include <string.h>
#include <new>
#include <type_traits>

namespace {

using namespace hrt;

constexpr int MAXL = HELIOS_RT_MAX_LAYERS;

// unroll factor of the isothermal sweep-1 loop (1: measured best; comparison builds override it)
#ifndef HRT_UNROLL_ISO
#define HRT_UNROLL_ISO 1
#endif
#ifndef HRT_PA_UNROLL
#define HRT_PA_UNROLL 2   /* config 2: 0.6787 ms at 2, 0.6845 at 4, 0.6851 at 8 */
#endif
#ifndef HRT_VOTE_SEL
#define HRT_VOTE_SEL (!TOA)
#endif
#define HRT_PRAGMA(x) _Pragma(#x)
#define HRT_UNROLL(n) HRT_PRAGMA(unroll n)

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

// phase A, per bin: where its Planck value goes (slots in doubles from the row's start; s1 = -1: one tile only,
// s1 = -2: more than two tiles own points of the bin -- the CSR lists them all) and 1 / (lam_hi - lam_lo)
struct __align__(16) BinSlot { int s0, s1; double inv_dlam; };

// S1 result per (column, level), built by phase A in the workspace
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
  const double *lnk;      // [nP][nT][row_stride] ln(kappa); rows padded to an even length, + a tail pad
  const double *tab_lp;   // [nP] log10(p)
  const double *tab_t;    // [nT]
  const double *edges;    // [nb+1]
  const double *gauss_w;  // [ng]
  const BinConst *bins;   // [nb]
  const double *gtab;     // Planck polynomial pieces (build_planck_table)
  const double *c2lam;    // [nb+1] h c / (k lam_edge): x = c2lam / T
  int nP, nT, N, nlev, nb, ng, npt, tiles, ncol;
  unsigned row_stride;
  double inv_dlp, inv_dt;   // 1 / mean spacing of the table grids: first guess of the cell search
  double cloud_p_top, cloud_p_bot, inv_g, inv_cp, inv_eps2, e_tau, gcrit_tol, w0_transition, f_toa;
  // per-step
  const double *p, *T, *mu, *fstar;
  double T_int;
  double *F_up, *F_down, *F_net, *dTdt, *F_beam, *F_toa_bin;
  // workspace
  unsigned char *ws_rec;  // [ncol] per-column record block (Lay::rec_bytes): LevelRec[nlev+1] | layer masses [N] | NaN flag
  unsigned char *ws_B;    // [ncol][tiles] per-(column, tile) band Planck block (Lay::b_bytes): [nlev+1][nbt], last row pi B(T_int)
  unsigned *flags;        // [ncol] levels of the column whose phase-A item is published (nlev + 1 = ready); zeroed
                          // again by the last block of the launch
  const int *slot_ptr;    // [nb+1] CSR: bin b's value goes to slots[slot_ptr[b] .. slot_ptr[b+1]) ...
  const int *slots;       // ... = (tile t) (b_bytes/8) + (b - first bin of tile t), for every tile t that owns points of b
  const BinSlot *bslot;   // [nb] the first two slots and 1/dlam of each bin in one 16-byte record
  int fused_prep;         // 1: rt_step_kernel runs phase A itself (cooperative launch: the whole grid is resident)
  double *stack;          // [blocks of the grid][N+1][warps][96 PPT] back-substitution coefficients
  size_t stack_block;     // doubles per block
  double *partial;        // [ncol][tiles][4][N+1]
  unsigned *counter;      // [ncol]   tiles of the column that have published their partial sums
  unsigned *queue;        // [tiles]  next column of each tile's queue;  queue[tiles] = blocks that have finished;
                          // queue[tiles + 1] = blocks that have finished phase A
};

// --------------------------------------------------------------------------------------------
// S5 for one (sub-)layer between a lower level "a" and an upper level "b": transmission t = psi/chi, reflection
// r = -xi/chi and the sources of  F_up[b] = t F_up[a] + r F_dn[b] + S_up,  F_dn[a] = t F_dn[b] + r F_up[a] + S_dn.
// --------------------------------------------------------------------------------------------
// the terms of S5 that depend on the asymmetry factor g0 alone.  On isothermal columns g0 is a per-(bin, cloud flag)
// constant, so they are built once per block (BinOpt); non-isothermal sub-layers average g0 and build them here.
struct G0Terms {
  double g0;
  double fg;   // Eq.(19): 1.225 - 0.1582 g0 - 0.07465 g0^2
  double fA;   // Eq.(19): -0.1777 + 0.2351 g0   (fit = fg + w0 (fA - 0.05582 w0))
  double geh;  // g0 / (2 eps2), (B8)
};
__device__ __forceinline__ G0Terms g0_terms(double g0, double inv_eps2) {
  G0Terms t;
  t.g0 = g0;
  t.fg = fma(g0, fma(kHC.fc, g0, kHC.fb), kHC.fa);
  t.fA = fma(g0, kHC.fe, kHC.fd);
  t.geh = 0.5 * g0 * inv_eps2;
  return t;
}

template <bool DAY, bool LINSRC>
__device__ __forceinline__ void layer_coeffs(const KParams &P, const double *__restrict__ T32, double w0, const G0Terms &gt,
                                             double dtau, double Ba, double Bb, double mu, double Fa, double Fb,
                                             double &t_out, double &r_out, double &Sup_out, double &Sdn_out) {
  // E, Eq.(19) L374 (readings R5, R6): E = max(1, fit) if w0 > 0.1 else 1
  const double g0 = gt.g0;
  const double fit = fma(w0, fma(kHC.ff, w0, gt.fA), gt.fg);
  // (one predicate, two selects: w0 > transition on the 64-bit pattern; fit >= 1 on the high word alone -- fit = 1
  // gives E = 1 either way.  Regular two-stream: the transition is +inf, launch_step)
  double E;
  asm("{\n\t.reg .pred p, q;\n\t"
      "setp.gt.s64 p, %1, %2;\n\t"
      "setp.ge.and.s32 q, %3, 0x3ff00000, p;\n\t"
      "selp.f64 %0, %4, 0d3FF0000000000000, q;\n\t}"
      : "=d"(E)
      : "l"(__double_as_longlong(w0)), "l"(__double_as_longlong(P.w0_transition)), "r"(__double2hiint(fit)), "d"(fit));
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
  const double Tr = exp_hot<2, true>(cap_pos<0x40762000>(ha * dtau), T32, &omT);   // transmission function (B2), 1 - T; argument capped near 354
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
    const double ma = (mu + mu) * ha;                        // (mu + mu: loop-invariant)
    double D = (ma - 1.0) * (ma + 1.0);                      // 4 E mu^2 (E-w0)(1-w0 g0) - 1
    D = abs_lt(D, P.gcrit_tol) ? -2.0 * mu : D;
    const double invD = rcp_fast(D);
    const double hP = 0.5 * (num * rs2);                     // 1 / (2 E (1 - w0 g0))
    const double geh = gt.geh;                               // g0 / (2 eps2)
    const double lead = (w0 * (den + geh)) * invD;           // (w0/2) (2 E (1 - w0 g0) + g0/eps2) / D
    const double last = w0 * (geh * hP);
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

// --------------------------------------------------------------------------------------------
// shared-memory layout of one block, PTX helpers
// --------------------------------------------------------------------------------------------
constexpr int STAGE_LD = 36;   // row stride (doubles) of the per-warp 8 x 32 staging tile: conflict-free transpose
constexpr int RING = 2;        // stages of the per-warp k-table row ring (one stage = the rows of one sweep iteration)

// per bin of the tile: [0][bin] clear level, [1][bin] cloudy level.  gt: the g0-only terms of S5 (G0Terms)
struct __align__(16) BinOpt { double sb, ss; G0Terms gt; double pad[2]; };
static_assert(sizeof(BinOpt) == 64, "BinOpt layout");

struct Lay {
  int nbt;         // max bins per tile
  int LP;          // N + 1 rounded up to a multiple of 8 (the reductions handle 8 interfaces at a time)
  unsigned rec_bytes, b_bytes;     // sizes of the per-column record block and of the per-(column, tile) Planck block
  unsigned off_rec[2], off_Bt[2];  // both double-buffered: the next column's blocks arrive while this one is swept
  unsigned off_bin, off_red, off_fin, off_vals, off_bar, off_u, total;   // off_u: per-warp sweep scratch
  unsigned u_stage, u_ring, ring_warp;                   // sweep view: [warp] staging tile; [warp] row ring
};

// ppt: spectral points per thread; depth: levels per sweep iteration (1 isothermal, 2 non-isothermal); rows: 1 TMA ring;
// bdirect: one Gauss point per bin -- the Planck block is read from the workspace, not staged
__host__ __device__ inline Lay make_lay(int N, int nlev, int warps, int ppt, int ng, int nb, bool toa, int depth, int rows,
                                        bool bdirect) {
  Lay L;
  const int tp = warps * 32 * ppt;
  const int nbt = bdirect ? tp : (tp + ng - 1) / ng + 1;   // bins a tile can touch (a tile may start inside a bin; one point per bin: tp)
  L.nbt = nbt < nb ? nbt : nb;
  L.LP = (N + 1 + 7) & ~7;
  L.rec_bytes = (unsigned)((sizeof(LevelRec) * (nlev + 1) + sizeof(double) * (N + 1) + 15) & ~size_t(15));   // LevelRec[nlev+1] | dm[N] | mu
  L.b_bytes = (unsigned)((sizeof(double) * (nlev + 1) * L.nbt + 15) & ~size_t(15));
  unsigned o = 0;
  auto take = [&](size_t bytes) { unsigned r = o; o += (unsigned)((bytes + 127) & ~size_t(127)); return r; };
  L.off_rec[0] = take(L.rec_bytes);
  L.off_rec[1] = take(L.rec_bytes);
  L.off_Bt[0] = take(bdirect ? 0 : L.b_bytes);
  L.off_Bt[1] = take(bdirect ? 0 : L.b_bytes);
  L.off_bin = take(sizeof(BinOpt) * 2 * L.nbt);
  L.off_red = take(toa ? 0 : sizeof(double) * warps * 4 * L.LP);       // F_up, R F_up, U + beam, beam
  L.off_fin = take(toa ? 0 : sizeof(double) * 4 * (N + 1));
  L.off_vals = take(sizeof(double) * tp);
  L.off_bar = take(8 * (RING * warps + 2));                            // row-ring barriers, then the two record barriers
  L.off_u = o;
  unsigned u = 0;
  auto utake = [&](size_t bytes) { unsigned r = u; u += (unsigned)((bytes + 15) & ~size_t(15)); return r; };
  // sweep scratch
  L.u_stage = utake(toa ? 0 : sizeof(double) * warps * 8 * STAGE_LD);
  u = (u + 127) & ~127u;
  L.ring_warp = rows == 1 ? (unsigned)(RING * depth * 4 * 32 * ppt * 8) : 0;
  L.u_ring = utake((size_t)L.ring_warp * warps);
  L.total = L.off_u + u;
  return L;
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// one-dimensional bulk async copy global -> shared (TMA; SASS UBLKCP), completion counted on the mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "HRT_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra HRT_DONE;\n"
      "bra HRT_WAIT;\n"
      "HRT_DONE:\n"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// drop a 128-byte line from L2 without writing it back (its contents are dead)
__device__ __forceinline__ void l2_discard(const void *p) {
  asm volatile("discard.global.L2 [%0], 128;" ::"l"(p) : "memory");
}

// address of element `off` (32-bit, unsigned) of a double array: one IMAD.WIDE.U32
__device__ __forceinline__ const double *elem_addr(const double *base, unsigned off) {
  unsigned long long a;
  asm("mad.wide.u32 %0, %1, 8, %2;" : "=l"(a) : "r"(off), "l"((unsigned long long)base));
  return (const double *)a;
}

// the four k-table corner values of PPT adjacent spectral points at one level
template <int PPT> struct RowsT { double v[4][PPT]; };

template <int PPT>
__device__ __forceinline__ void load_rows_g(RowsT<PPT> &r, const double *__restrict__ lnk_pt, const LevelRec *lv) {
  const uint4 o = *reinterpret_cast<const uint4 *>(&lv->o00);
  const unsigned off[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const double *a = elem_addr(lnk_pt, off[c]);
    if (PPT == 1) {
      r.v[c][0] = __ldg(a);
    } else {
#pragma unroll
      for (int h = 0; h < PPT / 2; ++h) {
        const double2 t = __ldg(reinterpret_cast<const double2 *>(a) + h);
        r.v[c][2 * h] = t.x;
        r.v[c][2 * h + 1] = t.y;
      }
    }
  }
}

// st: one level of a ring stage, [4][32 PPT] doubles
template <int PPT>
__device__ __forceinline__ void load_rows_s(RowsT<PPT> &r, const double *st, int lane) {
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const double *a = st + c * 32 * PPT + lane * PPT;
    if (PPT == 1) {
      r.v[c][0] = *a;
    } else {
#pragma unroll
      for (int h = 0; h < PPT / 2; ++h) {
        const double2 t = reinterpret_cast<const double2 *>(a)[h];
        r.v[c][2 * h] = t.x;
        r.v[c][2 * h + 1] = t.y;
      }
    }
  }
}

// Row feed of the sweep: DEPTH levels per iteration, top-down.  ROWS = 0: the next iteration's rows are held in
// registers: an iteration first consumes them (next), then re-loads the same registers for the following iteration
// (release) -- no copy, the loads are in flight for a whole iteration.  ROWS = 1: a per-warp ring of RING stages in
// shared memory, filled by bulk async copies that lane 0 issues two iterations ahead; each stage has its own mbarrier
// (expect-tx = the stage's bytes); the warp re-arms a stage itself once all its lanes have consumed it, so warps never
// wait on each other.  `kc` counts iterations since the barriers were initialised and runs across columns: iteration
// kc uses stage kc % RING in phase (kc / RING) & 1.
template <int PPT, int DEPTH, int ROWS> struct Feed;

template <int PPT, int DEPTH> struct Feed<PPT, DEPTH, 0> {
  RowsT<PPT> nx[DEPTH];
  const double *lnk_pt;
  const LevelRec *lv0;   // record of level 0 (lowest): prefetches below it are clamped
  __device__ __forceinline__ void load(const LevelRec *lv) {
#pragma unroll
    for (int d = 0; d < DEPTH; ++d) {
      const LevelRec *q = lv - d;
      load_rows_g<PPT>(nx[d], lnk_pt, q < lv0 ? lv0 : q);
    }
  }
  // lv: highest level of the first iteration
  __device__ __forceinline__ void prime(const LevelRec *lv, int /*iterations*/) { load(lv); }
  // the rows of this iteration (valid until release)
  __device__ __forceinline__ const RowsT<PPT> *next() { return nx; }
  // call once the iteration's rows have been used; lv_next: highest level of the next iteration
  __device__ __forceinline__ void release(const LevelRec *lv_next, const LevelRec *, bool) { load(lv_next); }
};

template <int PPT, int DEPTH> struct Feed<PPT, DEPTH, 1> {
  static constexpr uint32_t ROWB = 32 * PPT * 8, STGB = DEPTH * 4 * ROWB;
  RowsT<PPT> cur[DEPTH];
  const double *ring;    // this warp's ring (generic address)
  uint32_t ring_s, bar_s;
  const double *lnk_w;   // ln(kappa) table + first spectral point of the warp
  const LevelRec *lv0;
  uint32_t kc;
  int lane;
  __device__ __forceinline__ void fill(uint32_t stage, const LevelRec *lv) {   // lane 0
    const uint32_t bar = bar_s + 8 * stage, dst = ring_s + stage * STGB;
    mbar_expect_tx(bar, STGB);
#pragma unroll
    for (int d = 0; d < DEPTH; ++d) {
      const LevelRec *q = lv - d;
      q = q < lv0 ? lv0 : q;
      const uint4 o = *reinterpret_cast<const uint4 *>(&q->o00);
      bulk_g2s(dst + (d * 4 + 0) * ROWB, lnk_w + o.x, ROWB, bar);
      bulk_g2s(dst + (d * 4 + 1) * ROWB, lnk_w + o.y, ROWB, bar);
      bulk_g2s(dst + (d * 4 + 2) * ROWB, lnk_w + o.z, ROWB, bar);
      bulk_g2s(dst + (d * 4 + 3) * ROWB, lnk_w + o.w, ROWB, bar);
    }
  }
  __device__ __forceinline__ void prime(const LevelRec *lv, int iterations) {
    if (lane == 0) {
      fill(kc % RING, lv);
      if (iterations > 1) fill((kc + 1) % RING, lv - DEPTH);
    }
  }
  __device__ __forceinline__ const RowsT<PPT> *next() {
    const uint32_t stage = kc % RING;
    mbar_wait(bar_s + 8 * stage, (kc / RING) & 1u);
    const double *st = ring + (size_t)stage * (STGB / 8);
#pragma unroll
    for (int d = 0; d < DEPTH; ++d) load_rows_s<PPT>(cur[d], st + d * 4 * 32 * PPT, lane);
    return cur;
  }
  // call once the iteration's rows are in registers and have been used; lv_refill: highest level of the iteration
  // RING ahead (has = false: none left in this column)
  __device__ __forceinline__ void release(const LevelRec *, const LevelRec *lv_refill, bool has) {
    __syncwarp();
    if (lane == 0 && has) fill(kc % RING, lv_refill);
    ++kc;
  }
};

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

// Back-substitution workspace of one warp: N + 1 rows of 96 PPT doubles, row stride compile-time (immediate offsets).
// Row i holds (c_i, W d_i) of interface i [F_up[i] = c_i F_up[i-1] + d_i] and R_{i-1} [F_dn = R F_up + U at interface
// i-1]: the sweep stores R after the layer update, so no copy of the old R is kept (R_N = 0 is not stored).
// PPT = 1: [c][W d][R] x 32 lanes; PPT >= 2: 16-byte slots [q: (c, W d)] x 32 lanes, then [h: (R_2h, R_2h+1)] x 32
// lanes.  L2 only (.cg).
template <int PPT>
__device__ __forceinline__ void stk_store(double *row, int lane, const double (&c)[PPT], const double (&wd)[PPT],
                                          const double (&R)[PPT]) {
  if (PPT == 1) {
    __stcg(row + lane, c[0]);
    __stcg(row + 32 + lane, wd[0]);
    __stcg(row + 64 + lane, R[0]);
  } else {
    double2 *v = reinterpret_cast<double2 *>(row) + lane;
#pragma unroll
    for (int q = 0; q < PPT; ++q) __stcg(v + q * 32, make_double2(c[q], wd[q]));
#pragma unroll
    for (int h = 0; h < PPT / 2; ++h) __stcg(v + (PPT + h) * 32, make_double2(R[2 * h], R[2 * h + 1]));
  }
}
// (c, W d) of a row / the R of a row
template <int PPT>
__device__ __forceinline__ void stk_load_cw(const double *row, int lane, double (&c)[PPT], double (&wd)[PPT]) {
  if (PPT == 1) {
    c[0] = __ldcg(row + lane);
    wd[0] = __ldcg(row + 32 + lane);
  } else {
    const double2 *v = reinterpret_cast<const double2 *>(row) + lane;
#pragma unroll
    for (int q = 0; q < PPT; ++q) { const double2 t = __ldcg(v + q * 32); c[q] = t.x; wd[q] = t.y; }
  }
}
template <int PPT>
__device__ __forceinline__ void stk_load_R(const double *row, int lane, double (&R)[PPT]) {
  if (PPT == 1) {
    R[0] = __ldcg(row + 64 + lane);
  } else {
    const double2 *v = reinterpret_cast<const double2 *>(row) + lane;
#pragma unroll
    for (int h = 0; h < PPT / 2; ++h) { const double2 t = __ldcg(v + (PPT + h) * 32); R[2 * h] = t.x; R[2 * h + 1] = t.y; }
  }
}

// --------------------------------------------------------------------------------------------
// Phase A: S1 + S2.  One work item = one (column, level); items are independent (a thread recomputes the two or
// three ln p of its neighbours instead of sharing them), so they are spread over all threads of the grid with no
// barrier.  Results go to the workspace, read back by the sweeping blocks through bulk async copies.
//   S1 (L171, R9, R7): the level's p, T (interfaces by linear interpolation in ln p; ends extrapolated half a step
//       with T held), its LevelRec -- the four bilinear corner weights (1-w_p)(1-w_T) ..., the four k-table row
//       offsets, the (sub-)layer column mass, the cloud flag, a NaN flag (R19) -- and the layer mass for R14.
//   S2 (L171, L239, R8): the level's row of band Planck values: the thread walks the bin edges keeping the previous
//       edge's G (two edges per trip for instruction-level parallelism; consecutive lanes = consecutive levels of one
//       column, so a warp's x = hc/(lam k T) stay close and its lanes take the same branch of planck_G); every bin's
//       B_b goes to the Planck block of each tile that owns points of the bin (slots CSR).  The extra level nlev
//       carries T_int and yields F_BOA,b = pi B_b(T_int).
// --------------------------------------------------------------------------------------------
template <bool NONISO, bool VOTE, bool PACK4>
__device__ __forceinline__ void prep_item(const KParams &P, const Lay &L, const double *__restrict__ T32, int col, int l) {
  const int N = P.N, nlev = P.nlev;
  const double *pc = P.p + (size_t)col * N;
  const double *Tc = P.T + (size_t)col * N;
  unsigned char *rec = P.ws_rec + (size_t)col * L.rec_bytes;
  LevelRec *g_rec = (LevelRec *)rec;    // record 0 duplicates level 0 (prefetch pad); level l at [l + 1]
  double *g_dm = (double *)(rec + sizeof(LevelRec) * (nlev + 1));
  // ln p at interface i of the column (R9)
  auto lnp_int = [&](int i) -> double {
    if (N == 1) return log(pc[0]) + (i == 0 ? 0.5 : -0.5) * 2.302585092994045684;
    if (i == 0) { const double a = log(pc[0]); return a + 0.5 * (a - log(pc[1])); }
    if (i == N) { const double a = log(pc[N - 1]); return a - 0.5 * (log(pc[N - 2]) - a); }
    return 0.5 * (log(pc[i - 1]) + log(pc[i]));
  };
  auto T_int_face = [&](int i) -> double {
    if (N == 1 || i == 0) return Tc[0];
    if (i == N) return Tc[N - 1];
    return 0.5 * (Tc[i - 1] + Tc[i]);
  };
  double Tl;
  if (l < nlev) {
    double pl, lnpl, dm;
    if (!NONISO) {
      pl = pc[l]; Tl = Tc[l]; lnpl = log(pl);
      dm = (exp(lnp_int(l)) - exp(lnp_int(l + 1))) * P.inv_g;     // the layer between its two interfaces
      g_dm[l] = dm;
    } else if (l & 1) {
      const int i = l >> 1;                                      // centre of layer i; above it: interface i + 1
      pl = pc[i]; Tl = Tc[i]; lnpl = log(pl);
      const double p_up = exp(lnp_int(i + 1));
      dm = (pl - p_up) * P.inv_g;
      g_dm[i] = (exp(lnp_int(i)) - p_up) * P.inv_g;
    } else {
      const int i = l >> 1;                                      // interface i; above it: centre of layer i
      lnpl = lnp_int(i); pl = exp(lnpl); Tl = T_int_face(i);
      dm = (l < nlev - 1) ? (pl - pc[i]) * P.inv_g : 0.0;
    }
    LevelRec r;
    r.dm = dm;
    r.cloud = (pl >= P.cloud_p_top && pl <= P.cloud_p_bot) ? 1 : 0;
    r.pad = (pl != pl || Tl != Tl) ? 1 : 0;                       // NaN in the column's p or T
    // table cell + weights: bilinear in (log10 p, T), clamped (R7).  Cell = the one with grid[i] < x <= grid[i+1]
    // (x at or below the first node: cell 0); found from a uniform-grid guess corrected by a walk.
    double xp = lnpl * 0.43429448190325182765;
    xp = fmin(fmax(xp, P.tab_lp[0]), P.tab_lp[P.nP - 1]);
    int ip = (int)((xp - P.tab_lp[0]) * P.inv_dlp);
    ip = ip < 0 ? 0 : (ip > P.nP - 2 ? P.nP - 2 : ip);
    while (ip > 0 && !(xp > P.tab_lp[ip])) --ip;
    while (ip < P.nP - 2 && xp > P.tab_lp[ip + 1]) ++ip;
    const double wp = (xp - P.tab_lp[ip]) / (P.tab_lp[ip + 1] - P.tab_lp[ip]);
    const double xt = fmin(fmax(Tl, P.tab_t[0]), P.tab_t[P.nT - 1]);
    int it = (int)((xt - P.tab_t[0]) * P.inv_dt);
    it = it < 0 ? 0 : (it > P.nT - 2 ? P.nT - 2 : it);
    while (it > 0 && !(xt > P.tab_t[it])) --it;
    while (it < P.nT - 2 && xt > P.tab_t[it + 1]) ++it;
    const double wt = (xt - P.tab_t[it]) / (P.tab_t[it + 1] - P.tab_t[it]);
    r.c00 = (1.0 - wp) * (1.0 - wt);
    r.c01 = (1.0 - wp) * wt;
    r.c10 = wp * (1.0 - wt);
    r.c11 = wp * wt;
    r.o00 = (unsigned)(ip * P.nT + it) * P.row_stride;
    r.o01 = r.o00 + P.row_stride;
    r.o10 = r.o00 + (unsigned)P.nT * P.row_stride;
    r.o11 = r.o10 + P.row_stride;
    g_rec[1 + l] = r;
    if (l == 0) g_rec[0] = r;
  } else {
    Tl = P.T_int;
    const double mu = P.mu[col];
    g_dm[N] = mu;                                                 // mu rides along with the records
  }

  // ---------------- S2 ----------------
  double *Brow = (double *)(P.ws_B + (size_t)col * P.tiles * L.b_bytes) + (size_t)l * L.nbt;
  const bool hot = Tl > 0.0;
  const double invT = hot ? 1.0 / Tl : 0.0;
  const double T2 = Tl * Tl;
  const double scale = hot ? ((l == nlev) ? kPlanckC1 * kPi : kPlanckC1) * T2 * T2 : 0.0;   // row nlev: F_BOA = pi B(T_int), L239
  double low_p = 0.0, G_p = planck_G<VOTE>(__ldg(P.c2lam) * invT, P.gtab, T32, &low_p);
  auto one_bin = [&](int e) {
    double low_a;
    const double G_a = planck_G<VOTE>(__ldg(P.c2lam + e + 1) * invT, P.gtab, T32, &low_a);
    const int4 raw = __ldg(reinterpret_cast<const int4 *>(P.bslot + e));
    const double inv_dlam = __hiloint2double(raw.w, raw.z);
    const double B = scale * planck_dG(G_p, low_p, G_a, low_a) * inv_dlam;
    Brow[raw.x] = B;
    if (raw.y >= 0) Brow[raw.y] = B;
    else if (raw.y == -2)
      for (int k = __ldg(P.slot_ptr + e) + 1; k < __ldg(P.slot_ptr + e + 1); ++k) Brow[__ldg(P.slots + k)] = B;
    G_p = G_a; low_p = low_a;
  };
  if constexpr (PACK4) {
    int e = 0;
    if (P.ng == 1 && (L.nbt & 3) == 0) {
      // one Gauss point per bin (opacity sampling, thousands of bins): every bin has one slot, tiles hold a multiple of
      // 4 bins and rows are 32-byte aligned, so four consecutive bins leave as ONE 32-byte store (a whole sector) instead
      // of four 8-byte stores into it (config 6: RT step 10.6 -> 8.0 ms)
#pragma unroll 1
      for (; e + 4 <= P.nb; e += 4) {
        double B4[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          double low_a;
          const double G_a = planck_G<VOTE>(__ldg(P.c2lam + e + k + 1) * invT, P.gtab, T32, &low_a);
          B4[k] = scale * planck_dG(G_p, low_p, G_a, low_a) * __ldg(&P.bslot[e + k].inv_dlam);
          G_p = G_a; low_p = low_a;
        }
        double *dst = Brow + __ldg(&P.bslot[e].s0);
        asm volatile("st.global.L1::no_allocate.v4.b64 [%0], {%1, %2, %3, %4};" ::"l"(dst), "l"(__double_as_longlong(B4[0])),
                     "l"(__double_as_longlong(B4[1])), "l"(__double_as_longlong(B4[2])), "l"(__double_as_longlong(B4[3]))
                     : "memory");
      }
    }
    for (; e < P.nb; ++e) one_bin(e);
  } else {
HRT_UNROLL(HRT_PA_UNROLL)
    for (int e = 0; e < P.nb; ++e) one_bin(e);
  }
}

// phase A over the whole grid: item = (column, level) in column-major order
template <bool NONISO, bool VOTE, bool PACK4>
__device__ __forceinline__ void phase_a(const KParams &P, const Lay &L, const double *__restrict__ T32, long gtid, long gthreads,
                                        bool count) {
  const int nlevp = P.nlev + 1;
  const long nitems = (long)P.ncol * nlevp;
  for (long item = gtid; item < nitems; item += gthreads) {
    const int col = (int)(item / nlevp), l = (int)(item - (long)col * nlevp);
    prep_item<NONISO, VOTE, PACK4>(P, L, T32, col, l);
    if (count) {
      // count the warp's items of each column with one fence + one atomic (the warp barrier + the leader's fence
      // order every lane's stores before the count)
      const unsigned act = __activemask();
      const unsigned same = __match_any_sync(act, col);
      __syncwarp(act);
      if ((threadIdx.x & 31) == __ffs(same) - 1) {
        __threadfence();
        atomicAdd(P.flags + col, (unsigned)__popc(same));
      }
    }
  }
}

// cross-warp sum of the per-warp interface sums (s_red: [warp][4][LP] = F_up, diffuse F_dn part 1, part 2 (+ beam),
// beam), tile partials in fixed order, and the column's outputs written by its last tile.  A tile publishes its
// partial sums with a release atomic (no L1 invalidation); only the column's last tile takes the acquire fence.
__device__ __forceinline__ void column_epilogue(const KParams &P, const Lay &L, unsigned char *smem, const double *s_dm,
                                                int *s_is_last_p, int nwa, bool want_beam, int col, int tile, int col_nan) {
  const int N = P.N, LP = L.LP, tid = threadIdx.x, nthr = blockDim.x;
  double *s_red = (double *)(smem + L.off_red), *s_fin = (double *)(smem + L.off_fin);
  int &s_is_last = *s_is_last_p;
  const int nq = want_beam ? 4 : 3;
  const int nred = nq * (N + 1);
  if (P.tiles > 1) {
    // cross-warp sum in fixed order, published straight to this tile's partial-sum slot
    double *part = P.partial + ((size_t)col * P.tiles + tile) * 4 * (N + 1);
    for (int k = tid; k < nred; k += nthr) {
      const int q = k / (N + 1), lev = k - q * (N + 1);
      double sum = 0.0;
      for (int w = 0; w < nwa; ++w) sum += s_red[(size_t)w * 4 * LP + q * LP + lev];
      __stcg(part + k, sum);
    }
    __syncthreads();
    if (tid == 0) {
      unsigned prev;
      asm volatile("atom.add.release.gpu.global.u32 %0, [%1], 1;" : "=r"(prev) : "l"(P.counter + col) : "memory");
      s_is_last = (prev == (unsigned)(P.tiles - 1));
      if (s_is_last) {
        P.counter[col] = 0;   // re-arm for the next step
        __threadfence();      // acquire side: the other tiles' partial sums are visible below
      }
    }
    __syncthreads();
    if (!s_is_last) return;
    // the column's last tile sums the partial sums in tile order
    const double *pall = P.partial + (size_t)col * P.tiles * 4 * (N + 1);
    for (int k = tid; k < nred; k += nthr) {
      double sum = 0.0;
      for (int t = 0; t < P.tiles; ++t) sum += __ldcg(pall + (size_t)t * 4 * (N + 1) + k);
      s_fin[k] = sum;
    }
    __syncthreads();
  } else {
    for (int k = tid; k < nred; k += nthr) {
      const int q = k / (N + 1), lev = k - q * (N + 1);
      double sum = 0.0;
      for (int w = 0; w < nwa; ++w) sum += s_red[(size_t)w * 4 * LP + q * LP + lev];
      s_fin[k] = sum;
    }
    __syncthreads();
  }

  // final outputs of the column: F_down = sum W R F_up + sum W (U + beam)
  const double poison = col_nan ? nan("") : 0.0;
  for (int i = tid; i <= N; i += nthr) {
    const size_t o = (size_t)col * (N + 1) + i;
    const double fu = s_fin[i] + poison, fd = s_fin[N + 1 + i] + s_fin[2 * (N + 1) + i] + poison;
    if (P.F_up) P.F_up[o] = fu;
    if (P.F_down) P.F_down[o] = fd;
    if (P.F_net) P.F_net[o] = fu - fd;
    if (want_beam) P.F_beam[o] = s_fin[3 * (N + 1) + i] + poison;
  }
  if (P.dTdt) {
    for (int j = tid; j < N; j += nthr) {
      const double fn1 = s_fin[j + 1] - (s_fin[N + 1 + j + 1] + s_fin[2 * (N + 1) + j + 1]);
      const double fn0 = s_fin[j] - (s_fin[N + 1 + j] + s_fin[2 * (N + 1) + j]);
      P.dTdt[(size_t)col * N + j] = -(fn1 - fn0) * P.inv_cp / s_dm[j] + poison;   // reading R14
    }
  }
}

// --------------------------------------------------------------------------------------------
// rt_step_kernel: S1-S7.  Persistent grid = (tiles per column, workers): block (t, w) owns tile t of the spectral axis
// (warps x 32 x PPT consecutive points, bin-major, Gauss point fastest) and takes columns from queue[t].
//   NONISO  non-isothermal layers (Eqs. 4-9): two sub-layers and two levels per sweep iteration
//   TOA     HELIOS_RT_TOA_SPECTRUM: only F_up at the top per bin; no back-substitution
//   PPT     adjacent spectral points of one bin per thread (n_gauss must be a multiple): everything that depends only
//           on (column, level, bin) is issued once for the group and its PPT dependence chains interleave (ILP)
//   ROWS    0: k-table rows by register-prefetched loads; 1: by bulk async copies (TMA) into the per-warp ring
//   BDIRECT one Gauss point per bin (opacity sampling, L385): every thread has its own bin, so the Planck values are
//           read coalesced from the workspace instead of being staged (64 KB per block otherwise); PPT = 1
//   WARPS   warps per block as a compile-time constant, or 0 = taken from the launch
//   MAXT, MINB  launch bounds (register cap = 65536 / (MAXT MINB)); any block of <= MAXT threads may be launched
// --------------------------------------------------------------------------------------------
template <bool NONISO, bool TOA, int PPT, int ROWS, bool BDIRECT, int WARPS, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) rt_step_kernel(const KParams P) {
  static_assert(PPT == 1 || PPT == 2 || PPT == 4, "points per thread");
  static_assert(!BDIRECT || PPT == 1, "one Gauss point per bin: one point per thread");
  constexpr int DEPTH = NONISO ? 2 : 1;
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ double s_T32[32];
  __shared__ int s_is_last, s_col[2];
  const int N = P.N, nlev = P.nlev;
  // WARPS > 0: the block size is a compile-time constant (the shapes helios_rt_create picks); 0: any block <= MAXT
  const int tid = threadIdx.x, nthr = WARPS ? WARPS * 32 : blockDim.x, nwarps = nthr >> 5;
  const int warp = tid >> 5, lane = tid & 31;
  const Lay L = make_lay(N, nlev, nwarps, PPT, P.ng, P.nb, TOA, DEPTH, ROWS, BDIRECT);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  double *s_red = (double *)(smem + L.off_red);
  double *s_vals = (double *)(smem + L.off_vals);
  const int LP = L.LP, nbtS = L.nbt;

  // ---------------- constants of the tile (the block keeps its tile for the whole launch) ----------------
  const int tile = blockIdx.x;
  const int TP = nthr * PPT;
  const int pt0 = tile * TP;
  const int b_first = pt0 / P.ng;
  int pt_last = pt0 + TP - 1;
  if (pt_last > P.npt - 1) pt_last = P.npt - 1;
  const int nbt = pt_last / P.ng - b_first + 1;            // bins touched by this tile (<= L.nbt)
  const int nwa = (pt_last - pt0) / (32 * PPT) + 1;        // warps that own at least one spectral point
  // the group pt .. pt + PPT - 1: pt and n_gauss are multiples of PPT, so all its points lie in bin b
  int pt = pt0 + PPT * tid;
  const bool active = pt < P.npt;
  if (!active) pt = P.npt - PPT;
  const int b = pt / P.ng, gidx = pt - b * P.ng;
  const int bl = b - b_first;
  const bool warp_on = warp < nwa;          // a warp without any spectral point only joins the barriers
  const bool want_beam = !TOA && (P.F_beam != nullptr);
  double W[PPT];                            // dlam_b * w_g
  const double fstar_b = P.fstar[b];
  {
    const double dlam = P.bins[b].dlam;
#pragma unroll
    for (int q = 0; q < PPT; ++q) W[q] = active ? dlam * P.gauss_w[gidx + q] : 0.0;
  }

  if (tid < 32) s_T32[tid] = kExp2Tab[tid];
  for (int i = tid; i < 2 * nbt; i += nthr) {
    const int cl = i / nbt, k = i - cl * nbt;
    const BinConst bc = P.bins[b_first + k];
    BinOpt bo;
    bo.sb = bc.sb[cl]; bo.ss = bc.ss[cl]; bo.gt = g0_terms(bc.gg[cl], P.inv_eps2);
    bo.pad[0] = bo.pad[1] = 0.0;
    s_bin[cl * nbtS + k] = bo;
  }
  if (tid < RING * nwarps + 2) mbar_init(smem_u32(smem + L.off_bar) + 8 * tid, 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  const uint32_t rec_bar = smem_u32(smem + L.off_bar) + 8 * RING * nwarps;   // two barriers: one per record buffer
  const BinOpt *bin0 = s_bin + bl, *bin1 = s_bin + nbtS + bl;
  const double *T32 = s_T32;
  double *red_w = s_red + (size_t)warp * 4 * LP;
  double *stage_w = (double *)(smem + L.off_u + L.u_stage) + (size_t)warp * 8 * STAGE_LD;
  double *stage_wr = stage_w + lane;

  // ---------------- phase A: this block's share of the (column, level) items of S1 + S2 ----------------
#ifdef HRT_DIAG_SKIP_PHASE_A   /* timing-only diagnostic build (_work/): phase A on the handle's first launch only */
  if (P.fused_prep == 1) {
#else
  if (P.fused_prep) {
#endif
    __syncthreads();                       // s_T32
    const long nblk = (long)gridDim.x * gridDim.y;
    // (skipping the Planck forms no lane of a warp needs: -1.2 % on config 2, +0.9 % on config 5 -- per-class choice)
    phase_a<NONISO, HRT_VOTE_SEL, BDIRECT>(P, L, s_T32, ((long)blockIdx.y * gridDim.x + blockIdx.x) * nthr + tid, nblk * nthr, true);
    __syncthreads();
    if (tid == 0) {
      unsigned prev;
      asm volatile("atom.add.release.gpu.global.u32 %0, [%1], 1;" : "=r"(prev) : "l"(P.queue + P.tiles + 1) : "memory");
    }
  }

  Feed<PPT, DEPTH, ROWS> feed;
  if constexpr (ROWS == 0) {
    feed.lnk_pt = P.lnk + pt;
  } else {
    unsigned char *ring = smem + L.off_u + L.u_ring + (size_t)warp * L.ring_warp;
    feed.ring = (const double *)ring;
    feed.ring_s = smem_u32(ring);
    feed.bar_s = smem_u32(smem + L.off_bar) + 8 * RING * warp;
    feed.lnk_w = P.lnk + pt0 + warp * 32 * PPT;
    feed.kc = 0;
    feed.lane = lane;
  }

  // this block's slab of the back-substitution workspace: [warp][N + 1 rows][96 PPT]
  constexpr int SROW = 96 * PPT;            // doubles per row
  double *stk_w = nullptr;
  if (!TOA)
    stk_w = P.stack + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * P.stack_block + (size_t)warp * (N + 1) * SROW;

  // ---------------- phase B: columns of this tile's queue ----------------
  // The record block and the tile's Planck block of the NEXT column are fetched by bulk async copies (TMA) into the
  // other shared-memory buffer while this column is swept; thread 0 first waits for the column's publication flag.
  bool all_published = false;               // thread 0: every block has finished phase A -- no more flag polls
#ifdef HRT_DIAG_SKIP_PHASE_A
  if (P.fused_prep == 2) all_published = true;
#endif
  auto fetch_column = [&](int c, int buf) {   // thread 0
    // (the whole grid is resident -- cooperative launch -- and phase A waits for nothing, so this terminates; the
    // poll count is bounded all the same: a wedged GPU is worse than a wrong column)
    if (!all_published) {
      unsigned n;
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(n) : "l"(P.queue + P.tiles + 1) : "memory");
      all_published = (n == gridDim.x * gridDim.y);
      if (!all_published) {
        unsigned f, polls = 0;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(P.flags + c) : "memory");
        } while (f != (unsigned)(nlev + 1) && ++polls < (1u << 26));
      }
      asm volatile("fence.proxy.async.global;" ::: "memory");
    }
    const uint32_t bar = rec_bar + 8 * buf;
    mbar_expect_tx(bar, L.rec_bytes + (BDIRECT ? 0u : L.b_bytes));
    bulk_g2s(smem_u32(smem + L.off_rec[buf]), P.ws_rec + (size_t)c * L.rec_bytes, L.rec_bytes, bar);
    if (!BDIRECT)
      bulk_g2s(smem_u32(smem + L.off_Bt[buf]), P.ws_B + ((size_t)c * P.tiles + tile) * L.b_bytes, L.b_bytes, bar);
  };
  __syncthreads();                         // tile constants and barriers are set up; phase A scratch is dead
  int pend = 0;                            // thread 0: the queue entry after the next one, fetched one column early
  if (tid == 0) {
    const int c = (int)atomicAdd(P.queue + tile, 1u);
    pend = (int)atomicAdd(P.queue + tile, 1u);
    s_col[0] = c;
    if (c < P.ncol) fetch_column(c, 0);
  }
  __syncthreads();
  for (unsigned it = 0;; ++it) {
    const int buf = it & 1;
    const int col = s_col[buf];
    if (col >= P.ncol) break;
    if (tid == 0) {
      const int c = pend;
      pend = (int)atomicAdd(P.queue + tile, 1u);   // consumed at the top of the next column: its latency is hidden
      s_col[buf ^ 1] = c;
      if (c < P.ncol) fetch_column(c, buf ^ 1);    // the other buffer is free since the barrier that ended the last column
    }
    mbar_wait(rec_bar + 8 * buf, (it >> 1) & 1u);
    const LevelRec *s_lev = (const LevelRec *)(smem + L.off_rec[buf]) + 1;   // s_lev[-1] duplicates level 0
    const double *s_dm = (const double *)(smem + L.off_rec[buf] + sizeof(LevelRec) * (nlev + 1));
    // NaN in p, T or mu of this column poisons the column's outputs (and only them): the clamps and selects of the
    // sweeps would otherwise swallow it (R19).  Level flags from phase A; reduced at the barrier after the sweeps.
    int my_nan = 0;
    for (int l = tid; l < nlev; l += nthr) my_nan |= s_lev[l].pad;
    // B of level l: Bbase[l * Bstride] (the staged block, or the workspace block when every thread has its own bin)
    const double *Bbase = BDIRECT ? (const double *)(P.ws_B + ((size_t)col * P.tiles + tile) * L.b_bytes) + bl
                                  : (const double *)(smem + L.off_Bt[buf]) + bl;
    feed.lv0 = s_lev;

    if (warp_on) {
      const double mu = s_dm[N];
      const bool day = mu > 0.0;
      const double muF = day ? mu * fstar_b : 0.0;            // mu * F_star[b]
      const double inv_mu = day ? 1.0 / mu : 0.0;

      // back-substitution state per interface i = 0..N: F_up[i] = c F_up[i-1] + d (weight folded into d) and R with
      // F_dn[i] = R F_up[i] + U.  U itself is not kept: sum_points W (U + beam) is reduced on the way down.
      double R[PPT], U[PPT], Fb[PPT], Ct[PPT], Dt[PPT];
#pragma unroll
      for (int q = 0; q < PPT; ++q) {
        R[q] = 0.0; U[q] = P.f_toa;      // F_dn[N] = f_toa (Fig. 5)
        Fb[q] = muF;                     // beam at the TOA (full strength, L235)
        Ct[q] = 1.0; Dt[q] = 0.0;        // TOA mode: F_up[N] = Ct F_up[j] + Dt
      }

      // bookkeeping of interface i with (U, Fb) at that interface: stage W (U + beam) for the transposed sum
      auto push_stage = [&](int i) {
        if (!TOA) {
          double su = 0.0, sb = 0.0;
#pragma unroll
          for (int q = 0; q < PPT; ++q) { su = fma(W[q], U[q] + Fb[q], su); sb = fma(W[q], Fb[q], sb); }
          stage_wr[(i & 7) * STAGE_LD] = su;
          if ((i & 7) == 0) flush_stage(stage_w, red_w + 2 * LP + i, lane);
          if (want_beam) {
            const double wb = warp_sum(sb);
            if (lane == 0) red_w[3 * LP + i] = wb;
          }
        }
      };
      // row i of the workspace: (c_i, W d_i) and R_{i-1}, the R just updated by the layer below interface i
      int srow_i = N;     // row N: the first one sweep 1 writes
      auto keep = [&](const double (&c)[PPT], const double (&wd)[PPT], const double (&Rlow)[PPT]) {
        if (TOA) return;
        stk_store<PPT>(stk_w + (size_t)(srow_i--) * SROW, lane, c, wd, Rlow);   // (a running pointer measured 1 % slower)
      };

      // ---------------- sweep 1: TOA -> BOA (one instantiation per day / night: the loop body has no branch) ------
      auto sweep1 = [&](auto day_tag) {
        constexpr bool DAY = decltype(day_tag)::value;
        double tau[PPT];
#pragma unroll
        for (int q = 0; q < PPT; ++q) tau[q] = 0.0;
        if constexpr (!NONISO) {
          const LevelRec *lv = s_lev + (N - 1);
          const double *Bp = Bbase + (size_t)(N - 1) * nbtS;
          feed.prime(lv, N);
          HRT_UNROLL(HRT_UNROLL_ISO)
          for (int j = N - 1; j >= 0; --j, --lv, Bp -= nbtS) {
            const RowsT<PPT> *cur = feed.next();
            push_stage(j + 1);
            // S3 + Eqs. 17-18 for the group: shared corner weights and bin constants
            const double2 ca = *reinterpret_cast<const double2 *>(&lv->c00);
            const double2 cb = *reinterpret_cast<const double2 *>(&lv->c10);
            const BinOpt *bo = lv->cloud ? bin1 : bin0;
            const double2 sbss = *reinterpret_cast<const double2 *>(&bo->sb);
            const G0Terms gt = bo->gt;
            const double dm = lv->dm, Bj = *Bp;
            double lk[PPT];
#pragma unroll
            for (int q = 0; q < PPT; ++q)
              lk[q] = fma(cb.y, cur[0].v[3][q], fma(cb.x, cur[0].v[2][q], fma(ca.y, cur[0].v[1][q], ca.x * cur[0].v[0][q])));
            feed.release(lv - 1, lv - RING, j - RING >= 0);
            double cc[PPT], wd[PPT];
#pragma unroll
            for (int q = 0; q < PPT; ++q) {
              const double kx = exp_hot<0, false>(lk[q], T32, nullptr) + sbss.x;
              const double w0 = sbss.y * rcp_fast(kx);
              const double dtau = kx * dm;
              double Fa = 0.0;
              if (DAY) {
                tau[q] += dtau;
                Fa = muF * exp_hot<1, false>(cap_pos<0x40862000>(tau[q] * inv_mu), T32, nullptr);   // (B6)
              }
              double c, d;
              layer_forward<DAY, false>(P, T32, w0, gt, dtau, Bj, Bj, mu, Fa, Fb[q], R[q], U[q], c, d);
              Fb[q] = Fa;
              if (TOA) {
                Dt[q] = fma(Ct[q], d, Dt[q]);
                Ct[q] *= c;
              }
              cc[q] = c;
              wd[q] = W[q] * d;
            }
            keep(cc, wd, R);
          }
        } else {
          // levels alternate interface (even) / centre (odd); sub-layer s lies between levels s and s+1 and takes
          // the arithmetic mean of the two levels' kappa_ext, omega0, g0 (L171, reading R10).  The centre unknowns
          // are eliminated on the fly: F_up[j+1] = cu F_up[centre] + du, F_up[centre] = cl F_up[j] + dl.
          const LevelRec *lv = s_lev + (nlev - 1);
          const double *Bp = Bbase + (size_t)(nlev - 1) * nbtS;
          auto optics = [&](const RowsT<PPT> &rw, const LevelRec *l, double (&kx)[PPT], double (&w0)[PPT], double &g0) {
            const double2 ca = *reinterpret_cast<const double2 *>(&l->c00);
            const double2 cb = *reinterpret_cast<const double2 *>(&l->c10);
            const BinOpt *bo = l->cloud ? bin1 : bin0;
            const double2 sbss = *reinterpret_cast<const double2 *>(&bo->sb);
            g0 = bo->gt.g0;
#pragma unroll
            for (int q = 0; q < PPT; ++q) {
              const double lk = fma(cb.y, rw.v[3][q], fma(cb.x, rw.v[2][q], fma(ca.y, rw.v[1][q], ca.x * rw.v[0][q])));
              kx[q] = exp_hot<0, false>(lk, T32, nullptr) + sbss.x;
              w0[q] = sbss.y * rcp_fast(kx[q]);
            }
          };
          double kx_up[PPT], w0_up[PPT], g0_up;
          {
            RowsT<PPT> top;
            load_rows_g<PPT>(top, P.lnk + pt, lv);
            optics(top, lv, kx_up, w0_up, g0_up);
          }
          double B_up = *Bp;
          feed.prime(lv - 1, N);
#pragma unroll 1
          for (int j = N - 1; j >= 0; --j, lv -= 2, Bp -= 2 * nbtS) {
            const RowsT<PPT> *cur = feed.next();      // [0] centre (lv - 1), [1] lower interface (lv - 2)
            push_stage(j + 1);
            double kx_c[PPT], w0_c[PPT], g0_c, kx_lo[PPT], w0_lo[PPT], g0_lo;
            optics(cur[0], lv - 1, kx_c, w0_c, g0_c);
            optics(cur[1], lv - 2, kx_lo, w0_lo, g0_lo);
            feed.release(lv - 3, lv - 1 - 2 * RING, j - RING >= 0);
            const double B_c = Bp[-nbtS], B_lo = Bp[-2 * nbtS];
            const double dm_u = lv[-1].dm, dm_l = lv[-2].dm;
            const G0Terms gt_u = g0_terms(0.5 * (g0_c + g0_up), P.inv_eps2), gt_l = g0_terms(0.5 * (g0_lo + g0_c), P.inv_eps2);
            double cc[PPT], wd[PPT];
#pragma unroll
            for (int q = 0; q < PPT; ++q) {
              const double dtau_u = 0.5 * (kx_c[q] + kx_up[q]) * dm_u;
              const double dtau_l = 0.5 * (kx_lo[q] + kx_c[q]) * dm_l;
              double Fc = 0.0, Fa = 0.0;
              if (DAY) {
                const double tau_c = tau[q] + dtau_u;
                tau[q] = tau_c + dtau_l;
                Fc = muF * exp_hot<1, false>(cap_pos<0x40862000>(tau_c * inv_mu), T32, nullptr);   // (B6)
                Fa = muF * exp_hot<1, false>(cap_pos<0x40862000>(tau[q] * inv_mu), T32, nullptr);
              }
              double cu, du, cl, dl;
              layer_forward<DAY, true>(P, T32, 0.5 * (w0_c[q] + w0_up[q]), gt_u, dtau_u, B_c, B_up, mu, Fc, Fb[q],
                                       R[q], U[q], cu, du);
              layer_forward<DAY, true>(P, T32, 0.5 * (w0_lo[q] + w0_c[q]), gt_l, dtau_l, B_lo, B_c, mu, Fa, Fc,
                                       R[q], U[q], cl, dl);
              Fb[q] = Fa;
              kx_up[q] = kx_lo[q]; w0_up[q] = w0_lo[q];
              const double c2 = cu * cl, d2 = fma(cu, dl, du);
              if (TOA) {
                Dt[q] = fma(Ct[q], d2, Dt[q]);
                Ct[q] *= c2;
              }
              cc[q] = c2;
              wd[q] = W[q] * d2;
            }
            g0_up = g0_lo; B_up = B_lo;
            keep(cc, wd, R);
          }
        }
      };
      if (day) sweep1(std::true_type{}); else sweep1(std::false_type{});

      // ---------------- BOA, Eq.(10) L237 ----------------
      const double F_boa = Bbase[(size_t)nlev * nbtS];
      double Fup0[PPT];
#pragma unroll
      for (int q = 0; q < PPT; ++q) Fup0[q] = (U[q] + F_boa + Fb[q]) * rcp_fast(1.0 - R[q]);

      if (TOA) {
        // S7 (spectrum shape): F_up_toa_bin[b] = sum_g w_g F_up[N]
#pragma unroll
        for (int q = 0; q < PPT; ++q) s_vals[PPT * tid + q] = active ? P.gauss_w[gidx + q] * fma(Ct[q], Fup0[q], Dt[q]) : 0.0;
      } else {
        push_stage(0);
        {
          double c0[PPT], wd0[PPT];
#pragma unroll
          for (int q = 0; q < PPT; ++q) { c0[q] = 0.0; wd0[q] = W[q] * Fup0[q]; }
          keep(c0, wd0, R);
        }
        // ---------------- sweep 2: back-substitution Eq.(15) + S7 reduction, 8 interfaces at a time ----------------
        double wF[PPT];
#pragma unroll
        for (int q = 0; q < PPT; ++q) wF[q] = 0.0;
        // The coefficients come back from L2 (several hundred cycles): the 8 interfaces of a group are loaded at once
        // (immediate offsets from one row pointer), then used.  Whole groups need no test; the last group (1..8
        // interfaces, R_N = 0) tests per interface, uniformly, and repeats F_up[N] into rows of the reduction buffer
        // that are never read.  (Measured and rejected: a two-buffer prefetch of the next group,
        // a butterfly instead of the staged transposes.)
        const double *row = stk_w;
        auto group = [&](auto full_tag, int base) {
          constexpr bool FULL = decltype(full_tag)::value;
          const int nk = N + 1 - base;          // interfaces left (FULL: > 8)
          double gc[8][PPT], gwd[8][PPT], gR[8][PPT], sd[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            if (FULL || k < nk) stk_load_cw<PPT>(row + k * SROW, lane, gc[k], gwd[k]);
            else {
#pragma unroll
              for (int q = 0; q < PPT; ++q) { gc[k][q] = 1.0; gwd[k][q] = 0.0; }
            }
            if (FULL || k < nk - 1) stk_load_R<PPT>(row + (k + 1) * SROW, lane, gR[k]);
            else {
#pragma unroll
              for (int q = 0; q < PPT; ++q) gR[k][q] = 0.0;
            }
          }
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            double su = 0.0, s2 = 0.0;
#pragma unroll
            for (int q = 0; q < PPT; ++q) {
              wF[q] = fma(gc[k][q], wF[q], gwd[k][q]);
              su += wF[q];
              s2 = fma(gR[k][q], wF[q], s2);
            }
            stage_wr[k * STAGE_LD] = su;
            sd[k] = s2;
          }
          flush_stage(stage_w, red_w + base, lane);
#pragma unroll
          for (int k = 0; k < 8; ++k) stage_wr[k * STAGE_LD] = sd[k];
          flush_stage(stage_w, red_w + LP + base, lane);
          // rows base .. base+7 are dead (the R part of row base+8 is not: next group's discard): drop their lines from
          // L2 instead of writing them back
          const int n_lines = (FULL ? 8 : nk) * (SROW / 16);
          for (int ln = lane; ln < n_lines; ln += 32) l2_discard(row + ln * 16);
        };
        int base = 0;
#pragma unroll 1
        for (; base + 8 <= N; base += 8, row += 8 * SROW) group(std::true_type{}, base);
        group(std::false_type{}, base);
        if (P.F_toa_bin != nullptr) {
#pragma unroll
          for (int q = 0; q < PPT; ++q) s_vals[PPT * tid + q] = active ? wF[q] * P.bins[b].inv_dlam : 0.0;
        }
      }
    } else if (TOA || P.F_toa_bin != nullptr) {
#pragma unroll
      for (int q = 0; q < PPT; ++q) s_vals[PPT * tid + q] = 0.0;
    }
    const int col_nan = __syncthreads_or(my_nan | (s_dm[N] != s_dm[N]));

    if (TOA || P.F_toa_bin != nullptr) {
      for (int k = tid; k < nbt; k += nthr) {
        const int bb = b_first + k;
        int g_lo = bb * P.ng - pt0, g_hi = g_lo + P.ng;
        // a bin may straddle two tiles: every tile adds its own part
        const bool whole = (g_lo >= 0) && (g_hi <= TP);
        if (g_lo < 0) g_lo = 0;
        if (g_hi > TP) g_hi = TP;
        double sum = col_nan ? nan("") : 0.0;
        for (int q = g_lo; q < g_hi; ++q) sum += s_vals[q];
        double *dst = P.F_toa_bin + (size_t)col * P.nb + bb;
        if (whole) *dst = sum; else atomicAdd(dst, sum);
      }
    }
    if (!TOA) column_epilogue(P, L, smem, s_dm, &s_is_last, nwa, want_beam, col, tile, col_nan);
    __syncthreads();                       // this column's shared-memory state, record buffer included, is dead
  }

  // the last block of the grid to run out of work re-arms the queues and the publication counts for the next launch
  if (tid == 0) {
    const unsigned total = gridDim.x * gridDim.y;
    s_is_last = (atomicAdd(P.queue + P.tiles, 1u) == total - 1);
  }
  __syncthreads();
  if (s_is_last) {
    for (int c = tid; c < P.ncol; c += nthr) P.flags[c] = 0;
    for (int t = tid; t <= P.tiles + 1; t += nthr) P.queue[t] = 0;
  }
}

// --------------------------------------------------------------------------------------------
// rt_iter_kernel: the scheme Thomas's algorithm replaces (L258-270, L397), as a measured
// comparison.  Same S1-S5 code as rt_step_kernel (one point per thread, one block per (tile, column)); instead of the
// forward elimination the (t, r, S_up, S_dn) of every system layer go to thread-private arrays, and the flux arrays
// are swept n_iter times: upward pass Eq.(10) + Eq.(2) with the previous downward fluxes, downward pass Eq.(3) with
// the upward fluxes just computed; all diffuse fluxes start at 0 (reading R23).  The non-isothermal system keeps its
// centre levels as unknowns (2N system layers, L311-313).  S7 as in the Thomas path (column_epilogue).
// --------------------------------------------------------------------------------------------
template <bool NONISO>
__global__ void __launch_bounds__(128) rt_iter_kernel(const KParams P, const int n_iter) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ double s_T32[32];
  __shared__ int s_is_last;
  constexpr int MAXS = NONISO ? 2 * MAXL : MAXL;   // system layers
  const int N = P.N, nlev = P.nlev;
  const int tid = threadIdx.x, nthr = blockDim.x, nwarps = nthr >> 5;
  const Lay L = make_lay(N, nlev, nwarps, 1, P.ng, P.nb, false, NONISO ? 2 : 1, 0, false);
  const LevelRec *s_lev = (const LevelRec *)(smem + L.off_rec[0]) + 1;
  const double *s_B = (const double *)(smem + L.off_Bt[0]);
  BinOpt *s_bin = (BinOpt *)(smem + L.off_bin);
  double *s_red = (double *)(smem + L.off_red);

  const int tile = blockIdx.x, col = blockIdx.y;
  const int LP = L.LP, nbtS = L.nbt;
  const double mu = P.mu[col];
  const bool day = mu > 0.0;
  const int pt0 = tile * nthr;
  const int b_first = pt0 / P.ng;
  int pt_last = pt0 + nthr - 1;
  if (pt_last > P.npt - 1) pt_last = P.npt - 1;
  const int nbt = pt_last / P.ng - b_first + 1;
  const int nwa = ((pt_last - pt0) >> 5) + 1;
  if (tid < 32) s_T32[tid] = kExp2Tab[tid];
  for (int i = tid; i < 2 * nbt; i += nthr) {
    const int cl = i / nbt, k = i - cl * nbt;
    const BinConst bc = P.bins[b_first + k];
    BinOpt bo;
    bo.sb = bc.sb[cl]; bo.ss = bc.ss[cl]; bo.gt = g0_terms(bc.gg[cl], P.inv_eps2); bo.pad[0] = bo.pad[1] = 0.0;
    s_bin[cl * nbtS + k] = bo;
  }
  // S1 / S2 blocks of the column from the workspace (written by rt_prep_kernel, the launch before this one)
  {
    const double *src = (const double *)(P.ws_rec + (size_t)col * L.rec_bytes);
    double *dst = (double *)(smem + L.off_rec[0]);
    for (int i = tid; i < (int)(L.rec_bytes / 8); i += nthr) dst[i] = src[i];
    src = (const double *)(P.ws_B + ((size_t)col * P.tiles + tile) * L.b_bytes);
    dst = (double *)(smem + L.off_Bt[0]);
    for (int i = tid; i < (int)(L.b_bytes / 8); i += nthr) dst[i] = src[i];
  }
  __syncthreads();
  const double *s_dm = (const double *)(smem + L.off_rec[0] + sizeof(LevelRec) * (nlev + 1));
  int col_nan = (mu != mu) ? 1 : 0;
  for (int l = 0; l < nlev; ++l) col_nan |= s_lev[l].pad;

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

    auto optics = [&](const LevelRec *lv, double &kx, double &w0, double &g0) {
      RowsT<1> rw;
      load_rows_g<1>(rw, lnk_pt, lv);
      const double2 ca = *reinterpret_cast<const double2 *>(&lv->c00);
      const double2 cb = *reinterpret_cast<const double2 *>(&lv->c10);
      const double lk = fma(cb.y, rw.v[3][0], fma(cb.x, rw.v[2][0], fma(ca.y, rw.v[1][0], ca.x * rw.v[0][0])));
      const BinOpt *bo = lv->cloud ? bin1 : bin0;
      kx = exp_hot<0, false>(lk, T32, nullptr) + bo->sb;
      w0 = bo->ss * rcp_fast(kx);
      g0 = bo->gt.g0;
    };

    // ---- S3-S5 per system layer, TOA -> BOA (tau and the beam are running prefixes) ----
    auto coeffs = [&](auto day_tag) {
      constexpr bool DAY = decltype(day_tag)::value;
      double tau = 0.0, Fb = muF;
      bm[LS] = Fb;
      if (!NONISO) {
        for (int j = N - 1; j >= 0; --j) {
          const LevelRec *lv = s_lev + j;
          double kx, w0, g0;
          optics(lv, kx, w0, g0);
          const double dtau = kx * lv->dm;
          const double Bj = s_B[(size_t)j * nbtS + bl];
          double Fa = 0.0;
          if (DAY) {
            tau += dtau;
            Fa = muF * exp_hot<1, false>(cap_pos<0x40862000>(tau * inv_mu), T32, nullptr);
          }
          layer_coeffs<DAY, false>(P, T32, w0, g0_terms(g0, P.inv_eps2), dtau, Bj, Bj, mu, Fa, Fb, a_t[j], a_r[j], a_su[j], a_sd[j]);
          bm[j] = Fa;
          Fb = Fa;
        }
      } else {
        double kx_up, w0_up, g0_up;
        optics(s_lev + LS, kx_up, w0_up, g0_up);
        double B_up = s_B[(size_t)LS * nbtS + bl];
        for (int sl = LS - 1; sl >= 0; --sl) {
          const LevelRec *lv = s_lev + sl;
          double kx_lo, w0_lo, g0_lo;
          optics(lv, kx_lo, w0_lo, g0_lo);
          const double B_lo = s_B[(size_t)sl * nbtS + bl];
          const double dtau = 0.5 * (kx_lo + kx_up) * lv->dm;
          double Fa = 0.0;
          if (DAY) {
            tau += dtau;
            Fa = muF * exp_hot<1, false>(cap_pos<0x40862000>(tau * inv_mu), T32, nullptr);
          }
          layer_coeffs<DAY, true>(P, T32, 0.5 * (w0_lo + w0_up), g0_terms(0.5 * (g0_lo + g0_up), P.inv_eps2), dtau, B_lo, B_up,
                                  mu, Fa, Fb, a_t[sl], a_r[sl], a_su[sl], a_sd[sl]);
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
  column_epilogue(P, L, smem, s_dm, &s_is_last, nwa, P.F_beam != nullptr, col, tile, col_nan);
}

// phase A as a launch of its own: for the comparison path (rt_iter_kernel; tp = spectral points per tile of that kernel,
// count = 0) and for rt_step_kernel when the device cannot host its grid at once (count = 1)
template <bool NONISO>
__global__ void __launch_bounds__(128) rt_prep_kernel(const KParams P, const int tp, const int count, const int bdirect) {
  __shared__ double s_T32[32];
  // only the block sizes of the layout are used here
  const Lay L = make_lay(P.N, P.nlev, tp / 32, 1, P.ng, P.nb, true, NONISO ? 2 : 1, 0, bdirect != 0);
  if (threadIdx.x < 32) s_T32[threadIdx.x] = kExp2Tab[threadIdx.x];
  __syncthreads();
  phase_a<NONISO, true, true>(P, L, s_T32, (long)blockIdx.x * blockDim.x + threadIdx.x, (long)gridDim.x * blockDim.x, count != 0);
}

__global__ void zero_kernel(double *p, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    p[i] = 0.0;
}

// --------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------
typedef void (*kernel_fn)(const KParams);

struct Variant {
  bool noniso, toa, bdirect;
  int ppt, rows, warps;   // warps: block size compiled in, 0 = any
  int maxt, minb;      // launch bounds: register cap = 65536 / (maxt * minb)
  kernel_fn fn;
};

#define HRT_K(NI, TOA, PPT, ROWS, WARPS, MAXT, MINB) \
  {NI, TOA, false, PPT, ROWS, WARPS, MAXT, MINB, rt_step_kernel<NI, TOA, PPT, ROWS, false, WARPS, MAXT, MINB>}
// one Gauss point per bin (opacity sampling): Planck values read from the workspace; one point per thread
#define HRT_KB(NI, TOA, ROWS, WARPS, MAXT, MINB) \
  {NI, TOA, true, 1, ROWS, WARPS, MAXT, MINB, rt_step_kernel<NI, TOA, 1, ROWS, true, WARPS, MAXT, MINB>}

// Compiled instantiations, in order of preference for each (noniso, toa, ppt).  helios_rt_create takes the first
// match; helios_rt_debug_set_launch (tests, tuning) may select any other.
const Variant kVariants[] = {
#include "helios_rt_variants.inc"
};
constexpr int kNumVariants = (int)(sizeof(kVariants) / sizeof(kVariants[0]));

typedef void (*iter_fn)(const KParams, const int);

// spectral points per thread: isothermal columns whose number of Gauss points is a multiple of it, with enough points
// to fill the tiles.  2 with the back-substitution pass, 4 in TOA mode.
int default_ppt(int npt, int ng, bool noniso, bool toa) {
  const bool can2 = !noniso && ng > 1 && (ng % 2) == 0, can4 = can2 && toa && (ng % 4) == 0;
  if (npt < 256) return 1;
  return can4 ? 4 : (can2 ? 2 : 1);
}

// warps per block: tiles of 128 spectral points for long columns; small columns take the
// block with the fewest padded lanes, ties -> larger block (fewer tiles)
int default_warps(int npt, int ppt, bool noniso) {
  if (npt >= 256) return noniso ? 4 : (ppt == 4 ? 1 : (ppt == 2 ? 2 : 4));
  int best = 1;
  long best_waste = -1;
  for (int w = 1; w <= 4; ++w) {
    const long tp = 32L * w * ppt, tiles = (npt + tp - 1) / tp;
    const long waste = tiles * tp - npt;
    if (best_waste < 0 || waste < best_waste || (waste == best_waste && w > best)) { best = w; best_waste = waste; }
  }
  return best;
}

}  // namespace

struct helios_rt {
  helios_rt_config cfg;   // pointers nulled
  int npt, nlev;
  bool noniso, toa;
  // launch shape of rt_step_kernel
  int variant, warps, ppt, tiles, workers, occ;
  Lay lay;
  int iter_warps, iter_tiles;      // rt_iter_kernel keeps one point per thread
  unsigned row_stride;
  double inv_dlp, inv_dt;
  // device tables
  double *d_lnk, *d_tab_lp, *d_tab_t, *d_edges, *d_gw, *d_gtab, *d_c2lam;
  BinConst *d_bins;
  // workspace
  double *d_stack, *d_partial;
  unsigned char *d_ws_rec, *d_ws_B;
  size_t stack_block, stack_bytes, partial_bytes, ws_bytes;
  unsigned *d_counter, *d_queue, *d_flags;
  BinSlot *d_bslot, *d_bslot_iter;
  int *d_slot_ptr, *d_slots, *d_slot_ptr_iter, *d_slots_iter;   // bin -> Planck-block slots (step tiling / comparison tiling)
  unsigned epoch;
  Lay iter_lay;
  double *inv_dlam;          // host copy, [n_bins]
  // device + pinned host staging for step_host
  double *d_in, *d_out, *h_in, *h_out;
  cudaStream_t own_stream, copy_stream;
  cudaEvent_t ev_in[4], ev_done[4];
  int regs, lmem, sm_count;
  int force_two_launches;   // helios_rt_debug_force_two_launches: always take the fallback path (tests)
  cudaError_t last_err;
};

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
  if ((long long)c->n_ktab_p * c->n_ktab_t * ((long long)c->n_bins * c->n_gauss + 2) >= (1LL << 31)) return HELIOS_RT_EINVAL;   // 32-bit table offsets
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
  // kappa in [1e-300, 1e300]: |ln kappa| <= 691 stays inside the domain of the table exp (|x| <= 708)
  const size_t nk = (size_t)c->n_ktab_p * c->n_ktab_t * c->n_bins * c->n_gauss;
  for (size_t i = 0; i < nk; ++i) if (!(c->ktab[i] >= 1e-300) || !(c->ktab[i] <= 1e300)) return HELIOS_RT_EINVAL;
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
  cudaFree(h->d_gtab); cudaFree(h->d_c2lam); cudaFree(h->d_bins); cudaFree(h->d_partial); cudaFree(h->d_counter); cudaFree(h->d_queue);
  cudaFree(h->d_stack); cudaFree(h->d_in); cudaFree(h->d_out);
  cudaFree(h->d_ws_rec); cudaFree(h->d_ws_B); cudaFree(h->d_flags);
  cudaFree(h->d_slot_ptr); cudaFree(h->d_slots); cudaFree(h->d_slot_ptr_iter); cudaFree(h->d_slots_iter);
  cudaFree(h->d_bslot); cudaFree(h->d_bslot_iter);
  free(h->inv_dlam);
  if (h->h_in) cudaFreeHost(h->h_in);
  if (h->h_out) cudaFreeHost(h->h_out);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  for (int i = 0; i < 4; ++i) {
    if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
    if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
  }
  delete h;
  return HELIOS_RT_OK;
}

// bin -> slots of the per-(column, tile) Planck blocks: bin b is stored once in the block of every tile that owns
// points of it, at row offset (b - first bin of the tile)
static int build_slots(helios_rt *h, int tp, const Lay &lay, const double *inv_dlam, int **d_ptr, int **d_slots,
                       BinSlot **d_bslot) {
  const int nb = h->cfg.n_bins, ng = h->cfg.n_gauss;
  int *ptr = (int *)malloc(sizeof(int) * (nb + 1));
  int total = 0;
  if (!ptr) return HELIOS_RT_ENOMEM;
  for (int b = 0; b < nb; ++b) { ptr[b] = total; total += ((b + 1) * ng - 1) / tp - (b * ng) / tp + 1; }
  ptr[nb] = total;
  int *sl = (int *)malloc(sizeof(int) * (total > 0 ? total : 1));
  if (!sl) { free(ptr); return HELIOS_RT_ENOMEM; }
  for (int b = 0, k = 0; b < nb; ++b)
    for (int t = (b * ng) / tp; t <= ((b + 1) * ng - 1) / tp; ++t) sl[k++] = t * (int)(lay.b_bytes / 8) + (b - (t * tp) / ng);
  BinSlot *bs = (BinSlot *)malloc(sizeof(BinSlot) * nb);
  if (!bs) { free(ptr); free(sl); return HELIOS_RT_ENOMEM; }
  for (int b = 0; b < nb; ++b) {
    const int n = ptr[b + 1] - ptr[b];
    bs[b].s0 = sl[ptr[b]];
    bs[b].s1 = n == 1 ? -1 : (n == 2 ? sl[ptr[b] + 1] : -2);
    bs[b].inv_dlam = inv_dlam[b];
  }
  cudaError_t e = cudaMalloc((void **)d_ptr, sizeof(int) * (nb + 1));
  if (e == cudaSuccess) e = cudaMemcpy(*d_ptr, ptr, sizeof(int) * (nb + 1), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMalloc((void **)d_bslot, sizeof(BinSlot) * nb);
  if (e == cudaSuccess) e = cudaMemcpy(*d_bslot, bs, sizeof(BinSlot) * nb, cudaMemcpyHostToDevice);
  free(bs);
  if (e == cudaSuccess) e = cudaMalloc((void **)d_slots, sizeof(int) * (total > 0 ? total : 1));
  if (e == cudaSuccess) e = cudaMemcpy(*d_slots, sl, sizeof(int) * (total > 0 ? total : 1), cudaMemcpyHostToDevice);
  free(ptr); free(sl);
  if (e != cudaSuccess) { h->last_err = e; return e == cudaErrorMemoryAllocation ? HELIOS_RT_ENOMEM : HELIOS_RT_ECUDA; }
  return HELIOS_RT_OK;
}

// launch shape + workspace for the chosen variant / warps per block.  Frees and re-allocates the workspace whose size
// depends on the shape; called by create and by helios_rt_debug_set_launch.
static int configure_launch(helios_rt *h) {
  const helios_rt_config &c = h->cfg;
  const Variant &v = kVariants[h->variant];
  const int N = c.n_layers;
  h->ppt = v.ppt;
  if (h->warps * 32 > v.maxt || (v.warps != 0 && v.warps != h->warps)) return HELIOS_RT_EINVAL;
  const int tp = h->warps * 32 * h->ppt;
  h->tiles = (h->npt + tp - 1) / tp;
  h->lay = make_lay(N, h->nlev, h->warps, h->ppt, c.n_gauss, c.n_bins, h->toa, h->noniso ? 2 : 1, v.rows, v.bdirect);
  h->iter_lay = make_lay(N, h->nlev, h->iter_warps, 1, c.n_gauss, c.n_bins, false, h->noniso ? 2 : 1, 0, false);
  if (h->lay.total > 227u * 1024u) return HELIOS_RT_EINVAL;
  CK(h, cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->lay.total));
  cudaFuncAttributes fa;
  CK(h, cudaFuncGetAttributes(&fa, v.fn));
  h->regs = fa.numRegs;
  h->lmem = (int)fa.localSizeBytes;
  CK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ, v.fn, h->warps * 32, h->lay.total));
  if (h->occ < 1) return HELIOS_RT_EINVAL;
  // persistent grid: as many blocks as are resident at once, split evenly over the tiles; never more workers per
  // tile than columns
  long workers = (long)h->sm_count * h->occ / h->tiles;
  if (workers < 1) workers = 1;
  if (workers > c.max_columns) workers = c.max_columns;
  h->workers = (int)workers;
  // workspace
  cudaFree(h->d_stack); h->d_stack = nullptr;
  cudaFree(h->d_partial); h->d_partial = nullptr;
  cudaFree(h->d_queue); h->d_queue = nullptr;
  cudaFree(h->d_ws_rec); h->d_ws_rec = nullptr;
  cudaFree(h->d_ws_B); h->d_ws_B = nullptr;
  {
    // S1/S2 blocks of every column: sized for the step kernel's tiling and for the comparison kernel's
    size_t bB = (size_t)h->tiles * h->lay.b_bytes;
    if (!h->toa && (size_t)h->iter_tiles * h->iter_lay.b_bytes > bB) bB = (size_t)h->iter_tiles * h->iter_lay.b_bytes;
    const size_t bR = h->lay.rec_bytes;   // the same for both (depends on N and nlev only)
    h->ws_bytes = (size_t)c.max_columns * (bB + bR);
    CK(h, cudaMalloc((void **)&h->d_ws_rec, (size_t)c.max_columns * bR));
    CK(h, cudaMalloc((void **)&h->d_ws_B, (size_t)c.max_columns * bB));
  }
  cudaFree(h->d_slot_ptr); h->d_slot_ptr = nullptr;
  cudaFree(h->d_slots); h->d_slots = nullptr;
  cudaFree(h->d_slot_ptr_iter); h->d_slot_ptr_iter = nullptr;
  cudaFree(h->d_slots_iter); h->d_slots_iter = nullptr;
  cudaFree(h->d_bslot); h->d_bslot = nullptr;
  cudaFree(h->d_bslot_iter); h->d_bslot_iter = nullptr;
  {
    int rc = build_slots(h, tp, h->lay, h->inv_dlam, &h->d_slot_ptr, &h->d_slots, &h->d_bslot);
    if (rc == HELIOS_RT_OK && !h->toa)
      rc = build_slots(h, h->iter_warps * 32, h->iter_lay, h->inv_dlam, &h->d_slot_ptr_iter, &h->d_slots_iter, &h->d_bslot_iter);
    if (rc) return rc;
  }
  // back-substitution workspace: per block [warp][N + 1 rows][96 ppt]
  h->stack_block = (size_t)(N + 1) * h->warps * 96 * h->ppt;
  h->stack_bytes = !h->toa ? sizeof(double) * h->stack_block * h->tiles * h->workers : 0;
  if (h->stack_bytes) CK(h, cudaMalloc((void **)&h->d_stack, h->stack_bytes));
  const int mt = h->tiles > h->iter_tiles ? h->tiles : h->iter_tiles;
  h->partial_bytes = sizeof(double) * (size_t)c.max_columns * mt * 4 * (N + 1);
  CK(h, cudaMalloc((void **)&h->d_partial, h->partial_bytes));
  CK(h, cudaMalloc((void **)&h->d_queue, sizeof(unsigned) * (h->tiles + 2)));
  CK(h, cudaMemset(h->d_queue, 0, sizeof(unsigned) * (h->tiles + 2)));
  return HELIOS_RT_OK;
}

// first instantiation of the class that matches; one compiled for exactly `warps` warps is preferred to a generic one
static int find_variant(bool noniso, bool toa, bool bdirect, int ppt, int rows, int stk, int maxt, int minb, int warps) {
  for (int pass = 0; pass < 2; ++pass)
  for (int i = 0; i < kNumVariants; ++i) {
    const Variant &v = kVariants[i];
    if (v.noniso != noniso || v.toa != toa || v.bdirect != bdirect || v.ppt != ppt) continue;
    if (pass == 0 ? v.warps != warps : v.warps != 0) continue;
    if (rows >= 0 && v.rows != rows) continue;
    if (stk == 0) continue;   // the thread-private stack of round 1 is gone
    if (maxt >= 0 && v.maxt != maxt) continue;
    if (minb >= 0 && v.minb != minb) continue;
    return i;
  }
  return -1;
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
  h->nlev = h->noniso ? 2 * N + 1 : N;
  h->iter_warps = default_warps(h->npt, 1, false);
  h->iter_tiles = (h->npt + h->iter_warps * 32 - 1) / (h->iter_warps * 32);
  int ppt = default_ppt(h->npt, ng, h->noniso, h->toa);
  h->warps = default_warps(h->npt, ppt, h->noniso);
  h->variant = find_variant(h->noniso, h->toa, ng == 1, ppt, -1, -1, -1, -1, h->warps);
  if (h->variant < 0) {
    ppt = 1;
    h->warps = default_warps(h->npt, 1, h->noniso);
    h->variant = find_variant(h->noniso, h->toa, ng == 1, 1, -1, -1, -1, -1, h->warps);
  }
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (h->variant < 0) { helios_rt_destroy(h); return HELIOS_RT_EINVAL; }

  // ln(kappa) table (rows padded to an even length, zero-filled, + a tail so that a warp's bulk copy of its 32 PPT
  // points never leaves the allocation), log10 pressure grid, per-bin constants, Planck polynomial pieces
  h->row_stride = (unsigned)((h->npt + 1) & ~1);
  const size_t nrows = (size_t)cfg->n_ktab_p * cfg->n_ktab_t;
  const size_t nk = nrows * h->row_stride + 256;
  double *lnk = (double *)calloc(nk, sizeof(double));
  double *lp = (double *)malloc(sizeof(double) * cfg->n_ktab_p);
  BinConst *bins = (BinConst *)malloc(sizeof(BinConst) * nb);
  double *gtab = (double *)malloc(sizeof(double) * kGIntervals * kGCoef);
  if (!lnk || !lp || !bins || !gtab) { free(lnk); free(lp); free(bins); free(gtab); helios_rt_destroy(h); return HELIOS_RT_ENOMEM; }
  for (size_t r = 0; r < nrows; ++r)
    for (int i = 0; i < h->npt; ++i) lnk[r * h->row_stride + i] = log(cfg->ktab[r * h->npt + i]);
  for (int i = 0; i < cfg->n_ktab_p; ++i) lp[i] = log10(cfg->ktab_p[i]);
  h->inv_dlp = (cfg->n_ktab_p - 1) / (lp[cfg->n_ktab_p - 1] - lp[0]);
  h->inv_dt = (cfg->n_ktab_t - 1) / (cfg->ktab_t[cfg->n_ktab_t - 1] - cfg->ktab_t[0]);
  for (int b = 0; b < nb; ++b) {
    // Eqs.(17)-(18) in per-mass units: sb = what is added to kappa_abs, ss = scattering part, gg = g0
    BinConst &bc = bins[b];
    bc.dlam = cfg->bin_edges[b + 1] - cfg->bin_edges[b];
    bc.inv_dlam = 1.0 / bc.dlam;
    const double sg = cfg->scat_gas[b], kc = cfg->cloud_ext[b], sc = cfg->cloud_w0[b] * kc;
    bc.sb[0] = sg;            bc.sb[1] = sg + kc;
    bc.ss[0] = sg;            bc.ss[1] = sg + sc;
    bc.gg[0] = 0.0;           bc.gg[1] = (sg + sc > 0.0) ? sc * cfg->cloud_g0[b] / (sg + sc) : 0.0;
    // omega0 = ss / (kappa_abs + sb) must stay below 1 after rounding (E - omega0 = 0 is the singular conservative limit,
    // SURVEY.md Q5): a purely scattering constituent is capped one ulp below its extinction
    for (int cl = 0; cl < 2; ++cl)
      if (bc.ss[cl] > bc.sb[cl] * (1.0 - 0x1p-52)) bc.ss[cl] = bc.sb[cl] * (1.0 - 0x1p-52);
  }
  build_planck_table(gtab);
  h->inv_dlam = (double *)malloc(sizeof(double) * nb);
  if (!h->inv_dlam) { free(lnk); free(lp); free(bins); free(gtab); helios_rt_destroy(h); return HELIOS_RT_ENOMEM; }
  for (int b = 0; b < nb; ++b) h->inv_dlam[b] = bins[b].inv_dlam;
  cudaError_t e = cudaSuccess;
  auto step = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  step(upload(&h->d_lnk, lnk, nk));
  step(upload(&h->d_tab_lp, lp, (size_t)cfg->n_ktab_p));
  step(upload(&h->d_tab_t, cfg->ktab_t, (size_t)cfg->n_ktab_t));
  step(upload(&h->d_edges, cfg->bin_edges, (size_t)nb + 1));
  step(upload(&h->d_gw, cfg->gauss_w, (size_t)ng));
  step(upload(&h->d_bins, bins, (size_t)nb));
  step(upload(&h->d_gtab, gtab, (size_t)kGIntervals * kGCoef));
  {
    double *c2l = (double *)malloc(sizeof(double) * (nb + 1));
    if (!c2l) step(cudaErrorMemoryAllocation);
    else {
      for (int i = 0; i <= nb; ++i) c2l[i] = kPlanckC2 / cfg->bin_edges[i];
      step(upload(&h->d_c2lam, c2l, (size_t)nb + 1));
      free(c2l);
    }
  }
  free(lnk); free(lp); free(bins); free(gtab);
  const size_t ncol = (size_t)cfg->max_columns;
  step(cudaMalloc((void **)&h->d_counter, sizeof(unsigned) * ncol));
  if (e == cudaSuccess) step(cudaMemset(h->d_counter, 0, sizeof(unsigned) * ncol));
  step(cudaMalloc((void **)&h->d_flags, sizeof(unsigned) * ncol));
  if (e == cudaSuccess) step(cudaMemset(h->d_flags, 0, sizeof(unsigned) * ncol));
  // step_host staging: inputs packed as [p | T | mu | F*], outputs as [F_up | F_down | F_net | F_beam | dTdt | toa]
  const size_t n_in = ncol * (2 * (size_t)N + 1) + nb, n_out = ncol * (4 * ((size_t)N + 1) + N + nb);
  step(cudaMalloc((void **)&h->d_in, sizeof(double) * n_in));
  step(cudaMalloc((void **)&h->d_out, sizeof(double) * n_out));
  step(cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking));
  step(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  for (int i = 0; i < 4; ++i) {
    step(cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming));
    step(cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming));
  }
  if (e == cudaSuccess) {
    iter_fn it = h->noniso ? rt_iter_kernel<true> : rt_iter_kernel<false>;
    if (!h->toa)
      step(cudaFuncSetAttribute(it, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)make_lay(N, h->nlev, h->iter_warps, 1, ng, nb, false, h->noniso ? 2 : 1, 0, false).total));
  }
  if (e != cudaSuccess) {
    const bool oom = (e == cudaErrorMemoryAllocation);
    helios_rt_destroy(h);
    cudaGetLastError();
    return oom ? HELIOS_RT_ENOMEM : HELIOS_RT_ECUDA;
  }
  rc = configure_launch(h);
  if (rc) {
    const bool oom = (h->last_err == cudaErrorMemoryAllocation);
    helios_rt_destroy(h);
    cudaGetLastError();
    return oom ? HELIOS_RT_ENOMEM : rc;
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

// col0: first column of a chunk (step_host pipelines chunks; helios_rt_step passes 0); the chunk's inputs and outputs
// start at column 0 of the given pointers
static int launch_step(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out, cudaStream_t st,
                       int n_iter = 0) {
  const helios_rt_config &c = h->cfg;
  if (in->n_columns == 0) return HELIOS_RT_OK;
  KParams P;
  P.lnk = h->d_lnk; P.tab_lp = h->d_tab_lp; P.tab_t = h->d_tab_t; P.edges = h->d_edges; P.gauss_w = h->d_gw;
  P.bins = h->d_bins; P.gtab = h->d_gtab; P.c2lam = h->d_c2lam;
  P.nP = c.n_ktab_p; P.nT = c.n_ktab_t; P.N = c.n_layers; P.nlev = h->nlev; P.nb = c.n_bins; P.ng = c.n_gauss; P.npt = h->npt;
  P.tiles = n_iter > 0 ? h->iter_tiles : h->tiles;
  P.ncol = in->n_columns;
  P.row_stride = h->row_stride; P.inv_dlp = h->inv_dlp; P.inv_dt = h->inv_dt;
  P.cloud_p_top = c.cloud_p_top; P.cloud_p_bot = c.cloud_p_bot; P.inv_g = 1.0 / c.gravity; P.inv_cp = 1.0 / c.cp;
  P.inv_eps2 = 1.0 / c.eps2; P.e_tau = c.e_tau; P.gcrit_tol = c.gcrit_tol; P.w0_transition = (c.flags & HELIOS_RT_IMPROVED) ? c.w0_transition : INFINITY;   // regular two-stream: E = 1
  P.f_toa = c.f_toa;
  P.p = in->p; P.T = in->T; P.mu = in->mu_star; P.fstar = in->stellar_flux;
  P.T_int = in->f_internal > 0 ? sqrt(sqrt(in->f_internal / kSigmaSB)) : 0.0;
  P.F_up = out->F_up; P.F_down = out->F_down; P.F_net = out->F_net; P.dTdt = out->dTdt; P.F_beam = out->F_beam;
  P.F_toa_bin = out->F_up_toa_bin;
  P.ws_rec = h->d_ws_rec; P.ws_B = h->d_ws_B; P.flags = h->d_flags;
  P.slot_ptr = h->d_slot_ptr; P.slots = h->d_slots; P.bslot = h->d_bslot;
  ++h->epoch;
  P.fused_prep = 0;
  P.stack = h->d_stack; P.stack_block = h->stack_block;
  P.partial = h->d_partial; P.counter = h->d_counter; P.queue = h->d_queue;
  if (n_iter > 0) {
    if (in->n_columns > 65535) return HELIOS_RT_EINVAL;   // the comparison kernel puts columns in gridDim.y
    iter_fn fn = h->noniso ? rt_iter_kernel<true> : rt_iter_kernel<false>;
    const Lay &lay = h->iter_lay;
    const long items = (long)in->n_columns * (h->nlev + 1);
    const int pblocks = (int)((items + 127) / 128 < 16L * h->sm_count ? (items + 127) / 128 : 16L * h->sm_count);
    P.slot_ptr = h->d_slot_ptr_iter; P.slots = h->d_slots_iter; P.bslot = h->d_bslot_iter;
    if (h->noniso) rt_prep_kernel<true><<<pblocks, 128, 0, st>>>(P, h->iter_warps * 32, 0, 0);
    else rt_prep_kernel<false><<<pblocks, 128, 0, st>>>(P, h->iter_warps * 32, 0, 0);
    CK(h, cudaGetLastError());
    dim3 grid((unsigned)h->iter_tiles, (unsigned)in->n_columns);
    fn<<<grid, h->iter_warps * 32, lay.total, st>>>(P, n_iter);
    CK(h, cudaGetLastError());
    return HELIOS_RT_OK;
  }
  // bins that straddle two tiles are accumulated with atomics: start from zero
  const int tp = h->warps * 32 * h->ppt;
  if (P.F_toa_bin && h->tiles > 1 && (tp % c.n_gauss) != 0) {
    const size_t n = (size_t)in->n_columns * c.n_bins;
    zero_kernel<<<(unsigned)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024), 256, 0, st>>>(P.F_toa_bin, n);
  }
  int workers = h->workers;
  if (workers > in->n_columns) workers = in->n_columns;
  // One cooperative launch: phase A (S1 + S2 of all columns, spread over the grid) and phase B (the sweeps) in the same
  // kernel; blocks of phase B wait on per-column publication flags, which is safe because the cooperative launch
  // guarantees that the whole grid is resident.  If the device cannot host the grid at once (another context's kernels
  // hold SMs), phase A runs as a launch of its own instead.
  cudaLaunchConfig_t lc;
  memset(&lc, 0, sizeof(lc));
  lc.gridDim = dim3((unsigned)h->tiles, (unsigned)workers);
  lc.blockDim = dim3((unsigned)(h->warps * 32));
  lc.dynamicSmemBytes = h->lay.total;
  lc.stream = st;
  cudaLaunchAttribute attr;
  attr.id = cudaLaunchAttributeCooperative;
  attr.val.cooperative = 1;
  lc.attrs = &attr;
  lc.numAttrs = 1;
  P.fused_prep = h->epoch == 1 ? 1 : 2;   // (2: a later launch of the handle; only diagnostic builds care)
#ifdef HRT_DIAG_NOCOOP         /* diagnostic builds (_work/): plain launch / phase A as its own launch */
  lc.numAttrs = 0;
#endif
#ifdef HRT_DIAG_TWO_LAUNCH
  cudaError_t e = cudaErrorNotSupported;
#else
  cudaError_t e = h->force_two_launches ? cudaErrorCooperativeLaunchTooLarge : cudaLaunchKernelEx(&lc, kVariants[h->variant].fn, P);
#endif
  if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorNotSupported) {
    cudaGetLastError();
    P.fused_prep = 0;
    const long items = (long)in->n_columns * (h->nlev + 1);
    const int pblocks = (int)((items + 127) / 128 < 16L * h->sm_count ? (items + 127) / 128 : 16L * h->sm_count);
    const int tp2 = h->warps * 32 * h->ppt;
    const int bd = kVariants[h->variant].bdirect ? 1 : 0;
    if (h->noniso) rt_prep_kernel<true><<<pblocks, 128, 0, st>>>(P, tp2, 1, bd);
    else rt_prep_kernel<false><<<pblocks, 128, 0, st>>>(P, tp2, 1, bd);
    CK(h, cudaGetLastError());
    lc.numAttrs = 0;
    e = cudaLaunchKernelEx(&lc, kVariants[h->variant].fn, P);
  }
  CK(h, e);
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

// device alias of a host pointer that the device can write directly (page-locked, mapped: cudaHostAlloc /
// cudaHostRegister memory under unified addressing); nullptr for pageable memory
static double *mapped_alias(double *host) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return a.type == cudaMemoryTypeHost ? (double *)a.devicePointer : nullptr;
}

extern "C" int helios_rt_step_host(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out) {
  int rc = validate_step(h, in, out);
  if (rc) return rc;
  if (in->n_columns == 0) return HELIOS_RT_OK;
  const size_t ncol = (size_t)in->n_columns, N = (size_t)h->cfg.n_layers, nb = (size_t)h->cfg.n_bins;
  cudaStream_t st = h->own_stream;
  double *d_p = h->d_in, *d_T = d_p + ncol * N, *d_mu = d_T + ncol * N, *d_fs = d_mu + ncol;
  CK(h, cudaMemcpyAsync(d_p, in->p, sizeof(double) * ncol * N, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(d_T, in->T, sizeof(double) * ncol * N, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(d_mu, in->mu_star, sizeof(double) * ncol, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(d_fs, in->stellar_flux, sizeof(double) * nb, cudaMemcpyHostToDevice, st));
  helios_rt_inputs din = *in;
  din.p = d_p; din.T = d_T; din.mu_star = d_mu; din.stellar_flux = d_fs;
  // Outputs.  Page-locked, mapped host buffers are written by the kernel itself (each column's results leave over
  // PCIe as soon as its last tile has summed them, under the sweeps of the other columns); pageable buffers, and a
  // per-bin spectrum whose bins straddle tiles (accumulated with atomics), go through device staging and a copy each.
  const int tp = h->warps * 32 * h->ppt;
  const bool toa_atomics = h->tiles > 1 && (tp % h->cfg.n_gauss) != 0;
  double *const host[6] = {out->F_up, out->F_down, out->F_net, out->F_beam, out->dTdt, out->F_up_toa_bin};
  const size_t ni = ncol * (N + 1);
  const size_t count[6] = {ni, ni, ni, ni, ncol * N, ncol * nb};
  double *dev[6], *stage = h->d_out;
  bool staged[6];
  for (int k = 0; k < 6; ++k) {
    dev[k] = nullptr;
    staged[k] = false;
    if (host[k]) {
      double *alias = (k == 5 && toa_atomics) ? nullptr : mapped_alias(host[k]);
      dev[k] = alias ? alias : stage;
      staged[k] = alias == nullptr;
    }
    stage += count[k];
  }
  helios_rt_outputs dout;
  dout.F_up = dev[0]; dout.F_down = dev[1]; dout.F_net = dev[2]; dout.F_beam = dev[3]; dout.dTdt = dev[4];
  dout.F_up_toa_bin = dev[5];
  rc = launch_step(h, &din, &dout, st);
  if (rc) return rc;
  for (int k = 0; k < 6; ++k)
    if (staged[k]) CK(h, cudaMemcpyAsync(host[k], dev[k], sizeof(double) * count[k], cudaMemcpyDeviceToHost, st));
  CK(h, cudaStreamSynchronize(st));
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_launch_info(const helios_rt *h, int32_t info[8]) {
  if (!h || !info) return HELIOS_RT_EINVAL;
  info[0] = h->warps * 32; info[1] = h->tiles; info[2] = (int32_t)h->lay.total; info[3] = h->regs; info[4] = h->occ;
  info[5] = h->lmem;
  info[6] = 1;   // rt_step_kernel (+1 zero-fill launch when F_up_toa_bin bins straddle tiles)
  info[7] = h->sm_count;
  return HELIOS_RT_OK;
}

// ---- include/helios_rt_debug.h: not part of the product API ----
extern "C" int helios_rt_debug_set_launch(helios_rt *h, int32_t warps, int32_t ppt, int32_t rows, int32_t stk,
                                          int32_t maxt, int32_t minb) {
  if (!h) return HELIOS_RT_EINVAL;
  const Variant &cur = kVariants[h->variant];
  const int want_ppt = ppt > 0 ? ppt : cur.ppt;
  if (want_ppt > 1 && (h->noniso ? false : (h->cfg.n_gauss % want_ppt) != 0)) return HELIOS_RT_EINVAL;
  const int want_warps = warps > 0 ? warps : h->warps;
  const int v = find_variant(h->noniso, h->toa, cur.bdirect, want_ppt, rows, stk, maxt, minb, want_warps);
  if (v < 0) return HELIOS_RT_EINVAL;
  const int old_v = h->variant, old_w = h->warps;
  h->variant = v;
  h->warps = want_warps;
  int rc = configure_launch(h);
  if (rc) { h->variant = old_v; h->warps = old_w; configure_launch(h); }
  return rc;
}

extern "C" int helios_rt_debug_force_two_launches(helios_rt *h, int32_t on) {
  if (!h) return HELIOS_RT_EINVAL;
  h->force_two_launches = on != 0;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_debug_get_launch(const helios_rt *h, int32_t info[16]) {
  if (!h || !info) return HELIOS_RT_EINVAL;
  const Variant &v = kVariants[h->variant];
  info[0] = h->warps; info[1] = v.ppt; info[2] = v.rows; info[3] = 1; info[4] = v.maxt; info[5] = v.minb;
  info[6] = h->tiles; info[7] = h->workers; info[8] = h->occ; info[9] = h->regs; info[10] = h->lmem;
  info[11] = (int32_t)h->lay.total; info[12] = (int32_t)(h->stack_bytes >> 20); info[13] = h->variant;
  info[14] = kNumVariants; info[15] = 0;
  return HELIOS_RT_OK;
}
