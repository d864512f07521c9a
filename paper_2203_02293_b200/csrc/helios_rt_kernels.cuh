// helios_rt_kernels.cuh -- device code of the RT step (rt_step_kernel, rt_iter_kernel, rt_prep_kernel) and the table of compiled
// instantiations.  Included by helios_rt.cu (host side, comparison and fallback kernels) and by one translation unit per
// class of rt_step_kernel instantiations (helios_rt_k_*.cu): nvcc's code for a kernel depends on what else is optimised with
// it, so each class is compiled on its own and a change to one cannot move the others.
#pragma once

#include "../../include/helios_rt.h"
#include "../../include/helios_rt_debug.h"
#include "helios_rt_math.cuh"

#include <stdlib.h>
#include <string.h>
#include <new>
#include <type_traits>

namespace hrt_k {


using namespace hrt;

constexpr int MAXL = HELIOS_RT_MAX_LAYERS;

// unroll factor of the isothermal sweep-1 loop (1: measured best; comparison builds override it)
#ifndef HRT_UNROLL_ISO
#define HRT_UNROLL_ISO 1
#endif
// An empty asm that "modifies" a loop-invariant value: ptxas then keeps it in a register (or spills it) instead of
// recomputing it from thread / block indices inside the sweep loops
#define HRT_PIN_PTR(p) asm volatile("" : "+l"(p))
#define HRT_PIN_F64(x) asm volatile("" : "+d"(x))
#ifndef HRT_PIN_LEVEL
#define HRT_PIN_LEVEL 1
#endif
#ifndef HRT_PA_UNROLL
#define HRT_PA_UNROLL 2   /* config 2: 0.6787 ms at 2, 0.6845 at 4, 0.6851 at 8 */
#endif
#ifndef HRT_VOTE_SEL
#define HRT_VOTE_SEL (!TOA || BDIRECT)
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
  unsigned *err;          // the handle's error word (device alias of page-locked host memory): set to 1 by a block that
                          // gave up waiting for a column's publication flag (HELIOS_RT_ESTUCK)
  unsigned poll_limit;    // polls of a publication flag before giving up (2^26; tests force a small value)
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
  if (HRT_PIN_LEVEL >= 2) HRT_PIN_PTR(stage_wr);

  // ---------------- phase A: this block's share of the (column, level) items of S1 + S2 ----------------
  if (P.fused_prep) {
    __syncthreads();                       // s_T32
    const long nblk = (long)gridDim.x * gridDim.y;
    // (skipping the Planck forms no lane of a warp needs: -0.5 % on config 2, -1.2 % on configs 3 / 4, -7 % on config 6,
    // +0.9 % on config 5 -- per-class choice: HRT_VOTE_SEL)
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
    HRT_PIN_PTR(feed.lnk_pt);
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
  // the lane's own slots of a row: + lane (PPT = 1) or + lane 16-byte pairs
  double *stk_wl = stk_w ? stk_w + (PPT == 1 ? lane : 2 * lane) : nullptr;
  HRT_PIN_PTR(stk_w);
  if (HRT_PIN_LEVEL >= 2) HRT_PIN_PTR(stk_wl);

  // ---------------- phase B: columns of this tile's queue ----------------
  // The record block and the tile's Planck block of the NEXT column are fetched by bulk async copies (TMA) into the
  // other shared-memory buffer while this column is swept; thread 0 first waits for the column's publication flag.
  bool all_published = false;               // thread 0: every block has finished phase A -- no more flag polls
  auto fetch_column = [&](int c, int buf) {   // thread 0
    // (the whole grid is resident -- cooperative launch -- and phase A waits for nothing, so this terminates; the
    // poll count is bounded all the same, so that a lost flag cannot wedge the GPU.  A block that gives up says so in
    // the handle's error word: the step still runs to its end, on whatever the workspace holds, but the host
    // reports HELIOS_RT_ESTUCK for it -- its outputs are never passed off as results.)
    if (!all_published) {
      unsigned n;
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(n) : "l"(P.queue + P.tiles + 1) : "memory");
      all_published = (n == gridDim.x * gridDim.y);
      if (!all_published) {
        unsigned f, polls = 0;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(P.flags + c) : "memory");
        } while (f != (unsigned)(nlev + 1) && ++polls < P.poll_limit);
        if (f != (unsigned)(nlev + 1)) {
          *(volatile unsigned *)P.err = 1u;
          __threadfence_system();
        }
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
      double muF = day ? mu * fstar_b : 0.0;                  // mu * F_star[b]
      double inv_mu = day ? 1.0 / mu : 0.0;
      HRT_PIN_F64(muF); HRT_PIN_F64(inv_mu);

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
        stk_store<PPT>(stk_wl + (size_t)(srow_i--) * SROW, 0, c, wd, Rlow);   // (a running pointer measured 1 % slower)
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
        const double *row = stk_w, *row_l = stk_wl;
        auto group = [&](auto full_tag, int base) {
          constexpr bool FULL = decltype(full_tag)::value;
          const int nk = N + 1 - base;          // interfaces left (FULL: > 8)
          double gc[8][PPT], gwd[8][PPT], gR[8][PPT], sd[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            if (FULL || k < nk) stk_load_cw<PPT>(row_l + k * SROW, 0, gc[k], gwd[k]);
            else {
#pragma unroll
              for (int q = 0; q < PPT; ++q) { gc[k][q] = 1.0; gwd[k][q] = 0.0; }
            }
            if (FULL || k < nk - 1) stk_load_R<PPT>(row_l + (k + 1) * SROW, 0, gR[k]);
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
          // rows base .. base+7 are dead (the R part of row base+8 is not: next group's discard): drop the lines that
          // are still in L2 instead of writing them back (at the config-2 shape the oldest rows have already been
          // evicted to HBM by then: helios_rt.cu header)
          const int n_lines = (FULL ? 8 : nk) * (SROW / 16);
          for (int ln = lane; ln < n_lines; ln += 32) l2_discard(row + ln * 16);
        };
        int base = 0;
#pragma unroll 1
        for (; base + 8 <= N; base += 8, row += 8 * SROW, row_l += 8 * SROW) group(std::true_type{}, base);
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


// --------------------------------------------------------------------------------------------
// compiled instantiations: one table per class, defined in helios_rt_k_*.cu
// --------------------------------------------------------------------------------------------
struct Variant {
  bool noniso, toa, bdirect;
  int ppt, rows, warps;   // warps: block size compiled in, 0 = any
  int maxt, minb;      // launch bounds: register cap = 65536 / (maxt * minb)
  const void *fn;   // rt_step_kernel<...>, launched through cudaLaunchKernelExC
};

#define HRT_K(NI, TOA, PPT, ROWS, WARPS, MAXT, MINB) \
  {NI, TOA, false, PPT, ROWS, WARPS, MAXT, MINB, (const void *)rt_step_kernel<NI, TOA, PPT, ROWS, false, WARPS, MAXT, MINB>}
// one Gauss point per bin (opacity sampling): Planck values read from the workspace; one point per thread
#define HRT_KB(NI, TOA, ROWS, WARPS, MAXT, MINB) \
  {NI, TOA, true, 1, ROWS, WARPS, MAXT, MINB, (const void *)rt_step_kernel<NI, TOA, 1, ROWS, true, WARPS, MAXT, MINB>}

// In order of preference within a class: helios_rt_create takes the first match; helios_rt_debug_set_launch (tests, tuning)
// may select any other.  Shapes were chosen by same-box A/B runs.
extern const Variant kVariantsIsoFull[];   extern const int kNumIsoFull;     // helios_rt_k_iso.cu
extern const Variant kVariantsIsoToa[];    extern const int kNumIsoToa;      // helios_rt_k_toa.cu
extern const Variant kVariantsNoniso[];    extern const int kNumNoniso;      // helios_rt_k_noniso.cu
extern const Variant kVariantsSampling[];  extern const int kNumSampling;    // helios_rt_k_sampling.cu

}  // namespace hrt_k
