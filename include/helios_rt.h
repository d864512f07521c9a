/*
 * helios_rt.h -- C ABI of the B200-native (sm_100a) radiative-transfer step of THOR+HELIOS
 * (Deitrick et al., arXiv 2203.02293; line numbers below are PAPER.md lines).
 *
 * One call = one pass of the paper's per-timestep multi-wavelength RT module ("Alfrodull",
 * Sec. 2.2.6) over a batch of atmospheric columns, independently for every
 * (column, k-table bin, Gauss point):
 *   S1 level geometry            (Sec. 2.2.1; Fig. 3)
 *   S2 Planck source per bin     (L171, L239)
 *   S3 k-table P-T interpolation (Sec. 2.1.3)
 *   S4 omega0, g0, dtau, beam    (Eqs. 17-18; Eq. B6)
 *   S5 two-stream coefficients   (Eq. 19; Eqs. B1, B2, B5, B8 L1040-1091; Eq. 11)
 *   S6 Thomas solve of the block-tridiagonal flux system (Eqs. 2-10; Eqs. 12-15)
 *   S7 Gauss- and bin-weighted reduction to F_up, F_down (incl. beam, L235), F_net and the
 *      heating rate dT/dt = -dF_net / (c_P dm)            (L393, L1032)
 * Every stage runs in hand-written CUDA kernels in fp64; there is no CPU fallback.  Readings of
 * the paper where it is silent (interpolation scheme, band Planck, interface p/T, ...) are listed
 * in DESIGN.md ("Readings").
 *
 * Conventions: SI units (Pa, K, m, kg, W m^-2).  Layer j (0..N-1) lies between interface j (lower)
 * and j+1 (upper); index 0 = bottom of atmosphere (BOA), interface N = top (TOA).  mu_star > 0 is
 * the dayside (the paper's mu_star is -mu, App. B); mu_star <= 0: no beam.
 * All arrays are fp64 and C-contiguous, (bin, Gauss point) fastest in the k-table.
 *
 * Threading: a handle may be used by one host thread at a time, and the steps of one handle must be
 * stream-ordered (every step uses the handle's workspace, work queues and tile counters: two steps of one handle in
 * flight on different streams race; use one handle per stream).  The launch shape depends on the problem sizes
 * only -- never on the environment.  No call throws, aborts or prints.  Every function returns 0 on success or a
 * negative HELIOS_RT_E* code.
 *
 * Test and benchmark hooks are NOT in this header: launch-shape overrides live in helios_rt_debug.h, the device
 * self-tests and the fp64 FMA microbenchmark in helios_rt_selftest.h (a separate library).
 */
#ifndef HELIOS_RT_H
#define HELIOS_RT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HELIOS_RT_OK        0
#define HELIOS_RT_EINVAL   -1  /* NULL / negative size / non-monotone grid / sum(w) != 1 / w0 outside [0,1] /
                                  n_columns > max_columns / unsupported size / output set inconsistent with flags */
#define HELIOS_RT_ENOMEM   -2  /* host or device allocation failed */
#define HELIOS_RT_ECUDA    -3  /* a CUDA runtime call failed; helios_rt_last_cuda_error() names it */
#define HELIOS_RT_ENODEV   -4  /* no CUDA device, or the device is not compute capability 10.x */
#define HELIOS_RT_ESTUCK   -6  /* a step of this handle gave up waiting for the level data of a column (the flag that
                                  publishes it never arrived within 2^26 polls: a lost write, a device fault).  The step
                                  ran to its end, but its outputs are INVALID.  helios_rt_step_host returns it for its
                                  own step; the asynchronous helios_rt_step cannot know yet, so the NEXT call on the
                                  handle (step, step_host or step_iterative) returns it instead of launching anything,
                                  once.  After it the handle is usable again. */

/* flags */
#define HELIOS_RT_IMPROVED       1u  /* improved two-stream: E from Eq.(19); otherwise E = 1 (regular, L73) */
#define HELIOS_RT_NONISOTHERMAL  2u  /* source linear in tau, two sub-layers per layer (Eqs. 4-9, Fig. 3) */
#define HELIOS_RT_TOA_SPECTRUM   4u  /* post-processing shape (L385): only F_up_toa_bin is produced */

#define HELIOS_RT_MAX_LAYERS 64

typedef struct helios_rt helios_rt; /* opaque; owns all device tables and workspace */

/* ---- create-time configuration: every pointer is a HOST pointer, deep-copied by create ------- */
typedef struct {
  int32_t n_layers;        /* N, 1..HELIOS_RT_MAX_LAYERS                                             */
  int32_t n_bins;          /* k-table wavelength bins                                                */
  int32_t n_gauss;         /* Gauss points per bin (L145)                                            */
  int32_t n_ktab_p;        /* >= 2                                                                   */
  int32_t n_ktab_t;        /* >= 2                                                                   */
  int32_t max_columns;     /* workspace is sized for this many columns per step                      */
  const double *ktab_p;    /* [n_ktab_p] Pa, strictly ascending                                      */
  const double *ktab_t;    /* [n_ktab_t] K,  strictly ascending                                      */
  const double *ktab;      /* [n_ktab_p][n_ktab_t][n_bins][n_gauss] absorption opacity, m^2/kg, > 0  */
  const double *bin_edges; /* [n_bins+1] wavelength, m, strictly ascending, > 0                      */
  const double *gauss_w;   /* [n_gauss], > 0, |sum - 1| <= 1e-10                                     */
  const double *scat_gas;  /* [n_bins] gas (Rayleigh) scattering opacity sigma_scat,gas/mbar, m^2/kg */
  const double *cloud_ext; /* [n_bins] f_cloud (sigma_abs+sigma_scat)_cloud/mbar, m^2/kg; 0 = none   */
  const double *cloud_w0;  /* [n_bins] cloud single-scattering albedo in [0,1]                       */
  const double *cloud_g0;  /* [n_bins] cloud asymmetry factor in [0,1)                               */
  double cloud_p_top;      /* Pa; cloud present at levels with cloud_p_top <= p <= cloud_p_bot       */
  double cloud_p_bot;      /* Pa                                                                     */
  double gravity;          /* m s^-2 (Table 3: 47)                                                   */
  double cp;               /* J kg^-1 K^-1 (Table 3: 12436)                                          */
  double eps2;             /* second Eddington coefficient of the beam, default 2/3 (L1094)          */
  double e_tau;            /* thin sub-layer tolerance, 1e-4 (L209)                                  */
  double gcrit_tol;        /* mu_star,crit guard tolerance, 1e-5 (L252)                              */
  double w0_transition;    /* regular -> improved switch, 0.1 (Eq.19)                                */
  double f_toa;            /* diffuse downward flux per unit wavelength at the TOA, 0 (Fig.5)  */
  uint32_t flags;          /* HELIOS_RT_*                                                            */
} helios_rt_config;

/* ---- per-step inputs: DEVICE pointers (helios_rt_step) or HOST pointers (helios_rt_step_host),
 *      caller-owned, never written ------------------------------------------------------------ */
typedef struct {
  int32_t n_columns;          /* 0..max_columns (0: nothing is launched)                             */
  const double *p;            /* [n_columns][n_layers] layer-centre pressure, Pa; layer 0 = bottom;
                                 strictly decreasing with the layer index                            */
  const double *T;            /* [n_columns][n_layers] K                                             */
  const double *mu_star;      /* [n_columns] cosine of the stellar zenith angle                      */
  const double *stellar_flux; /* [n_bins] TOA normal-incidence flux per unit wavelength, W m^-2 m^-1 */
  double f_internal;          /* W m^-2 >= 0; T_int = (f_internal/sigma_SB)^(1/4),
                                 F_BOA,b = pi B_b(T_int) (Eq.10)                           */
} helios_rt_inputs;

/* ---- per-step outputs: DEVICE (step) or HOST (step_host) pointers, caller-owned; NULL = not wanted
 *      Without HELIOS_RT_TOA_SPECTRUM at least one pointer must be non-NULL; with it, F_up_toa_bin
 *      must be non-NULL and all others NULL. ---------------------------------------------------- */
typedef struct {
  double *F_up;          /* [n_columns][n_layers+1] W m^-2                                           */
  double *F_down;        /* [n_columns][n_layers+1] diffuse + direct beam (L235)                     */
  double *F_net;         /* [n_columns][n_layers+1] F_up - F_down                                    */
  double *dTdt;          /* [n_columns][n_layers]   K s^-1                                           */
  double *F_beam;        /* [n_columns][n_layers+1] direct-beam part of F_down (Fig. 10 check, L245) */
  double *F_up_toa_bin;  /* [n_columns][n_bins]     sum_g w_g F_up at the TOA, W m^-2 m^-1           */
} helios_rt_outputs;

/* Validates cfg, uploads the k-table as ln(kappa) and all per-bin constants, allocates every
 * workspace needed for max_columns.  The caller may free its tables as soon as this returns.
 * On failure *out is NULL. */
int helios_rt_create(const helios_rt_config *cfg, helios_rt **out);

/* One RT step over in->n_columns columns: ONE kernel launch (rt_step_kernel, S1-S7 fused).  Asynchronous: it is
 * enqueued on `cuda_stream` (a cudaStream_t; NULL = the legacy default stream); no host synchronisation, no
 * allocation, no host<->device copy.  Outputs are complete when the stream reaches this point.  NaN inputs
 * propagate to the outputs of their own column only; (p, T) outside the table are clamped to its
 * edge (no extrapolation, not an error).
 *
 * One exception to "one launch" and to bit-reproducibility, for F_up_toa_bin only: when the thread-block tile of the
 * spectral axis (helios_rt_launch_info: info[0] x points per thread) is not a multiple of n_gauss, some bins have
 * their Gauss points in two tiles (BASELINE config 5: tiles of 128 points, n_gauss = 20).  Such a step first
 * launches a zero-fill of F_up_toa_bin (info[6] = 2 for a TOA_SPECTRUM handle; a full-output handle does the same in
 * the steps that ask for F_up_toa_bin) and the tiles add their parts with atomicAdd.  With at most two
 * tiles per bin (n_gauss <= tile) the sum of two terms is the same in either order, so the result is still
 * bit-reproducible; with n_gauss > tile (three or more tiles per bin) the last bits may differ from run to run.
 * F_up, F_down, F_net, dTdt and F_beam are always summed in a fixed order. */
int helios_rt_step(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out,
                   void *cuda_stream);

/* Same step with HOST buffers: copies the inputs to device staging owned by the handle, runs the step on the
 * handle's own stream and synchronises.  Output buffers that are page-locked and mapped (cudaHostAlloc /
 * cudaHostRegister memory) are written by the kernel directly, column by column while the step runs; pageable ones
 * (and a per-bin spectrum whose bins straddle thread-block tiles) are staged on the device and copied back.  Inputs
 * may be pageable or page-locked (page-locked recommended).  This is the end-to-end path bench.py times ("e2e"). */
int helios_rt_step_host(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out);

/* the scheme Thomas's algorithm replaces (L258-270, L397), as a measured comparison:
 * same step, but the flux system is "solved" by n_iterations pair-wise sweeps over the atmosphere (all diffuse
 * fluxes start at 0; one iteration = one upward pass, Eq.(10) then Eq.(2), with the previous downward fluxes,
 * followed by one downward pass, Eq.(3), with the upward fluxes just computed; HELIOS used 200, Oreshenko et
 * al. ~10; reading R23).  Same arguments and outputs as helios_rt_step; HELIOS_RT_TOA_SPECTRUM handles are not
 * supported (EINVAL); n_iterations >= 1. */
int helios_rt_step_iterative(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out,
                             int32_t n_iterations, void *cuda_stream);

/* Frees every device and host resource of the handle (NULL is accepted). */
int helios_rt_destroy(helios_rt *h);

/* Static description of a code returned above. */
const char *helios_rt_strerror(int code);

/* cudaGetErrorString of the last CUDA failure seen by this handle ("" if none). */
const char *helios_rt_last_cuda_error(const helios_rt *h);

/* Launch geometry of the step kernel, for benchmarks and profiles:
 * info[0] = threads per block, [1] = tiles of the spectral axis per column (the persistent grid is tiles x workers),
 * [2] = dynamic shared memory bytes, [3] = registers per thread, [4] = resident blocks per SM (occupancy API),
 * [5] = local-memory bytes per thread, [6] = kernels launched per step (1; 2 for a TOA_SPECTRUM handle whose bins
 * straddle tiles, see helios_rt_step), [7] = SM count of the device. */
int helios_rt_launch_info(const helios_rt *h, int32_t info[8]);

/* ---- the steps either side of the RT step.  DEVICE pointers, fp64,
 *      C-contiguous, caller-owned; asynchronous on `cuda_stream`; no allocation, no synchronisation (so they can
 *      be captured in a CUDA graph together with helios_rt_step). ------------------------------------------- */

/* Post-processing column extension (L385): p_ext, T_ext [n_columns][n_layers + n_extra] receive the input
 * column followed by n_extra layers above the model top, equally spaced in ln p with the per-layer ratio
 * q = min(p[N-1]/p[N-2], (p_min/p[N-1])^(1/n_extra)) (so the new top is <= p_min; reading R21) and
 * T = T[N-1] ("isothermal above the original model top"). */
int helios_rt_extend_top(int32_t n_columns, int32_t n_layers, int32_t n_extra, double p_min, const double *p,
                         const double *T, double *p_ext, double *T_ext, void *cuda_stream);

/* Phase curve on the icosahedral grid, Eqs.(25)-(26) (L546-552):
 *   F_phase_bin[a][b] = sum_i F_toa_bin[i][b] / pi * mu_i(alpha_a) * area[i],
 *   mu_i = cos(lat_i) cos(lon_i - alpha_a) where that cosine is > 0 (visible hemisphere, modulo 2 pi), else 0;
 * area[i] = A_i / R_p^2.  If F_phase_band is non-NULL also the wavelength integral of Eq.(23) (L521):
 *   F_phase_band[a] = sum_b |[bin_edges[b], bin_edges[b+1]] n [lam1, lam2]| * F_phase_bin[a][b]
 * (HST-WFC3: 1.1-1.7 um).  F_toa_bin [n_columns][n_bins] is the TOA_SPECTRUM output of helios_rt_step; lon, lat,
 * area [n_columns] (radians, steradians); alpha [n_phases]; bin_edges [n_bins+1]; F_phase_bin
 * [n_phases][n_bins] (required); F_phase_band [n_phases] or NULL; workspace: DEVICE scratch of
 * helios_rt_phase_curve_workspace_bytes(...) bytes, caller-owned (partial sums per chunk of 128 columns).
 * The column sum runs in a fixed order (within a chunk, then over chunks): deterministic run to run. */
int helios_rt_phase_curve(int32_t n_columns, int32_t n_bins, int32_t n_phases, const double *F_toa_bin,
                          const double *lon, const double *lat, const double *area, const double *alpha,
                          const double *bin_edges, double lam1, double lam2, double *F_phase_bin,
                          double *F_phase_band, double *workspace, void *cuda_stream);

/* Size in bytes of the scratch buffer helios_rt_phase_curve needs (>= 8; negative = HELIOS_RT_EINVAL). */
int64_t helios_rt_phase_curve_workspace_bytes(int32_t n_columns, int32_t n_bins, int32_t n_phases);

/* ---- helios_rt_phase_curve for callers that must not allocate --------------------------------------------------
 *
 * Who this is for.  helios_rt_phase_curve needs a scratch buffer (the partial sums per chunk of 128 columns), and
 * normally the caller gets it from cudaMalloc or from a framework's allocator.  Some callers cannot do either at
 * the point where they want the phase curve: code running inside a host callback or a plug-in hook of a larger
 * application that owns all device memory and hands out none; a real-time or fault-handling path that must not
 * enter the driver's allocator (an allocation can block for milliseconds, fail when the device is full, or
 * synchronise the whole device and so stall other streams); a worker whose memory budget was fixed at start-up
 * and is already spent on its handles.  For them this variant brings its own scratch: a fixed array of
 * HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES that is part of the library image itself (a file-scope
 * `static __device__` array in helios_post.cu).  The call performs no cudaMalloc / cudaFree and calls no library
 * routine that allocates; the caller passes inputs and outputs only.
 *
 * Same arguments, results and errors as helios_rt_phase_curve, minus `workspace`: the two paths run the same
 * kernels in the same order, so for the same inputs the outputs are bit-identical.
 *
 * What it costs and what to watch:
 *   - Size limit.  helios_rt_phase_curve_workspace_bytes(n_columns, n_bins, n_phases) must not exceed
 *     HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES (8 MiB: e.g. 2562 columns x 64 phases x 780 bins, or 10242 columns x
 *     64 phases x 200 bins).  Anything larger is refused with HELIOS_RT_ETOOBIG before any work is queued; use
 *     helios_rt_phase_curve with your own buffer for those.
 *   - Memory.  Every GPU on which this process loads the library's device code carries the 8 MiB from then until
 *     the process exits, whether or not this function is ever called.
 *   - First call on a device.  The first call made while a given device is current looks up where the array lives
 *     on THAT device (cudaGetSymbolAddress; one array exists per device, at different addresses) and remembers the
 *     answer; later calls on that device only read it.  The look-up may make the CUDA runtime load the library's
 *     device code, so make this first call during start-up, outside any stream capture.  The device that is current
 *     at the call must be the device `cuda_stream` and all the pointers belong to.
 *   - One array, shared.  All calls on a device use the same scratch, and it keeps whatever the last call left in
 *     it.  Nothing in it needs to start at zero (every element the second kernel reads is first written by the
 *     first kernel of the same call), so no clearing is done.  But two calls that can overlap on the GPU -- issued on
 *     different streams, or from different host threads, without an event or synchronisation ordering them -- write
 *     over each other's partial sums and both results are garbage.  Keep calls on one device stream-ordered.
 *   - Host threads.  The one-time look-up is guarded by a lock; after it the function is as thread-safe as
 *     helios_rt_phase_curve, subject to the previous point. */
#define HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES 8388608
#define HELIOS_RT_ETOOBIG  -5  /* helios_rt_phase_curve_noalloc: the problem needs more scratch than the built-in
                                  array holds (HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES)                       */
int helios_rt_phase_curve_noalloc(int32_t n_columns, int32_t n_bins, int32_t n_phases, const double *F_toa_bin,
                                  const double *lon, const double *lat, const double *area, const double *alpha,
                                  const double *bin_edges, double lam1, double lam2, double *F_phase_bin,
                                  double *F_phase_band, void *cuda_stream);

/* "1-D mode" (Sec. 3): explicit temperature step T <- T + dt * dTdt (dTdt NULL: T unchanged) followed
 * by the hydrostatic re-balance of Eq.(20) on the fixed altitude grid z [n_layers] (m, ascending): p[.][0] =
 * p_ref, p_i = p_{i-1} (1/dz - g/(2 R_d T_{i-1})) / (1/dz + g/(2 R_d T_i)) (sign of the denominator: reading
 * R25), rho = p / (R_d T) (rho may be NULL).  T [n_columns][n_layers] is updated in place; p, rho are outputs. */
int helios_rt_advance_1d(int32_t n_columns, int32_t n_layers, double dt, double gravity, double R_d, double p_ref,
                         const double *z, const double *dTdt, double *T, double *p, double *rho, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* HELIOS_RT_H */
